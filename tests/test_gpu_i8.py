"""GPU parity of step a4 on the INT8 tensor cores (contract_i8.cuh): the +R / -R pair form of the Rp contraction
(Eq. 70) with every FP64 operand split exactly into six signed base-256 digits, 21 digit-pair INT8 GEMMs
(tcgen05.mma kind::i8, INT32 accumulators in TMEM) recombined in 64-bit integers and rounded once.
Checked against the CPU oracle (which knows nothing of digits) and against the FP64 tensor-core pair kernel on the same
inputs: several tiles per CTA (accumulator hand-over between the MMA and the epilogue warps), ring wrap-around, ragged
row / column / depth tails, the cluster (multicast) variants, the stacked multi-k form, extreme operand scales and
all-zero columns.  Bar: max |d out| <= 1e-10 max(out)  (north_star, reading R10); the digit-split error itself is
~1e-13 of a column's scale.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _relerr(got, ref):
    return float(np.max(np.abs(got - ref)) / np.max(np.abs(ref)))


@pytest.fixture(scope="module")
def env():
    import torch
    import oracle
    from paper_2111_14999_b200 import binding, build, harness, workloads as wl
    build.build()
    binding.load_library()
    assert torch.cuda.is_available()
    return dict(torch=torch, oracle=oracle, binding=binding, harness=harness, wl=wl)


def _inputs(wl, w, ik=0):
    return dict(gW=wl.gW_full(w), Re=wl.Re_vectors(w), Rp=wl.Rp_vectors(w), k=wl.k_points(w)[ik], Uk=wl.U_k(w, ik),
                q=wl.q_points(w, ik), Ukq=wl.U_kq(w, ik), ev=wl.ph_eigvecs(w, ik), om=wl.omega(w, ik))


def _ctx(env, w, gW_np, nq_max, i8, **kw):
    ctx = env["harness"].make_context(w, env["torch"].from_numpy(gW_np).cuda(), nq_max=nq_max, **kw)
    ctx.set_tuning("tile", 64)
    ctx.set_tuning("pair", 2)
    ctx.set_tuning("i8", i8)
    return ctx


#         nw nb1 nb2 nm  grid_p     nq    what
CASES = [(5, 4, 5, 6, (3, 3, 3), 333),       # 3 x 4 tiles, ragged rows (333 = 2 x 128 + 77) and columns (2 N = 240)
         (8, 8, 8, 6, (5, 5, 3), 2500),      # 20 x 12 = 240 tiles > 148 CTAs: a second tile per CTA; depth 85 -> 4 chunks
         (3, 2, 3, 3, (7, 7, 5), 130),       # deep and narrow: 2 N = 36 < one column tile, 245 vectors -> more chunks than stages
         (4, 4, 4, 3, (2, 3, 1), 64)]        # vectors without a partner, fewer rows than one row tile


@pytest.mark.parametrize("case", CASES, ids=lambda c: "nw%d_nb%d_%d_nm%d_p%d%d%d_nq%d" % (c[:4] + c[4] + (c[5],)))
def test_i8_matches_oracle_and_fp64_pair_kernel(env, case):
    wl, oracle, harness = env["wl"], env["oracle"], env["harness"]
    nw, nb1, nb2, nm, grid_p, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=(2, 2, 1), grid_p=grid_p, nq=nq, cfg_id=170)
    a = _inputs(wl, w)
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = _ctx(env, w, a["gW"], nq, 1)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    out_i8 = ctx.q_batch(*d).cpu().numpy()
    assert ctx.get_tuning("i8") == 1                       # the last a4 DID run on the INT8 path
    n0 = ctx.launch_counts()["contract"]
    ctx.set_tuning("i8", 0)
    out_f64 = ctx.q_batch(*d).cpu().numpy()
    assert ctx.get_tuning("i8") == 0 and ctx.launch_counts()["contract"] == n0 + 1
    ctx.set_tuning("i8", 1)                                # and back: the digit planes are still valid
    out_again = ctx.q_batch(*d).cpu().numpy()
    ctx.close()
    assert _relerr(out_i8, ref) <= TOL
    assert _relerr(out_f64, ref) <= TOL
    assert _relerr(out_i8, out_f64) <= 1e-12               # both are exact up to rounding: far inside the bar
    assert np.array_equal(out_i8, out_again)               # integer accumulation: bit-reproducible


@pytest.mark.parametrize("cl", [1, 2, 4, 8])
def test_i8_cluster_variants_are_bit_identical(env, cl):
    """Clusters of 1 / 2 / 4 / 8 CTAs (A digit planes multicast) compute the same integers: identical bits; an odd number of
    column tiles leaves one CTA of the last cluster without a tile of its own."""
    wl, oracle, harness = env["wl"], env["oracle"], env["harness"]
    w = wl.custom(nw=6, nb1=5, nb2=6, nm=9, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nq=700, cfg_id=171)   # 2 N = 540: 9 column tiles
    a = _inputs(wl, w)
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = _ctx(env, w, a["gW"], 700, 1)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    base = ctx.q_batch(*d).cpu().numpy()
    ctx.set_tuning("i8_cluster", cl)
    out = ctx.q_batch(*d).cpu().numpy()
    assert ctx.get_tuning("i8_cluster") == cl
    ctx.close()
    assert _relerr(out, ref) <= TOL
    assert np.array_equal(out, base)


@pytest.mark.parametrize("scale", [1e-140, 1e-30, 1.0, 1e30, 1e140])
def test_i8_operand_scale_extremes(env, scale):
    """The column scales are powers of two taken from the data: g_W scaled by 1e-140 .. 1e140 gives |g|^2 scaled by its
    square with the SAME relative accuracy (nothing in the digit split depends on the magnitude)."""
    wl, oracle, harness = env["wl"], env["oracle"], env["harness"]
    w = wl.custom(nw=4, nb1=3, nb2=4, nm=3, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nq=200, cfg_id=172)
    a = _inputs(wl, w)
    gW = a["gW"] * scale
    ref = oracle.elph(gW, a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = _ctx(env, w, gW, 200, 1)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    out = ctx.q_batch(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])).cpu().numpy()
    assert ctx.get_tuning("i8") == 1
    ctx.close()
    assert np.all(np.isfinite(out)) and ref.max() > 0.0
    assert _relerr(out, ref) <= TOL


def test_i8_zero_columns_and_mixed_magnitudes(env):
    """Columns of g1' that are identically zero (scale 1, zero digits) and columns 1e-9 times smaller than their
    neighbours (each column has its OWN scale, so the small ones keep their relative accuracy)."""
    wl, oracle, harness = env["wl"], env["oracle"], env["harness"]
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nq=260, cfg_id=173)
    a = _inputs(wl, w)
    gW = a["gW"].copy()                     # [nRp][nRe][w1][w2][mode]; the columns of g1' are (b1, w2, mode)
    gW[:, :, :, 1, :] = 0.0                 # every column with w2 = 1 is zero
    gW[:, :, :, 3, :] *= 1e-9               # and those with w2 = 3 are tiny
    ref = oracle.elph(gW, a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    # the same with ONLY the tiny columns kept: their own contribution, to full relative accuracy
    gW_small = np.zeros_like(gW)
    gW_small[:, :, :, 3, :] = gW[:, :, :, 3, :]
    ref_small = oracle.elph(gW_small, a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    outs = []
    for g in (gW, gW_small):
        ctx = _ctx(env, w, g, 260, 1)
        ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
        outs.append(ctx.q_batch(*d).cpu().numpy())
        assert ctx.get_tuning("i8") == 1
        ctx.close()
    assert np.all(np.isfinite(outs[0])) and np.all(np.isfinite(outs[1]))
    assert _relerr(outs[0], ref) <= TOL
    assert ref_small.max() < 1e-15 * ref.max() and _relerr(outs[1], ref_small) <= TOL


def test_i8_stacked_multi_k_and_fallback(env):
    """q_batch_multi: a stack of 128-row multiples runs on the INT8 path (a row tile never straddles two k slots) and
    equals the per-k calls bit for bit; any other stack height takes the FP64 pair kernel."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nk = 3
    for nq, expect_i8 in ((256, 1), (192, 0)):       # (the stacked form wants multiples of 64)
        w = wl.custom(nw=4, nb1=3, nb2=4, nm=3, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nk=nk, nq=nq, cfg_id=174)
        gW_np = wl.gW_full(w)
        ctx = _ctx(env, w, gW_np, nk * nq, 1, nk_max=nk)
        Uks = np.stack([wl.U_k(w, i) for i in range(nk)])
        st = [np.ascontiguousarray(np.stack([f(w, i) for i in range(nk)]))
              for f in (wl.q_points, wl.U_kq, wl.ph_eigvecs, wl.omega)]
        d = harness.to_device(st)
        ctx.set_k_batch(wl.k_points(w), harness.to_device([Uks])[0])
        multi = ctx.q_batch_multi(*d).cpu().numpy()
        assert ctx.get_tuning("i8") == expect_i8
        per_k = []
        for i in range(nk):
            ctx.select_k(i)
            per_k.append(ctx.q_batch(*[t[i].contiguous() for t in d]).cpu().numpy())
            assert ctx.get_tuning("i8") == 1
        ctx.close()
        per_k = np.stack(per_k)
        if expect_i8:
            assert np.array_equal(multi, per_k)
        assert _relerr(multi, per_k) <= 1e-12
        for i in range(nk):
            ref = oracle.elph(gW_np, wl.Re_vectors(w), wl.Rp_vectors(w), None, None, wl.k_points(w)[i], Uks[i],
                              st[0][i], st[1][i], st[2][i], st[3][i])
            assert _relerr(multi[i], ref) <= TOL


def test_i8_non_finite_input_becomes_nan(env):
    """A NaN in g_W must not come out as a finite number.  It reaches one column (w2, kappa) of g1' for every b1 (0 * NaN in the
    U_k rotation), the column-maximum pass flags that column, the contraction returns NaN there, and the two rotations spread it
    over every |g|^2 -- on the INT8 path exactly as on the FP64 one."""
    wl, harness = env["wl"], env["harness"]
    w = wl.custom(nw=4, nb1=3, nb2=4, nm=3, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nq=140, cfg_id=176)
    a = _inputs(wl, w)
    gW = a["gW"].copy()
    gW[5, 1, 1, 2, 0] = np.nan                 # [p][e][w1][w2][kappa]
    for i8 in (1, 0):
        ctx = _ctx(env, w, gW, 140, i8)
        ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
        out = ctx.q_batch(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])).cpu().numpy()
        assert ctx.get_tuning("i8") == i8
        ctx.close()
        assert np.all(np.isnan(out))


def test_i8_row_limit_falls_back_to_fp64(env):
    """Exact INT32 accumulation holds for up to 16384 pair rows (6 digit pairs x rows x 128^2 < 2^31): a longer lattice-vector
    list takes the FP64 pair kernel, one just below the limit stays on the INT8 path (128 chunks per tile through a 6-stage ring)."""
    wl, oracle, harness = env["wl"], env["oracle"], env["harness"]
    for grid_p, expect_i8 in (((27, 27, 23), 0), ((25, 25, 25), 1)):          # 16767 and 15625 vectors
        w = wl.custom(nw=2, nb1=2, nb2=2, nm=1, grid_e=(1, 1, 1), grid_p=grid_p, lam=40.0, nq=130, cfg_id=177)
        a = _inputs(wl, w)
        ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
        ctx = _ctx(env, w, a["gW"], 130, 1)
        rows = ctx.get_tuning("pair_rows")
        assert (rows > 16384) == (expect_i8 == 0)
        ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
        out = ctx.q_batch(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])).cpu().numpy()
        assert ctx.get_tuning("i8") == expect_i8
        ctx.close()
        assert _relerr(out, ref) <= TOL


def test_i8_bits_do_not_depend_on_the_batching(env):
    """Integer accumulation has no rounding order: the same q-points give the same bits whether they are contracted in one
    launch, in sub-batches of 128 (tuning nq_sub), as a prefix of the list, or in another position of a longer list."""
    wl, harness = env["wl"], env["harness"]
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nq=700, cfg_id=178)
    a = _inputs(wl, w)
    ctx = _ctx(env, w, a["gW"], 700, 1)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    whole = ctx.q_batch(*d).cpu().numpy()
    ctx.set_tuning("nq_sub", 128)
    split = ctx.q_batch(*d).cpu().numpy()
    assert ctx.launch_counts()["contract"] == 1 + 6
    ctx.set_tuning("nq_sub", 1 << 20)
    prefix = ctx.q_batch(*[t[:300].contiguous() for t in d]).cpu().numpy()
    shifted = ctx.q_batch(*[t[211:].contiguous() for t in d]).cpu().numpy()
    ctx.close()
    assert np.array_equal(whole, split)
    assert np.array_equal(whole[:300], prefix)
    assert np.array_equal(whole[211:], shifted)
