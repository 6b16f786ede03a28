"""GPU parity of the +R / -R pair form of step a4 (contract_pair.cuh): the Rp contraction as a REAL x complex GEMM,
    w e^{i th} g1'[p] + w e^{-i th} g1'[pbar] = (w cos th)(g1'[p] + g1'[pbar]) + (w sin th) i (g1'[p] - g1'[pbar]),
against the CPU oracle (which knows nothing of pairs) and against the planar three-multiply kernel: symmetric grids,
lists with vectors that have no partner, unequal degeneracies inside a pair, the opposite phase sign (Eq. 5
conventions), the stacked multi-k form.  Bar: max |d out| <= 1e-10 max(out)  (north_star, reading R10).
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


#        grid_p      deg_p      pair  expected real rows (None = only check > nRp): cosine block padded to 16 + sine block
CASES = [((3, 3, 3), None, 1, 29),            # symmetric: 13 pairs + R = 0 -> 14 -> 16 cosine rows, 13 sine rows
         ((5, 3, 1), None, 2, 23),            # 7 pairs + R = 0 -> 8 -> 16, + 7 (forced: 4 x 23 rows > 6 x 15 vectors)
         ((3, 3, 3), "broken", 1, 31),         # unequal weights inside two pairs -> those four vectors have no partner: 15 + 1, + 15
         ((3, 3, 3), "symmetric", 1, 29),      # non-trivial but inversion-symmetric degeneracies
         ((2, 3, 1), None, 2, None),           # x in {-1, 0}: the x = -1 vectors have no partner
         ((4, 1, 1), None, 2, None)]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "grid%d%d%d_%s_pair%d" % (c[0] + (c[1], c[2])))
def test_pair_form_matches_oracle_and_planar(env, case):
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    grid_p, degs, pair, rows = case
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(2, 2, 1), grid_p=grid_p, nq=333, cfg_id=140)
    a = _inputs(wl, w)
    deg_p = None
    if degs == "broken":
        deg_p = np.ones(w.nRp); deg_p[0] = 2.0; deg_p[5] = 3.0
    elif degs == "symmetric":
        deg_p = 1.0 + np.abs(a["Rp"]).sum(axis=1)
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, deg_p, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=333, deg_p=deg_p)
    ctx.set_tuning("tile", 64)
    ctx.set_tuning("pair", pair)
    kr = ctx.get_tuning("pair_rows")
    assert kr == rows if rows is not None else kr > w.nRp
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    out_pair = ctx.q_batch(*d).cpu().numpy()
    ctx.set_tuning("pair", 0)
    assert ctx.get_tuning("pair_rows") == 0
    out_planar = ctx.q_batch(*d).cpu().numpy()
    ctx.set_tuning("pair", pair)                 # and back: the operand copy is re-packed in the other form
    out_again = ctx.q_batch(*d).cpu().numpy()
    ctx.close()
    assert _relerr(out_pair, ref) <= TOL
    assert _relerr(out_planar, ref) <= TOL
    assert np.array_equal(out_pair, out_again)


def test_pair_form_opposite_phase_sign_and_stacked(env):
    """phase_sign = -1 (the Eq. 5 conventions) flips the sine rows; the stacked multi-k form switches pair-row slabs."""
    wl, torch, harness = env["wl"], env["torch"], env["harness"]
    nk = 3
    w = wl.custom(nw=4, nb1=3, nb2=4, nm=3, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nk=nk, nq=128, cfg_id=141)
    gW_np = wl.gW_full(w)
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=nk * 128, nk_max=nk)
    ctx.set_tuning("tile", 64)
    Uks = np.stack([wl.U_k(w, i) for i in range(nk)])
    st = [np.ascontiguousarray(np.stack([f(w, i) for i in range(nk)]))
          for f in (wl.q_points, wl.U_kq, wl.ph_eigvecs, wl.omega)]
    d = harness.to_device(st)
    res = {}
    for sign, conj in ((1, (False, True, False)), (-1, (True, True, True))):
        ctx.set_conventions(sign, *conj)
        for pair in (1, 0):
            ctx.set_tuning("pair", pair)
            ctx.set_k_batch(wl.k_points(w), harness.to_device([Uks])[0])
            res[(sign, pair)] = ctx.q_batch_multi(*d).cpu().numpy()
            per_k = []
            for i in range(nk):
                ctx.select_k(i)
                per_k.append(ctx.q_batch(*[t[i].contiguous() for t in d]).cpu().numpy())
            assert _relerr(res[(sign, pair)], np.stack(per_k)) <= 1e-12       # equal up to the rounding order
        assert _relerr(res[(sign, 1)], res[(sign, 0)]) <= 1e-12
    assert _relerr(res[(1, 1)], res[(-1, 1)]) > 1e-3          # the conventions really differ
    ctx.close()


def _run_custom_lists(env, gW, Re, Rp, deg_p, k, Uk, q, Ukq, ev, om, pair):
    """The C ABI over explicit lattice-vector lists (not a grid of workloads.py) -> (out, real rows of the pair form)."""
    torch, binding, harness = env["torch"], env["binding"], env["harness"]
    ctx = binding.ElphContext(torch.from_numpy(gW).cuda(), Re, Rp, None, deg_p, nb1_max=Uk.shape[1],
                              nb2_max=Ukq.shape[2], nq_max=len(q))
    ctx.set_tuning("tile", 64)
    ctx.set_tuning("pair", pair)
    rows = ctx.get_tuning("pair_rows")
    ctx.set_k(k, harness.to_device([Uk])[0])
    out = ctx.q_batch(*harness.to_device([q, Ukq, ev, om])).cpu().numpy()
    ctx.close()
    return out, rows


def _custom_inputs(wl, nRe, nRp, seed, nw=4, nb1=3, nb2=4, nm=6, nq=200):
    rng = np.random.default_rng(seed)
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=(nRe, 1, 1), grid_p=(nRp, 1, 1), nq=nq, cfg_id=142)
    gW = (rng.standard_normal((nRp, nRe, nw, nw, nm)) + 1j * rng.standard_normal((nRp, nRe, nw, nw, nm)))
    return w, rng, gW, wl.k_points(w)[0], wl.U_k(w), wl.q_points(w), wl.U_kq(w), wl.ph_eigvecs(w), wl.omega(w)


@pytest.mark.parametrize("kind", ["generic", "symmetric"])
@pytest.mark.parametrize("pair", [0, 1, 2])
def test_non_integer_lattice_vectors(env, kind, pair):
    """Reading R12: Re / Rp are doubles and need not be integers (only Eq. 87's periodicity needs that).  generic: no
    vector has an inversion partner (the pair map degenerates to two rows per vector); symmetric: non-integer vectors
    that do come in exact +R / -R pairs, plus the origin."""
    wl, oracle = env["wl"], env["oracle"]
    nRe, nRp = 5, 11
    w, rng, gW, k, Uk, q, Ukq, ev, om = _custom_inputs(wl, nRe, nRp, 7)
    Re = rng.uniform(-2.5, 2.5, (nRe, 3))
    if kind == "generic":
        Rp = rng.uniform(-3.0, 3.0, (nRp, 3))
    else:
        half = rng.uniform(-3.0, 3.0, (nRp // 2, 3))
        Rp = np.concatenate([half, np.zeros((1, 3)), -half[::-1]])
        Rp = Rp[rng.permutation(nRp)]
    ref = oracle.elph(gW, Re, Rp, None, None, k, Uk, q, Ukq, ev, om)
    out, rows = _run_custom_lists(env, gW, Re, Rp, None, k, Uk, q, Ukq, ev, om, pair)
    if kind == "symmetric" and pair == 2:
        assert rows == 16 + 5         # 5 pairs + the origin -> 6 -> 16 cosine rows, 5 sine rows (forced: too short a list to pay)
    assert _relerr(out, ref) <= TOL


@pytest.mark.parametrize("pair", [0, 1, 2])
def test_duplicated_lattice_vectors(env, pair):
    """An Rp list that names the same vector more than once (each entry with its own slab of g_W and its own
    degeneracy): the sum of Eq. 13 runs over list ENTRIES, so duplicates simply add.  Pair-map edge cases: a vector
    with two copies and one partner, a duplicated origin, a duplicated partner."""
    wl, oracle = env["wl"], env["oracle"]
    Rp = np.array([[1, 0, 0], [-1, 0, 0], [1, 0, 0], [0, 0, 0], [0, 0, 0], [0, 2, -1], [0, -2, 1], [0, -2, 1],
                   [2, 1, 0], [1, 0, 0]], dtype=np.float64)
    nRp, nRe = len(Rp), 3
    w, rng, gW, k, Uk, q, Ukq, ev, om = _custom_inputs(wl, nRe, nRp, 11)
    Re = wl.Re_vectors(w)
    deg_p = np.array([1, 1, 1, 2, 2, 1, 1, 3, 1, 2], dtype=np.float64)
    ref = oracle.elph(gW, Re, Rp, None, deg_p, k, Uk, q, Ukq, ev, om)
    out, rows = _run_custom_lists(env, gW, Re, Rp, deg_p, k, Uk, q, Ukq, ev, om, pair)
    assert _relerr(out, ref) <= TOL
    # q -> q + G (Eq. 87) still holds for this integer list
    out2, _ = _run_custom_lists(env, gW, Re, Rp, deg_p, k, Uk, q + np.array([1.0, -2.0, 3.0]), Ukq, ev, om, pair)
    assert _relerr(out2, ref) <= TOL
