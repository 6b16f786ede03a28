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


#        grid_p      deg_p      pair  expected real rows (None = only check > nRp)
CASES = [((3, 3, 3), None, 1, 27),            # symmetric: 13 pairs x 2 + R = 0
         ((5, 3, 1), None, 1, 15),
         ((3, 3, 3), "broken", 1, 31),         # unequal weights inside two pairs -> those four vectors have no partner
         ((3, 3, 3), "symmetric", 1, 27),      # non-trivial but inversion-symmetric degeneracies
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
            assert np.array_equal(res[(sign, pair)], np.stack(per_k))
        assert _relerr(res[(sign, 1)], res[(sign, 0)]) <= 1e-12
    assert _relerr(res[(1, 1)], res[(-1, 1)]) > 1e-3          # the conventions really differ
    ctx.close()
