"""GPU parity of steps a5-a7 on the tensor cores (k_rotate_v3: persistent, producer warp + TMA rings, packed (b1, kappa)
columns, three-multiply product): every k-step count KS = ceil(nm/4) in 1..12 and every residue of nm mod 4 (the padded
row pitch of C for nm = 0 mod 4, the interleaved kappa order for nm = 2 mod 4), one and two 8-row tiles of b2 per warp
item, every b1-per-item variant, odd nb1 (the half-used b1 pair), ragged nb2 / nw, several b1 groups per q (C panel
larger than a stage), forced stage geometries, and the fused linewidth sum -- each element by element against the CPU
oracle, and against the plain DFMA kernel (tuning "rot_plain") on the same input.
Bar: max |out_gpu - out_oracle| <= 1e-10 * max(out_oracle)  (north_star, reading R10).
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
    a = dict(gW=wl.gW_full(w), Re=wl.Re_vectors(w), Rp=wl.Rp_vectors(w), k=wl.k_points(w)[ik], Uk=wl.U_k(w, ik),
             q=wl.q_points(w, ik), Ukq=wl.U_kq(w, ik), ev=wl.ph_eigvecs(w, ik), om=wl.omega(w, ik))
    a["eps_k"], a["eps_kq"] = wl.band_energies(w, ik)
    return a


#        nw nb1 nb2 nm  nq
CASES = [(5, 3, 4, nm, 37) for nm in (4, 5, 17, 21, 22, 25, 33, 37, 41, 48)] + \
        [(12, 5, 12, nm, 21) for nm in (3, 7, 12, 13, 20, 24, 28, 30, 36, 40, 44, 47)] + [
    (32, 5, 12, 30, 9),       # several b1 groups per q (C panel of a q > 64 KB), KS = 8
    (40, 9, 20, 12, 7),       # several groups, KS = 3 (b1 pairs), three 8-row tiles of b2 (odd: one clamped)
    (16, 16, 16, 12, 130),    # the 4-atom cell's shape
    (8, 4, 4, 6, 1100),       # the band-window shape, 8 q per stage, ragged last stage
    (8, 8, 8, 6, 700),        # the si-like shape: two items per q
    (9, 9, 3, 2, 900),        # KS = 1 with 8 b1 per item (+ one left over)
    (20, 4, 20, 3, 300),       # KS = 1, two m-tiles, 4 b1 per item
    (9, 2, 9, 8, 200),        # KS = 2, two m-tiles, 2 b1 per item, nm = 0 mod 8
    (7, 6, 7, 16, 100),       # KS = 4, 2 b1 per item
    (32, 32, 32, 30, 5),      # the large cell's shape: b1 groups, two rings
    (64, 3, 64, 6, 10),       # U_kq stages of 68 KB: three do not fit shared memory -> the plain kernel takes over
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "nw%d_nb%d_%d_nm%d" % c[:4])
def test_rotation_matches_oracle_and_plain_kernel(env, case):
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nw, nb1, nb2, nm, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=(2, 1, 1), grid_p=(1, 2, 1), nq=nq, cfg_id=120 + nm)
    a = _inputs(wl, w)
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=nq)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    out2 = ctx.q_batch(*d).cpu().numpy()
    ctx.set_tuning("rot_plain", 1)
    out1 = ctx.q_batch(*d).cpu().numpy()
    ctx.close()
    assert out2.shape == ref.shape
    assert _relerr(out2, ref) <= TOL
    assert _relerr(out1, ref) <= TOL
    assert _relerr(out2, out1) <= TOL


@pytest.mark.parametrize("knob", [{"rot_qg": 1}, {"rot_qg": 3}, {"rot_gb1": 2}, {"rot_gb1": 1}, {"rot_mtw": 1},
                                  {"rot_blk": 1}, {"rot_blk": 2}, {"rot_blk": 2, "rot_gb1": 2}, {"rot_blk": 2, "rot_qg": 3}],
                         ids=lambda k: "_".join("%s%d" % kv for kv in k.items()))
def test_rotation_forced_stage_geometry(env, knob):
    """q-points per stage, b1 per C stage (the two-ring form on a small problem) and m-tiles per item forced."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=12, nb1=5, nb2=12, nm=10, grid_e=(2, 1, 1), grid_p=(1, 2, 1), nq=333, cfg_id=119)
    a = _inputs(wl, w)
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=w.nq)
    for key, val in knob.items():
        ctx.set_tuning(key, val)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    out = ctx.q_batch(*d).cpu().numpy()
    again = ctx.q_batch(*d).cpu().numpy()
    ctx.close()
    assert _relerr(out, ref) <= TOL
    assert np.array_equal(out, again)


@pytest.mark.parametrize("case", [(12, 5, 12, 12, 150), (12, 5, 12, 30, 40), (40, 9, 20, 12, 7), (5, 3, 4, 21, 300)],
                         ids=lambda c: "nw%d_nb%d_%d_nm%d" % c[:4])
def test_rotation_fused_rates(env, case):
    """Eq. 29 linewidth sum inside the epilogue (two m-tiles per item, b1 pairs, several groups)."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nw, nb1, nb2, nm, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=(2, 1, 1), grid_p=(1, 2, 1), nq=nq, cfg_id=160 + nm)
    a = _inputs(wl, w)
    P = dict(wl.RATE_PARAMS)
    out_ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ref = np.zeros(nb1)
    oracle.rates(out_ref, a["eps_k"], a["eps_kq"], a["om"], P["kT"], P["mu"], P["sigma"], P["pref"], rate=ref)
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=nq)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    for store in (False, True):
        d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"], a["eps_k"], a["eps_kq"], np.zeros(nb1)])
        rate, out = ctx.q_batch_rates(*d, store_out=store, **P)
        assert _relerr(rate.cpu().numpy(), ref) <= TOL
        if store:
            assert _relerr(out.cpu().numpy(), out_ref) <= TOL
    ctx.close()
