"""GPU parity of the three-phonon coupling (Eq. 5, the second workload with the Eq. 70
shape, readings R25-R27): the same kernels under phoebe_elph_set_conventions(phase_sign=-1, all three eigenvector
matrices conjugated) against the independent oracle oracle.v3sq (a plain 7-deep loop over Eq. 5), element by element:
    max |out_gpu - out_oracle| <= 1e-10 * max(out_oracle)."""
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


CASES = [
    # nm  n0  n1  grid_R     grid_R'    nq
    (3, 3, 3, (3, 3, 1), (3, 2, 2), 70),          # one atom
    (6, 6, 6, (3, 2, 2), (2, 2, 3), 130),         # two atoms
    (6, 2, 5, (2, 2, 2), (3, 1, 2), 33),          # a window of modes at q and q'
    (12, 12, 12, (2, 2, 1), (2, 1, 2), 64),       # the 4-atom cell
    (51, 2, 2, (2, 1, 1), (1, 2, 1), 5),          # nm > 48: plain rotation path
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "nm%d_%d_%d_nq%d" % (c[0], c[1], c[2], c[5]))
@pytest.mark.parametrize("batch", [False, True], ids=["set_k", "set_k_batch"])
def test_three_phonon_matches_oracle(env, case, batch):
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nm, n0, n1, gR, gR2, nq = case
    w = wl.custom(nw=nm, nb1=n0, nb2=n1, nm=nm, grid_e=gR, grid_p=gR2, nk=2, nq=nq, cfg_id=20 + nm)
    V3, R, R2 = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
    qs = wl.k_points(w)
    zs = np.stack([wl.U_k(w, i) for i in range(2)])              # z_q [nm][n0] of two first-phonon wavevectors
    ctx = harness.make_context(w, torch.from_numpy(V3).cuda(), nq_max=nq, nk_max=2 if batch else 0)
    ctx.set_conventions(phase_sign=-1, conj_Uk=True, conj_Ukq=True, conj_ev=True)
    half = torch.full((nq, nm), 0.5, dtype=torch.float64, device="cuda")
    if batch:
        ctx.set_k_batch(qs[:2], harness.to_device([zs])[0])
    for i in ((1, 0) if batch else (0,)):
        if batch:
            ctx.select_k(i)
        else:
            ctx.set_k(qs[i], harness.to_device([zs[i]])[0])
        q1, z1, z2, _ = wl.q_inputs(w, i)
        ref = oracle.v3sq(V3, R, R2, qs[i], zs[i], q1, z1, z2)
        out = ctx.q_batch(*harness.to_device([q1, z1, z2]), half).cpu().numpy()
        assert out.shape == ref.shape == (nq, n0, n1, nm)
        assert _relerr(out, ref) <= TOL
    ctx.close()


def test_conventions_switch_back_and_errors(env):
    wl, oracle, torch, harness, binding = env["wl"], env["oracle"], env["torch"], env["harness"], env["binding"]
    w = wl.custom(nw=6, nb1=4, nb2=5, nm=6, grid_e=(3, 2, 1), grid_p=(2, 2, 2), nq=40, cfg_id=29)
    gW, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
    k, Uk = wl.k_points(w)[0], wl.U_k(w)
    q, Ukq, ev, om = wl.q_inputs(w)
    ctx = harness.make_context(w, torch.from_numpy(gW).cuda(), nq_max=40)
    d = harness.to_device([q, Ukq, ev, om])
    ctx.set_k(k, harness.to_device([Uk])[0])
    ctx.set_conventions(-1, True, True, True)
    with pytest.raises(binding.PhoebeElphError) as e:              # the g1' of the other conventions is not reused
        ctx.q_batch(*d)
    assert e.value.code == -4
    # every flag on its own, against the el-ph oracle with the correspondingly transformed inputs
    for sign, cu, cq, cz in [(-1, False, True, False), (1, True, True, False), (1, False, False, False), (1, False, True, True)]:
        ctx.set_conventions(sign, cu, cq, cz)
        ctx.set_k(k, harness.to_device([Uk])[0])
        out = ctx.q_batch(*d).cpu().numpy()
        ref = oracle.elph(gW, Re, Rp, None, None, sign * k, Uk.conj() if cu else Uk, sign * q,
                          Ukq if cq else Ukq.conj(), ev.conj() if cz else ev, om)
        assert _relerr(out, ref) <= TOL
    ctx.set_conventions()                                          # defaults again
    ctx.set_k(k, harness.to_device([Uk])[0])
    out = ctx.q_batch(*d).cpu().numpy()
    assert _relerr(out, oracle.elph(gW, Re, Rp, None, None, k, Uk, q, Ukq, ev, om)) <= TOL
    with pytest.raises(binding.PhoebeElphError) as e:
        ctx.set_conventions(phase_sign=0)
    assert e.value.code == -2
    pol = wl.polar_inputs(w, h=1)
    ctx.set_polar(**pol)
    with pytest.raises(binding.PhoebeElphError) as e:              # polar term belongs to the el-ph conventions
        ctx.set_conventions(-1, True, True, True)
    assert e.value.code == -2
    ctx.close()
