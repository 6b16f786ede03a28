"""GPU parity of the q <-> -q fold of step a4 (qfold.cuh): q lists that contain -q with q are contracted once per pair,
C(+-q) = Ce +- Co with Ce / Co the sums over the cosine / sine rows of the pair form.  The pairs are found on the device.
Against the CPU oracle (which knows nothing of it) and against the plain path (tuning "qfold" = 0): uniform meshes with
their self-inverse points (q = 0, zone boundary), lists with only some pairs, too few pairs (plain path taken), duplicated
q-points, -q only modulo a reciprocal lattice vector, non-integer lattice vectors (pairs only for the literal -q), fused
linewidths and the polar term on top.  Bar: max |d out| <= 1e-10 max(out)  (north_star, reading R10)."""
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


def _mesh(n):
    i = np.arange(n ** 3)
    return np.stack([i // (n * n), (i // n) % n, i % n], axis=1).astype(np.float64) / n


def _q_lists(rng):
    mesh8 = _mesh(8)                                             # 512 points, 8 self-inverse (components in {0, 1/2})
    r = rng.random((300, 3))
    some = np.concatenate([r, 1.0 - r[:200], rng.random((100, 3))])          # 200 pairs modulo G, 200 singles
    some = some[rng.permutation(len(some))]
    few = np.concatenate([rng.random((500, 3)), -rng.random((20, 3))])       # no pairs at all
    few[510] = -few[3]                                                         # ... but one
    dup = np.concatenate([mesh8, mesh8[100:200], mesh8[37:38]])                # 101 duplicates: each its own representative
    r20 = rng.integers(1, 1 << 20, (150, 3)) / float(1 << 20)                  # 20-bit fractions: G - q is exact
    shifted = np.concatenate([r20, np.array([3.0, -2.0, 1.0]) - r20])          # -q + G with G != (1,1,1)
    return {"mesh8": (mesh8, 260), "some_pairs": (some, 400), "few_pairs": (few, 0), "duplicates": (dup, 361),
            "shifted": (shifted, 150)}


@pytest.mark.parametrize("name", ["mesh8", "some_pairs", "few_pairs", "duplicates", "shifted"])
def test_qfold_matches_oracle_and_plain_path(env, name):
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    q, reps = _q_lists(np.random.default_rng(3))[name]
    nq = len(q)
    w = wl.custom(nw=6, nb1=5, nb2=6, nm=6, grid_e=(2, 2, 1), grid_p=(3, 3, 3), nq=nq, cfg_id=190)
    gW_np, Re, Rp, k, Uk = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)[0], wl.U_k(w)
    _, Ukq, ev, om = wl.q_inputs(w)
    ref = oracle.elph(gW_np, Re, Rp, None, None, k, Uk, q, Ukq, ev, om)
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=nq)
    ctx.set_tuning("tile", 64)
    ctx.set_tuning("qfold", 1)
    ctx.set_k(k, harness.to_device([Uk])[0])
    d = harness.to_device([q, Ukq, ev, om])
    out = ctx.q_batch(*d).cpu().numpy()
    got_reps = ctx.get_tuning("qfold_reps")
    again = ctx.q_batch(*d).cpu().numpy()
    ctx.set_tuning("qfold", 0)
    plain = ctx.q_batch(*d).cpu().numpy()
    assert ctx.get_tuning("qfold_reps") == 0
    ctx.close()
    if reps is not None:
        assert got_reps == reps, got_reps
    else:
        assert 0 < got_reps < nq
    assert _relerr(out, ref) <= TOL and _relerr(plain, ref) <= TOL
    assert np.array_equal(out, again)
    assert _relerr(out, plain) <= 1e-12


def test_qfold_non_integer_lattice_vectors_pair_only_the_literal_negative(env):
    """With non-integer Rp the phases are not periodic in q: only q' = -q exactly is a pair, q' = 1 - q is not."""
    wl, oracle, torch, binding, harness = env["wl"], env["oracle"], env["torch"], env["binding"], env["harness"]
    rng = np.random.default_rng(5)
    nRe, nw, nb, nm = 3, 4, 4, 6
    half = rng.uniform(-2.0, 2.0, (6, 3))
    Rp = np.concatenate([half, np.zeros((1, 3)), -half])
    Re = rng.uniform(-1.0, 1.0, (nRe, 3))
    gW = rng.standard_normal((len(Rp), nRe, nw, nw, nm)) + 1j * rng.standard_normal((len(Rp), nRe, nw, nw, nm))
    r = rng.random((200, 3))
    q = np.concatenate([r, -r[:120], 1.0 - r[120:200]])           # 120 literal pairs, 80 that are pairs only modulo G
    nq = len(q)
    w = wl.custom(nw=nw, nb1=nb, nb2=nb, nm=nm, grid_e=(nRe, 1, 1), grid_p=(len(Rp), 1, 1), nq=nq, cfg_id=191)
    k, Uk = wl.k_points(w)[0], wl.U_k(w)
    _, Ukq, ev, om = wl.q_inputs(w)
    ref = oracle.elph(gW, Re, Rp, None, None, k, Uk, q, Ukq, ev, om)
    ctx = binding.ElphContext(torch.from_numpy(gW).cuda(), Re, Rp, None, None, nb1_max=nb, nb2_max=nb, nq_max=nq)
    ctx.set_tuning("tile", 64)
    ctx.set_tuning("pair", 2)             # 13 vectors: too short a list for the pair form to be chosen by itself
    ctx.set_tuning("qfold", 1)
    ctx.set_k(k, harness.to_device([Uk])[0])
    out = ctx.q_batch(*harness.to_device([q, Ukq, ev, om])).cpu().numpy()
    assert ctx.get_tuning("qfold_reps") == nq - 120
    ctx.close()
    assert _relerr(out, ref) <= TOL


def test_qfold_with_rates_and_polar(env):
    """The fold sits in front of the rotation kernel: fused linewidths and the polar term see the same C."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    q = _mesh(8)
    w = wl.custom(nw=6, nb1=4, nb2=5, nm=6, grid_e=(2, 2, 1), grid_p=(3, 3, 1), nq=len(q), cfg_id=192)
    gW_np, Re, Rp, k, Uk = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)[0], wl.U_k(w)
    _, Ukq, ev, om = wl.q_inputs(w)
    eps_k, eps_kq = wl.band_energies(w)
    P = dict(wl.RATE_PARAMS)
    ref = oracle.elph(gW_np, Re, Rp, None, None, k, Uk, q, Ukq, ev, om)
    rref = oracle.rates(ref, eps_k, eps_kq, om, P["kT"], P["mu"], P["sigma"], P["pref"])
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=len(q))
    ctx.set_tuning("tile", 64)
    ctx.set_tuning("pair", 2)             # 9 vectors: too short a list for the pair form to be chosen by itself
    ctx.set_tuning("qfold", 1)
    ctx.set_k(k, harness.to_device([Uk])[0])
    d = harness.to_device([q, Ukq, ev, om, eps_k, eps_kq, np.zeros(w.nb1)])
    rate, out = ctx.q_batch_rates(*d, store_out=True, **P)
    assert ctx.get_tuning("qfold_reps") == 260
    assert _relerr(out.cpu().numpy(), ref) <= TOL and _relerr(rate.cpu().numpy(), rref) <= TOL
    pol = wl.polar_inputs(w)
    ctx.set_polar(**pol)
    Pq = oracle.polar_amplitude(q, ev, pol["recip"], pol["G"], pol["Zstar"], pol["eps_inf"], pol["coeff"])
    g1_ref = oracle.setk(gW_np, Re, None, k, Uk)
    pref = oracle.qbatch_polar(g1_ref, Rp, None, q, Ukq, ev, om, Uk, Pq)
    outp = ctx.q_batch(*d[:4]).cpu().numpy()
    assert ctx.get_tuning("qfold_reps") == 260
    ctx.close()
    assert _relerr(outp, pref) <= TOL
