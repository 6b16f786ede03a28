"""GPU parity of the polar long-range term (Eq. 14-15, readings R20-R24): phoebe_elph_set_polar
followed by q_batch / q_batch_rates against the CPU oracle (oracle.polar_amplitude -> oracle.qbatch_polar) on the same
seeded inputs, to the north-star bar  max |out_gpu - out_oracle| <= 1e-10 * max(out_oracle)."""
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


def _case(wl, w, ik=0):
    return dict(gW=wl.gW_full(w), Re=wl.Re_vectors(w), Rp=wl.Rp_vectors(w), k=wl.k_points(w)[ik], Uk=wl.U_k(w, ik),
                q=wl.q_points(w, ik), Ukq=wl.U_kq(w, ik), ev=wl.ph_eigvecs(w, ik), om=wl.omega(w, ik))


def _oracle(oracle, a, pol, Uk=None, sl=slice(None)):
    Uk = a["Uk"] if Uk is None else Uk
    g1 = oracle.setk(a["gW"], a["Re"], None, a["k"], Uk)
    P = oracle.polar_amplitude(a["q"][sl], a["ev"][sl], pol["recip"], pol["G"], pol["Zstar"], pol["eps_inf"], pol["coeff"])
    return oracle.qbatch_polar(g1, a["Rp"], None, a["q"][sl], np.ascontiguousarray(a["Ukq"][sl]),
                               np.ascontiguousarray(a["ev"][sl]), a["om"][sl], Uk, P)


CASES = [
    # nw nb1 nb2 nm  grid_e     grid_p     nq
    (2, 2, 2, 3, (3, 3, 3), (3, 3, 3), 64),        # the tiny config's shape
    (3, 2, 1, 3, (5, 1, 1), (7, 1, 1), 1),
    (5, 4, 3, 6, (3, 3, 2), (2, 5, 3), 257),       # several q per CTA, ragged last CTA
    (8, 4, 4, 6, (3, 3, 3), (3, 3, 3), 700),       # band-window shape (rectangular U)
    (7, 7, 7, 15, (2, 2, 1), (2, 3, 1), 40),       # NT = 2, nb2 % 8 != 0
    (9, 9, 9, 30, (2, 1, 1), (3, 1, 1), 20),       # NT = 4 (the "large" cell's mode count)
    (16, 16, 16, 12, (2, 2, 1), (2, 2, 2), 300),   # the 4-atom cell's band / mode counts
    (2, 2, 2, 51, (2, 1, 1), (2, 1, 1), 70),       # nm > 48: plain rotation path
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "nw%d_nb%d_%d_nm%d_nq%d" % (c[0], c[1], c[2], c[3], c[6]))
def test_polar_matches_oracle(env, case):
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nw, nb1, nb2, nm, ge, gp, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=ge, grid_p=gp, nq=nq, cfg_id=30 + nw)
    a, pol = _case(wl, w), wl.polar_inputs(w)
    ref = _oracle(oracle, a, pol)
    plain = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    assert _relerr(ref, plain) > 1e-2               # the recipe's long-range term is not negligible
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=nq)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
    ctx.set_polar(**pol)
    out = ctx.q_batch(*d).cpu().numpy()
    assert _relerr(out, ref) <= TOL
    assert ctx.launch_counts()["polar"] == 1
    ctx.set_polar()                                 # off again: the short-range result is back
    out = ctx.q_batch(*d).cpu().numpy()
    assert _relerr(out, plain) <= TOL
    assert ctx.launch_counts()["polar"] == 1
    ctx.close()


def test_polar_with_k_batch_sub_batches_rates_and_host(env):
    """The overlap uses the U_k of the SELECTED k slot; internal q sub-batches; the fused linewidths and the host entry
    points see the same amplitudes."""
    wl, oracle, torch, harness, binding = env["wl"], env["oracle"], env["torch"], env["harness"], env["binding"]
    w = wl.custom(nw=6, nb1=5, nb2=6, nm=9, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nk=3, nq=300, cfg_id=37)
    pol = wl.polar_inputs(w, h=1)
    gW_np, ks = wl.gW_full(w), wl.k_points(w)
    Uks = np.stack([wl.U_k(w, ik) for ik in range(3)])
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=300, nk_max=3)
    ctx.set_tuning("nq_sub", 128)
    ctx.set_polar(**pol)
    ctx.set_k_batch(ks, harness.to_device([Uks])[0])
    P = dict(wl.RATE_PARAMS)
    for ik in (2, 0, 1):
        a = _case(wl, w, ik)
        a["k"] = ks[ik]
        ref = _oracle(oracle, a, pol, Uk=Uks[ik])
        ctx.select_k(ik)
        d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
        assert _relerr(ctx.q_batch(*d).cpu().numpy(), ref) <= TOL
        eps_k, eps_kq = wl.band_energies(w, ik)
        want = oracle.rates(ref, eps_k, eps_kq, a["om"], P["kT"], P["mu"], P["sigma"], P["pref"])
        rate = torch.zeros(5, dtype=torch.float64, device="cuda")
        ctx.q_batch_rates(*d, *harness.to_device([eps_k, eps_kq]), rate, **P)
        assert _relerr(rate.cpu().numpy(), want) <= TOL
        out = np.empty((300, 5, 6, 9))
        ctx.q_batch_host(a["q"], a["Ukq"], a["ev"], a["om"], out)
        assert _relerr(out, ref) <= TOL
    assert ctx.launch_counts()["polar"] == 3 * 3 * 3
    # host set_k after the batch: slot 0 again
    a = _case(wl, w, 1)
    ctx.set_k_host(ks[1], Uks[1])
    out = np.empty((300, 5, 6, 9))
    ctx.q_batch_host(a["q"], a["Ukq"], a["ev"], a["om"], out)
    a["k"] = ks[1]
    assert _relerr(out, _oracle(oracle, a, pol, Uk=Uks[1])) <= TOL
    # errors
    with pytest.raises(binding.PhoebeElphError) as e:
        ctx.set_polar(pol["recip"], np.zeros((5000, 3)), pol["Zstar"], pol["eps_inf"], 1.0)
    assert e.value.code == -2
    ctx.close()
    w2 = wl.custom(nw=2, nm=4, grid_e=(2, 1, 1), nq=4, cfg_id=38)
    ctx = harness.make_context(w2, torch.from_numpy(wl.gW_full(w2)).cuda(), nq_max=4)
    with pytest.raises(binding.PhoebeElphError) as e:      # nmodes not a multiple of 3
        ctx._check(ctx._lib.phoebe_elph_set_polar(ctx._ctx, pol["recip"].ctypes.data, 1, pol["G"].ctypes.data,
                                                  pol["Zstar"].ctypes.data, pol["eps_inf"].ctypes.data, 1.0), "set_polar")
    assert e.value.code == -2
    ctx.close()


def test_polar_q_equal_minus_G_is_skipped(env):
    """R23: at q = 0 (and at q = -G for a G of the list) the singular term is left out and the result is finite."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=3, nb1=3, nb2=3, nm=6, grid_e=(2, 2, 1), grid_p=(2, 2, 1), nq=8, cfg_id=39)
    a, pol = _case(wl, w), wl.polar_inputs(w, h=1)
    a["q"] = a["q"].copy(); a["q"][0] = 0.0; a["q"][5] = [1.0, -1.0, 0.0]
    ref = _oracle(oracle, a, pol)
    assert np.all(np.isfinite(ref))
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=8)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    ctx.set_polar(**pol)
    out = ctx.q_batch(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])).cpu().numpy()
    assert _relerr(out, ref) <= TOL
    ctx.close()
