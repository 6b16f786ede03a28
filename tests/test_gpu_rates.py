"""GPU parity of the fused linewidth accumulation (Eq. 29 L229 + Eq. 61):
phoebe_elph_q_batch_rates against the CPU oracle (oracle.elph -> oracle.rates) on the same seeded inputs.

Bar: max_b1 |rate_gpu - rate_oracle| <= 1e-10 * max_b1 |rate_oracle|  (the north-star tolerance carried through the
linear sum; derivation in DESIGN.md "Tolerance"), and |g|^2, when also stored, to the bar of test_gpu_parity.py.
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


def _case(wl, w, ik=0):
    a = dict(gW=wl.gW_full(w), Re=wl.Re_vectors(w), Rp=wl.Rp_vectors(w), k=wl.k_points(w)[ik], Uk=wl.U_k(w, ik),
             q=wl.q_points(w, ik), Ukq=wl.U_kq(w, ik), ev=wl.ph_eigvecs(w, ik), om=wl.omega(w, ik))
    a["eps_k"], a["eps_kq"] = wl.band_energies(w, ik)
    return a


def _oracle_rates(oracle, a, P, rate0=None, om=None):
    om = a["om"] if om is None else om
    out = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], om)
    rate = np.zeros(a["Uk"].shape[1]) if rate0 is None else rate0.copy()
    oracle.rates(out, a["eps_k"], a["eps_kq"], om, P["kT"], P["mu"], P["sigma"], P["pref"], rate=rate)
    return rate, out


CASES = [
    # nw nb1 nb2 nm  grid_e     grid_p     nq
    (2, 2, 2, 3, (3, 3, 3), (3, 3, 3), 64),        # the tiny config's shape
    (3, 2, 1, 2, (5, 1, 1), (7, 1, 1), 1),
    (5, 4, 3, 6, (3, 3, 2), (2, 5, 3), 257),       # several q per CTA, ragged last CTA
    (8, 4, 4, 6, (3, 3, 3), (3, 3, 3), 700),       # band-window shape
    (7, 7, 7, 15, (2, 2, 1), (2, 3, 1), 40),       # NT = 2, nb2 % 8 != 0
    (9, 9, 9, 30, (2, 1, 1), (3, 1, 1), 20),       # NT = 4 (the "large" cell's mode count)
    (16, 16, 16, 12, (2, 2, 1), (2, 2, 2), 300),   # the 4-atom cell's band / mode counts (two 8-row b2 tiles)
    (2, 2, 2, 51, (2, 1, 1), (2, 1, 1), 70),       # nm > 48: plain rotation path + stand-alone rate sum
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "nw%d_nb%d_%d_nm%d_nq%d" % (c[0], c[1], c[2], c[3], c[6]))
@pytest.mark.parametrize("store", [False, True], ids=["rates_only", "rates_and_out"])
def test_rates_match_oracle(env, case, store):
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nw, nb1, nb2, nm, ge, gp, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=ge, grid_p=gp, nq=nq, cfg_id=90 + nw)
    a = _case(wl, w)
    P = dict(wl.RATE_PARAMS)
    inc, out_ref = _oracle_rates(oracle, a, P)
    rate0 = inc[::-1] * np.linspace(0.3, 0.7, nb1)  # accumulated INTO: start from a non-zero array of the same scale
    ref = rate0 + inc
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=nq)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"], a["eps_k"], a["eps_kq"], rate0])
    rate, out = ctx.q_batch_rates(*d, store_out=store, **P)
    rate = rate.cpu().numpy()
    assert _relerr(rate - rate0, ref - rate0) <= TOL
    if store:
        assert _relerr(out.cpu().numpy(), out_ref) <= TOL
    else:
        assert out is None
    n = ctx.launch_counts()
    assert n["rate_reduce"] == 1
    ctx.close()


def test_rates_sub_batches_accumulate_and_are_reproducible(env):
    """Several internal q sub-batches and several calls accumulate into the same array (RP5 on the GPU); omega <= 0
    contributes nothing (R18); two runs give bit-identical sums (fixed summation order)."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=4, nb1=3, nb2=4, nm=3, grid_e=(3, 3, 3), nq=300, cfg_id=95)
    a = _case(wl, w)
    om = a["om"].copy(); om[5, 1] = 0.0; om[299, 2] = -0.3
    P = dict(wl.RATE_PARAMS)
    ref, _ = _oracle_rates(oracle, a, P, om=om)
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=300)
    ctx.set_tuning("nq_sub", 128)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    q_d, U_d, z_d, w_d, e1_d, e2_d = harness.to_device([a["q"], a["Ukq"], a["ev"], om, a["eps_k"], a["eps_kq"]])
    runs = []
    for _ in range(2):
        rate = torch.zeros(3, dtype=torch.float64, device="cuda")
        ctx.q_batch_rates(q_d, U_d, z_d, w_d, e1_d, e2_d, rate, **P)
        runs.append(rate.cpu().numpy())
    assert _relerr(runs[0], ref) <= TOL
    assert np.array_equal(runs[0], runs[1])
    # two calls on halves of the q list == one call
    rate = torch.zeros(3, dtype=torch.float64, device="cuda")
    for sl in (slice(0, 170), slice(170, 300)):
        ctx.q_batch_rates(q_d[sl].contiguous(), U_d[sl].contiguous(), z_d[sl].contiguous(), w_d[sl].contiguous(), e1_d,
                          e2_d[sl].contiguous(), rate, **P)
    assert _relerr(rate.cpu().numpy(), ref) <= TOL
    assert ctx.launch_counts()["rate_reduce"] == 3 + 3 + 2 + 2
    ctx.close()


def test_rates_host_entry_point_and_errors(env):
    wl, oracle, torch, harness, binding = env["wl"], env["oracle"], env["torch"], env["harness"], env["binding"]
    w = wl.custom(nw=6, nb1=5, nb2=6, nm=9, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nq=150, cfg_id=96)
    a = _case(wl, w)
    P = dict(kT=0.01, mu=0.03, sigma=0.02, pref=0.7)
    ref, out_ref = _oracle_rates(oracle, a, P)
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=150)
    ctx.set_k_host(a["k"], a["Uk"])
    rate = np.zeros(5)
    ctx.q_batch_rates_host(a["q"], a["Ukq"], a["ev"], a["om"], a["eps_k"], a["eps_kq"], rate, **P)
    assert _relerr(rate, ref) <= TOL
    rate2, out = np.zeros(5), np.empty((150, 5, 6, 9))
    ctx.q_batch_rates_host(a["q"], a["Ukq"], a["ev"], a["om"], a["eps_k"], a["eps_kq"], rate2, out=out, **P)
    assert np.array_equal(rate2, rate)
    assert _relerr(out, out_ref) <= TOL
    for bad in (dict(P, kT=0.0), dict(P, sigma=-1.0)):
        with pytest.raises(binding.PhoebeElphError) as e:
            ctx.q_batch_rates_host(a["q"], a["Ukq"], a["ev"], a["om"], a["eps_k"], a["eps_kq"], rate, **bad)
        assert e.value.code == -2
    ctx.close()


def test_rates_si_like_full(env):
    """BASELINE.json configs[1] with the recipe's band energies: all 4096 q, linewidth of the 8 bands."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.CONFIGS["si-like"]
    a = _case(wl, w)
    P = dict(wl.RATE_PARAMS)
    ref, _ = _oracle_rates(oracle, a, P)
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda())
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    rate = torch.zeros(w.nb1, dtype=torch.float64, device="cuda")
    ctx.q_batch_rates(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"], a["eps_k"], a["eps_kq"]]), rate, **P)
    assert np.all(ref > 0)
    assert _relerr(rate.cpu().numpy(), ref) <= TOL
    ctx.close()


def test_rates_async_pipelined_host_batches(env):
    """q_batch_rates_host_async: several k-points in flight over the two staging slots, one rate array per call, mixed
    with q_batch_host_async; rates (and |g|^2 where asked for) against the oracle after wait()."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nk=3, nq=210, cfg_id=97)
    gW_np, Re, Rp, ks = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=210, nk_max=3)
    Uks = np.stack([wl.U_k(w, ik) for ik in range(3)])
    P = dict(wl.RATE_PARAMS)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    ins, eps, refs, rref = [], [], [], []
    for ik in range(3):
        a = _case(wl, w, ik)
        ins.append([pin(a[n]) for n in ("q", "Ukq", "ev", "om")])
        eps.append([pin(a["eps_k"]), pin(a["eps_kq"])])
        out = oracle.elph(gW_np, Re, Rp, None, None, ks[ik], Uks[ik], a["q"], a["Ukq"], a["ev"], a["om"])
        refs.append(out)
        rref.append(oracle.rates(out, a["eps_k"], a["eps_kq"], a["om"], P["kT"], P["mu"], P["sigma"], P["pref"]))
    rates = torch.zeros((3, 4), dtype=torch.float64).pin_memory()
    outs = [torch.empty((210, 4, 5, 6), dtype=torch.float64).pin_memory() for _ in range(3)]
    plain = torch.empty((210, 4, 5, 6), dtype=torch.float64).pin_memory()
    for rep in range(2):
        rates.zero_()
        ctx.set_k_batch_host(ks, Uks)
        for ik in (0, 1, 2):
            ctx.select_k(ik)
            ctx.q_batch_rates_host_async(*[t.numpy() for t in ins[ik]], eps[ik][0].numpy(), eps[ik][1].numpy(),
                                         rates[ik].numpy(), out=outs[ik].numpy() if ik == 1 else None, **P)
            if ik == 1:
                ctx.q_batch_host_async(*[t.numpy() for t in ins[ik]], plain.numpy())
        ctx.wait()
        for ik in range(3):
            assert _relerr(rates[ik].numpy(), rref[ik]) <= TOL
        assert _relerr(outs[1].numpy(), refs[1]) <= TOL and _relerr(plain.numpy(), refs[1]) <= TOL
    ctx.close()


@pytest.mark.parametrize("shape", [(8, 4, 4, 6, 192, {}), (12, 5, 12, 12, 128, {}), (5, 3, 4, 21, 64, {"rot_qg": 1}),
                                   (8, 4, 4, 6, 192, {"rot_qg": 5})],
                         ids=["band_window_shape", "two_m_tiles", "one_q_per_stage", "qg_not_dividing"])
def test_rates_multi_equals_oracle_per_k(env, shape):
    """phoebe_elph_q_batch_rates_multi: the q lists of all k slots of a set_k_batch stacked into one pass; every k slot's
    linewidths (and |g|^2 when stored) against the oracle, and against per-k q_batch_rates calls."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nw, nb1, nb2, nm, nq, knobs = shape
    nk = 3
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=(2, 2, 1), grid_p=(2, 1, 2), nk=nk, nq=nq, cfg_id=97)
    P = dict(wl.RATE_PARAMS)
    cases = [_case(wl, w, ik) for ik in range(nk)]
    gW_np = cases[0]["gW"]
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=nk * nq, nk_max=nk)
    for key, val in knobs.items():
        ctx.set_tuning(key, val)
    ks = wl.k_points(w)
    Uks = np.stack([c["Uk"] for c in cases])
    ctx.set_k_batch(ks, harness.to_device([Uks])[0])
    st = lambda key: np.ascontiguousarray(np.stack([c[key] for c in cases]))
    d = harness.to_device([st("q"), st("Ukq"), st("ev"), st("om"), st("eps_k"), st("eps_kq")])
    rate0 = np.linspace(0.1, 0.2, nk * nb1).reshape(nk, nb1) * 1e-3
    (rate_d,) = harness.to_device([rate0])
    rate, out = ctx.q_batch_rates_multi(*d, rate_d, store_out=True, **P)
    rate, out = rate.cpu().numpy(), out.cpu().numpy()
    # rates only (|g|^2 never stored) gives the same sums bit for bit
    (rate2_d,) = harness.to_device([rate0])
    ctx.q_batch_rates_multi(*d, rate2_d, **P)
    assert np.array_equal(rate2_d.cpu().numpy(), rate)
    for ik, c in enumerate(cases):
        ref, out_ref = _oracle_rates(oracle, c, P)
        assert _relerr(rate[ik] - rate0[ik], ref) <= TOL
        assert _relerr(out[ik], out_ref) <= TOL
        ctx.select_k(ik)
        dk = harness.to_device([c["q"], c["Ukq"], c["ev"], c["om"], c["eps_k"], c["eps_kq"], np.zeros(nb1)])
        rk, _ = ctx.q_batch_rates(*dk, **P)
        assert _relerr(rk.cpu().numpy(), ref) <= TOL
    ctx.close()


def test_stacked_host_async_pipelines_k_batches(env):
    """phoebe_elph_q_batch_multi_host_async / _rates_multi_host_async: four k batches of three k-points each, the
    k-stacked pinned arrays of a batch per call, batches pipelined over the two staging slots with the NEXT
    set_k_batch_host issued while the previous batch's results are still being copied out; |g|^2 and linewidths of
    every (batch, k) against the oracle after wait()."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nk, nbatch, nq = 3, 4, 128
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nk=nk * nbatch, nq=nq, cfg_id=98)
    gW_np, ks = wl.gW_full(w), wl.k_points(w)
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=nk * nq, nk_max=nk)
    P = dict(wl.RATE_PARAMS)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    cases = [_case(wl, w, ik) for ik in range(nk * nbatch)]
    st = lambda b, key: pin(np.stack([cases[b * nk + j][key] for j in range(nk)]))
    held = []
    for b in range(nbatch):
        Uks = np.stack([cases[b * nk + j]["Uk"] for j in range(nk)])
        ctx.set_k_batch_host(ks[b * nk:(b + 1) * nk], Uks)
        ins = [st(b, key) for key in ("q", "Ukq", "ev", "om")]
        out = torch.empty((nk, nq, w.nb1, w.nb2, w.nm), dtype=torch.float64).pin_memory()
        if b % 2 == 0:
            ctx.q_batch_multi_host_async(*[t.numpy() for t in ins], out.numpy())
            held.append((b, ins, out, None))
        else:
            eps = [st(b, "eps_k"), st(b, "eps_kq")]
            rate = torch.zeros((nk, w.nb1), dtype=torch.float64).pin_memory()
            ctx.q_batch_rates_multi_host_async(*[t.numpy() for t in ins], eps[0].numpy(), eps[1].numpy(), rate.numpy(),
                                               out=out.numpy() if b == 1 else None, **P)
            held.append((b, ins + eps, out if b == 1 else None, rate))
    ctx.wait()
    for b, _, out, rate in held:
        for j in range(nk):
            rref, oref = _oracle_rates(oracle, cases[b * nk + j], P)
            if out is not None:
                assert _relerr(out.numpy()[j], oref) <= TOL
            if rate is not None:
                assert _relerr(rate.numpy()[j], rref) <= TOL
    ctx.close()


def test_rates_async_copy_out_outlasts_copy_in(env):
    """Six pipelined q_batch_rates_host_async batches WITH |g|^2 copied out (3 MB per batch against 0.3 MB copied in):
    the copy-out of batch n-2 is still running when the inputs of batch n arrive.  Each call has its own initial rate
    values; a copy-in that overtook the copy-out of the rate staging buffer would hand back the wrong batch's sums."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=8, nb1=8, nb2=8, nm=6, grid_e=(2, 2, 1), grid_p=(3, 3, 1), nk=1, nq=1024, cfg_id=99)
    a = _case(wl, w, 0)
    P = dict(wl.RATE_PARAMS)
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=w.nq)
    ctx.set_k_host(a["k"], a["Uk"])
    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
    ins = [pin(a[key]) for key in ("q", "Ukq", "ev", "om", "eps_k", "eps_kq")]
    rref, oref = _oracle_rates(oracle, a, P)
    held = []
    for n in range(6):
        rate = pin(np.full(w.nb1, 1e-3 * (n + 1)))
        out = torch.empty((w.nq, w.nb1, w.nb2, w.nm), dtype=torch.float64).pin_memory()
        ctx.q_batch_rates_host_async(*[t.numpy() for t in ins], rate.numpy(), out=out.numpy(), **P)
        held.append((n, rate, out))
    ctx.wait()
    for n, rate, out in held:
        assert _relerr(rate.numpy() - 1e-3 * (n + 1), rref) <= 1e-9
        assert _relerr(out.numpy(), oref) <= TOL
    ctx.close()
