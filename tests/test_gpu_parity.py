"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by
element, on the same seeded inputs.  Bar (BASELINE.json north_star, reading R10):
    max |out_gpu - out_oracle| <= 1e-10 * max(out_oracle)
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


def _run_gpu(env, w, gW_np, k, Uk, q, Ukq, ev, om, deg_e=None, deg_p=None, nq_max=None, host=False):
    torch, harness = env["torch"], env["harness"]
    gW = torch.from_numpy(gW_np).cuda()
    ctx = harness.make_context(w, gW, nq_max=nq_max or len(q), deg_e=deg_e, deg_p=deg_p)
    if host:
        ctx.set_k_host(k, Uk)
        out = np.empty((len(q), Uk.shape[1], Ukq.shape[2], w.nm))
        ctx.q_batch_host(q, Ukq, ev, om, out)
        g1 = ctx.copy_g1().cpu().numpy()
    else:
        (Uk_d,) = harness.to_device([Uk])
        ctx.set_k(k, Uk_d)
        q_d, Ukq_d, ev_d, om_d = harness.to_device([q, Ukq, ev, om])
        out = ctx.q_batch(q_d, Ukq_d, ev_d, om_d).cpu().numpy()
        g1 = ctx.copy_g1().cpu().numpy()
    torch.cuda.synchronize()
    ctx.close()
    return out, g1


def _inputs(wl, w, ik=0):
    return dict(gW=wl.gW_full(w), Re=wl.Re_vectors(w), Rp=wl.Rp_vectors(w), k=wl.k_points(w)[ik], Uk=wl.U_k(w, ik),
                q=wl.q_points(w, ik), Ukq=wl.U_kq(w, ik), ev=wl.ph_eigvecs(w, ik), om=wl.omega(w, ik))


def test_tiny_full(env):
    wl, oracle = env["wl"], env["oracle"]
    w = wl.CONFIGS["tiny"]
    a = _inputs(wl, w)
    out, g1 = _run_gpu(env, w, a["gW"], a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    g1_ref = oracle.setk(a["gW"], a["Re"], None, a["k"], a["Uk"])
    assert _relerr(g1, g1_ref) < 1e-12
    ref = oracle.qbatch(g1_ref, a["Rp"], None, a["q"], a["Ukq"], a["ev"], a["om"])
    assert out.shape == ref.shape == (64, 2, 2, 3)
    assert _relerr(out, ref) <= TOL
    # and against the un-factorised double sum on a few q
    d = oracle.direct(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"][:4], a["Ukq"][:4], a["ev"][:4],
                      a["om"][:4])
    assert _relerr(out[:4], d) <= TOL


RAGGED = [
    # nw nb1 nb2 nm  grid_e     grid_p     nq
    (3, 2, 1, 2, (5, 1, 1), (7, 1, 1), 1),
    (3, 3, 2, 3, (1, 2, 3), (3, 3, 1), 130),
    (4, 1, 4, 1, (2, 2, 2), (1, 1, 1), 65),
    (5, 4, 3, 6, (3, 3, 2), (2, 5, 3), 257),
    (1, 1, 1, 1, (1, 1, 1), (1, 1, 2), 3),
    (8, 4, 4, 6, (3, 3, 3), (3, 3, 3), 200),
    (6, 6, 5, 9, (4, 3, 2), (3, 2, 5), 96),
    (7, 7, 7, 15, (2, 2, 1), (2, 3, 1), 40),      # NT = 2, nw % 4 = 3
    (9, 9, 10 - 1, 30, (2, 1, 1), (3, 1, 1), 20),  # NT = 4 (the "large" cell's mode count)
    (3, 3, 3, 45, (2, 1, 1), (1, 2, 1), 6),       # NT = 6
    (2, 2, 2, 51, (2, 1, 1), (2, 1, 1), 9),       # nm > 48: plain DFMA rotation fallback
]


@pytest.mark.parametrize("case", RAGGED, ids=lambda c: "nw%d_nb%d_%d_nm%d_nq%d" % (c[0], c[1], c[2], c[3], c[6]))
@pytest.mark.parametrize("host", [False, True], ids=["dev", "host"])
def test_ragged_small_cases(env, case, host):
    wl, oracle = env["wl"], env["oracle"]
    nw, nb1, nb2, nm, ge, gp, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=ge, grid_p=gp, nq=nq, cfg_id=70 + nw)
    a = _inputs(wl, w)
    rng = np.random.default_rng(nq)
    deg_e = rng.integers(1, 4, w.nRe).astype(np.float64)
    deg_p = rng.integers(1, 4, w.nRp).astype(np.float64)
    out, g1 = _run_gpu(env, w, a["gW"], a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"], deg_e, deg_p, host=host)
    g1_ref = oracle.setk(a["gW"], a["Re"], deg_e, a["k"], a["Uk"])
    assert _relerr(g1, g1_ref) < 1e-12
    ref = oracle.qbatch(g1_ref, a["Rp"], deg_p, a["q"], a["Ukq"], a["ev"], a["om"])
    assert out.shape == ref.shape
    assert _relerr(out, ref) <= TOL


@pytest.mark.parametrize("knob", [{"tile": 32, "m3": 0}, {"tile": 64, "m3": 0}, {"tile": 32, "m3": 1},
                                  {"tile": 64, "m3": 1}, {"tile": 64, "m3": 1, "planar": 0}, {"rot_plain": 1}, {"tile": 64, "pair": 2}, {"tile": 64, "pair": 0},
                                  {"tile": 64, "pair": 2, "i8": 0}, {"tile": 64, "pair": 2, "i8": 1, "i8_cluster": 2}],
                         ids=lambda k: "_".join("%s%d" % kv for kv in k.items()))
def test_forced_kernel_variants(env, knob):
    """Every kernel variant the dispatcher can pick is parity-checked on the same input."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=6, nb1=5, nb2=6, nm=9, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nq=150, cfg_id=84)
    a = _inputs(wl, w)
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=150)
    for key, val in knob.items():
        ctx.set_tuning(key, val)
        if key == "m3":
            assert ctx.get_tuning(key) == val
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    out = ctx.q_batch(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])).cpu().numpy()
    assert _relerr(out, ref) <= TOL
    ctx.close()


def test_nonpositive_omega_and_sub_batches(env):
    """R7 (omega <= 0 -> 0) and the internal q sub-batching (nq_sub smaller than nq)."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=4, nb1=3, nb2=4, nm=3, grid_e=(3, 3, 3), nq=300, cfg_id=81)
    a = _inputs(wl, w)
    om = a["om"].copy(); om[5, 1] = 0.0; om[299, 2] = -0.3
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], om)
    gW = torch.from_numpy(a["gW"]).cuda()
    ctx = harness.make_context(w, gW, nq_max=300)
    ctx.set_tuning("nq_sub", 128)
    (Uk_d,) = harness.to_device([a["Uk"]])
    ctx.set_k(a["k"], Uk_d)
    q_d, Ukq_d, ev_d, om_d = harness.to_device([a["q"], a["Ukq"], a["ev"], om])
    out = ctx.q_batch(q_d, Ukq_d, ev_d, om_d).cpu().numpy()
    assert np.all(out[5, :, :, 1] == 0.0) and np.all(out[299, :, :, 2] == 0.0)
    assert _relerr(out, ref) <= TOL
    n = ctx.launch_counts()
    assert n["contract"] == 3 and n["qphase"] == 3 and n["rotate_epilogue"] == 3 and n["setk_stream"] == 1
    ctx.close()


def test_band_windows_change_between_calls_and_errors(env):
    """nb1 may change on every set_k, nb2 on every q_batch; error codes."""
    wl, oracle, torch, harness, binding = env["wl"], env["oracle"], env["torch"], env["harness"], env["binding"]
    w = wl.custom(nw=6, nm=3, grid_e=(3, 2, 3), nq=40, cfg_id=82)
    a = _inputs(wl, w)
    gW = torch.from_numpy(a["gW"]).cuda()
    ctx = harness.make_context(w, gW, nq_max=40)
    q_d, ev_d, om_d = harness.to_device([a["q"], a["ev"], a["om"]])
    with pytest.raises(binding.PhoebeElphError) as e:
        ctx.q_batch(q_d, harness.to_device([a["Ukq"]])[0], ev_d, om_d)
    assert e.value.code == -4
    for nb1, nb2 in [(6, 6), (2, 5), (5, 1), (1, 6)]:
        Uk = np.ascontiguousarray(a["Uk"][:, :nb1]); Ukq = np.ascontiguousarray(a["Ukq"][:, :, :nb2])
        Uk_d, Ukq_d = harness.to_device([Uk, Ukq])
        ctx.set_k(a["k"], Uk_d)
        out = ctx.q_batch(q_d, Ukq_d, ev_d, om_d).cpu().numpy()
        ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], Uk, a["q"], Ukq, a["ev"], a["om"])
        assert out.shape == (40, nb1, nb2, 3)
        assert _relerr(out, ref) <= TOL
    # nq beyond nq_max
    big = torch.zeros((41, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(binding.PhoebeElphError) as e:
        ctx.q_batch(big, torch.zeros((41, 6, 6), dtype=torch.complex128, device="cuda"),
                    torch.zeros((41, 3, 3), dtype=torch.complex128, device="cuda"),
                    torch.zeros((41, 3), dtype=torch.float64, device="cuda"))
    assert e.value.code == -2
    ctx.close()


KBATCH = [
    # nw nb1 nb2 nm  grid_e     grid_p    nk  nq
    (3, 2, 3, 2, (5, 1, 1), (3, 1, 1), 1, 5),        # nRe = 5 (k padding), X = 18 (one ragged column tile)
    (4, 4, 4, 3, (3, 3, 3), (2, 2, 2), 9, 40),       # BM = 16, ragged rows
    (6, 5, 6, 4, (2, 3, 3), (3, 3, 1), 20, 33),      # BM = 32, X = 144 (128 + ragged 16)
    (8, 8, 8, 6, (3, 3, 3), (3, 3, 3), 8, 70),       # BM = 8 exactly, X = 384 = 3 tiles
    (5, 3, 2, 9, (4, 2, 3), (1, 1, 2), 32, 7),       # the most k a batch takes
]


@pytest.mark.parametrize("case", KBATCH, ids=lambda c: "nw%d_nk%d" % (c[0], c[6]))
@pytest.mark.parametrize("host", [False, True], ids=["dev_m3", "host_4m"])
def test_set_k_batch_matches_oracle_per_k(env, case, host):
    """one pass over g_W for nk k-points == nk independent Eq. 71 precomputes."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    nw, nb1, nb2, nm, ge, gp, nk, nq = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=ge, grid_p=gp, nk=nk, nq=nq, cfg_id=60 + nw)
    gW_np, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
    rng = np.random.default_rng(nk)
    deg_e = rng.integers(1, 4, w.nRe).astype(np.float64)
    deg_p = rng.integers(1, 4, w.nRp).astype(np.float64)
    ks = wl.k_points(w)
    Uks = np.stack([wl.U_k(w, ik) for ik in range(nk)])
    gW = torch.from_numpy(gW_np).cuda()
    ctx = harness.make_context(w, gW, nq_max=nq, nk_max=nk, deg_e=deg_e, deg_p=deg_p)
    ctx.set_tuning("m3", 0 if host else 1)      # host leg: four-multiply product; device leg: three-multiply
    if host:
        ctx.set_k_batch_host(ks, Uks)
    else:
        ctx.set_k_batch(ks, harness.to_device([Uks])[0])
    worst = 0.0
    for ik in reversed(range(nk)):
        ctx.select_k(ik)
        g1 = ctx.copy_g1().cpu().numpy()
        g1_ref = oracle.setk(gW_np, Re, deg_e, ks[ik], Uks[ik])
        assert _relerr(g1, g1_ref) < 1e-12
        q, Ukq, ev, om = wl.q_inputs(w, ik)
        out = ctx.q_batch(*harness.to_device([q, Ukq, ev, om])).cpu().numpy()
        ref = oracle.qbatch(g1_ref, Rp, deg_p, q, Ukq, ev, om)
        worst = max(worst, _relerr(out, ref))
    assert worst <= TOL
    n = ctx.launch_counts()
    assert n["setk_gemm"] == 1 and n["setk_stream"] == 0 and n["setk_rotate"] == 1
    with pytest.raises(env["binding"].PhoebeElphError) as e:
        ctx.select_k(nk)
    assert e.value.code == -2
    # a plain set_k afterwards overwrites slot 0 and is what q_batch then uses
    ctx.set_k(ks[nk - 1], harness.to_device([Uks[nk - 1]])[0])
    q, Ukq, ev, om = wl.q_inputs(w, nk - 1)
    out = ctx.q_batch(*harness.to_device([q, Ukq, ev, om])).cpu().numpy()
    ref = oracle.elph(gW_np, Re, Rp, deg_e, deg_p, ks[nk - 1], Uks[nk - 1], q, Ukq, ev, om)
    assert _relerr(out, ref) <= TOL
    ctx.close()


def test_set_k_batch_needs_nk_max(env):
    wl, torch, harness, binding = env["wl"], env["torch"], env["harness"], env["binding"]
    w = wl.custom(nw=2, nm=3, grid_e=(3, 1, 1), nk=2, nq=4, cfg_id=61)
    ctx = harness.make_context(w, torch.from_numpy(wl.gW_full(w)).cuda(), nq_max=4)      # nk_max = 0
    Uks = np.stack([wl.U_k(w, i) for i in range(2)])
    with pytest.raises(binding.PhoebeElphError) as e:
        ctx.set_k_batch(wl.k_points(w), harness.to_device([Uks])[0])
    assert e.value.code == -2
    ctx.close()


def test_periodicity_on_gpu(env):
    """Eq. 87: out(k, q+G) = out(k, q) for integer G -- a property that holds at any size."""
    wl, torch, harness = env["wl"], env["torch"], env["harness"]
    w = wl.custom(nw=4, nm=3, grid_e=(3, 3, 3), nq=64, cfg_id=83)
    a = _inputs(wl, w)
    gW = torch.from_numpy(a["gW"]).cuda()
    ctx = harness.make_context(w, gW, nq_max=64)
    Uk_d, Ukq_d, ev_d, om_d = harness.to_device([a["Uk"], a["Ukq"], a["ev"], a["om"]])
    ctx.set_k(a["k"], Uk_d)
    (q_d,) = harness.to_device([a["q"]])
    base = ctx.q_batch(q_d, Ukq_d, ev_d, om_d).cpu().numpy()
    (q2_d,) = harness.to_device([a["q"] + np.array([1.0, -2.0, 3.0])])
    shifted = ctx.q_batch(q2_d, Ukq_d, ev_d, om_d).cpu().numpy()
    assert _relerr(shifted, base) < 1e-11
    ctx.set_k(a["k"] + np.array([-1.0, 2.0, 1.0]), Uk_d)
    shifted_k = ctx.q_batch(q_d, Ukq_d, ev_d, om_d).cpu().numpy()
    assert _relerr(shifted_k, base) < 1e-11
    ctx.close()


def test_empty_batch_is_a_noop(env):
    """nq = 0 in every q_batch* entry point: OK, nothing launched, nothing written, `rate` untouched; the next
    non-empty batch is unaffected."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=3, nb1=2, nb2=3, nm=3, grid_e=(3, 2, 1), grid_p=(2, 2, 2), nq=70, cfg_id=86)
    a = _inputs(wl, w)
    ctx = harness.make_context(w, torch.from_numpy(a["gW"]).cuda(), nq_max=70)
    ctx.set_k(a["k"], harness.to_device([a["Uk"]])[0])
    before = dict(ctx.launch_counts())
    z = lambda *s, dt=torch.float64: torch.zeros(s, dtype=dt, device="cuda")
    c128 = torch.complex128
    out = ctx.q_batch(z(0, 3), z(0, 3, 3, dt=c128), z(0, 3, 3, dt=c128), z(0, 3))
    assert out.shape == (0, 2, 3, 3)
    rate = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    ctx.q_batch_rates(z(0, 3), z(0, 3, 3, dt=c128), z(0, 3, 3, dt=c128), z(0, 3), z(2), z(0, 3), rate,
                      kT=0.02, mu=0.0, sigma=0.01, pref=1.0)
    e = lambda *s, dt=np.float64: np.zeros(s, dtype=dt)
    ctx.q_batch_host(e(0, 3), e(0, 3, 3, dt=np.complex128), e(0, 3, 3, dt=np.complex128), e(0, 3), e(0, 2, 3, 3))
    ctx.q_batch_host_async(e(0, 3), e(0, 3, 3, dt=np.complex128), e(0, 3, 3, dt=np.complex128), e(0, 3), e(0, 2, 3, 3))
    ctx.wait()
    assert dict(ctx.launch_counts()) == before
    assert rate.cpu().tolist() == [7.0, 7.0]
    got = ctx.q_batch(*harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])).cpu().numpy()
    ref = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    assert _relerr(got, ref) <= TOL
    ctx.close()


def test_si_like_full(env):
    """BASELINE.json configs[1], every one of the 4096 q."""
    wl, oracle = env["wl"], env["oracle"]
    w = wl.CONFIGS["si-like"]
    a = _inputs(wl, w)
    out, g1 = _run_gpu(env, w, a["gW"], a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
    g1_ref = oracle.setk(a["gW"], a["Re"], None, a["k"], a["Uk"])
    assert _relerr(g1, g1_ref) < 1e-12
    ref = oracle.qbatch(g1_ref, a["Rp"], None, a["q"], a["Ukq"], a["ev"], a["om"])
    assert _relerr(out, ref) <= TOL


def test_band_window_three_k(env):
    """BASELINE.json configs[3] (rectangular U, nb < nw): 3 of the 256 k, all 4096 q each."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.CONFIGS["band-window"]
    gW_np = wl.gW_full(w)
    gW = torch.from_numpy(gW_np).cuda()
    ctx = harness.make_context(w, gW)
    Re, Rp, ks = wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    worst = 0.0
    for ik in (0, 101, 255):
        Uk = wl.U_k(w, ik)
        q, Ukq, ev, om = wl.q_inputs(w, ik)
        ctx.set_k(ks[ik], harness.to_device([Uk])[0])
        out = ctx.q_batch(*harness.to_device([q, Ukq, ev, om])).cpu().numpy()
        ref = oracle.elph(gW_np, Re, Rp, None, None, ks[ik], Uk, q, Ukq, ev, om)
        assert out.shape == (4096, 4, 4, 6)
        worst = max(worst, _relerr(out, ref))
    assert worst <= TOL
    ctx.close()


def test_async_pipelined_host_batches(env):
    """q_batch_host_async: several k-points and batches in flight over the two staging slots, mixed with the
    synchronous entry point; every batch element by element against the oracle."""
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nk=3, nq=210, cfg_id=85)
    gW_np, Re, Rp, ks = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=210, nk_max=3)
    Uks = np.stack([wl.U_k(w, ik) for ik in range(3)])
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    ins = [[pin(x) for x in wl.q_inputs(w, ik)] for ik in range(3)]
    refs = [oracle.elph(gW_np, Re, Rp, None, None, ks[ik], Uks[ik], *wl.q_inputs(w, ik)) for ik in range(3)]
    for rep in range(2):
        outs = []
        ctx.set_k_batch_host(ks, Uks)
        for ik in range(3):
            ctx.select_k(ik)
            for sl in (slice(0, 100), slice(100, 210)):           # 6 batches in flight, slots reused 3 times
                o = torch.empty((sl.stop - sl.start, 4, 5, 6), dtype=torch.float64).pin_memory()
                q, U, z, om = [t[sl] for t in ins[ik]]
                ctx.q_batch_host_async(q.numpy(), U.numpy(), z.numpy(), om.numpy(), o.numpy())
                outs.append((ik, sl, o))
        ctx.wait()
        for ik, sl, o in outs:
            assert _relerr(o.numpy(), refs[ik][sl]) <= TOL
        # synchronous call right after (and, on the second round, without an explicit wait in between)
        ctx.select_k(1)
        if rep == 1:
            o = torch.empty((210, 4, 5, 6), dtype=torch.float64).pin_memory()
            ctx.q_batch_host_async(*[t.numpy() for t in ins[1]], o.numpy())
        out = np.empty((210, 4, 5, 6))
        ctx.q_batch_host(*[t.numpy() for t in ins[1]], out)
        assert _relerr(out, refs[1]) <= TOL
        if rep == 1:
            assert _relerr(o.numpy(), refs[1]) <= TOL
    ctx.close()


@pytest.mark.parametrize("batch", [False, True], ids=["set_k", "set_k_batch"])
def test_re_pool_partial_g1_sums_to_eq71(env, batch):
    """two contexts, each set up with one Re shard (its Re vectors, its slab of g_W),
    give partial g1'; their in-place sum through g1_view (what the pool's all-reduce does across GPUs) is the g1' of
    Eq. 71, and q_batch on it matches the oracle on the full problem.  (One device: the two shards run one after the
    other; the collective itself is covered by the world_size-2 gloo test.)"""
    from paper_2111_14999_b200 import sharding
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    w = wl.custom(nw=5, nb1=4, nb2=5, nm=6, grid_e=(3, 3, 2), grid_p=(3, 2, 2), nk=3, nq=90, cfg_id=86)
    gW_np, Re, Rp, ks = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    deg_e = np.random.default_rng(8).integers(1, 4, w.nRe).astype(np.float64)
    nk = 3 if batch else 1
    Uks = np.stack([wl.U_k(w, ik) for ik in range(nk)])
    from paper_2111_14999_b200 import binding
    ctxs = []
    for r in range(2):
        lo, hi = sharding.shard_range(w.nRe, r, 2)
        slab = torch.from_numpy(np.ascontiguousarray(gW_np[:, lo:hi])).cuda()
        c = binding.ElphContext(slab, Re[lo:hi], Rp, deg_e[lo:hi], None, nb1_max=w.nb1, nb2_max=w.nb2, nq_max=w.nq,
                                nk_max=nk if batch else 0)
        if batch:
            sharding.pool_set_k_batch(c, ks[:nk], harness.to_device([Uks])[0])      # world = 1: no collective
        else:
            sharding.pool_set_k(c, ks[0], harness.to_device([Uks[0]])[0])
        ctxs.append(c)
    a, b = ctxs[0].g1_view(-1), ctxs[1].g1_view(-1)
    assert a.shape == b.shape and a.data_ptr() != b.data_ptr()
    a.add_(b)                                          # what all_reduce(SUM) leaves on every rank of the pool
    for ik in reversed(range(nk)):
        ctxs[0].select_k(ik)
        g1_ref = oracle.setk(gW_np, Re, deg_e, ks[ik], Uks[ik])
        assert _relerr(ctxs[0].copy_g1().cpu().numpy(), g1_ref) < 1e-12
        v = ctxs[0].g1_view(ik).cpu().numpy()
        assert _relerr(v[..., 0] + 1j * v[..., 1], g1_ref) < 1e-12
        q, Ukq, ev, om = wl.q_inputs(w, ik)
        out = ctxs[0].q_batch(*harness.to_device([q, Ukq, ev, om])).cpu().numpy()
        assert _relerr(out, oracle.qbatch(g1_ref, Rp, None, q, Ukq, ev, om)) <= TOL
    with pytest.raises(binding.PhoebeElphError) as e:
        ctxs[0].g1_view(nk)
    assert e.value.code == -2
    for c in ctxs:
        c.close()


@pytest.mark.parametrize("knob", [{}, {"tile": 32}, {"nq_sub": 128}, {"m3": 0}, {"tile": 64, "planar": 0}, {"tile": 64}],
                         ids=["auto", "tile32", "sub128", "4m", "tile64_interleaved", "tile64_planar"])
def test_q_batch_multi_equals_per_k_calls(env, knob):
    """phoebe_elph_q_batch_multi: the q lists of the k slots stacked along the rows of ONE contraction, row block j
    against the g1' of slot j -- element by element against the oracle, and bit-identical to select_k + q_batch."""
    wl, oracle, torch, harness, binding = env["wl"], env["oracle"], env["torch"], env["harness"], env["binding"]
    nk, nq = 5, 192
    w = wl.custom(nw=8, nb1=4, nb2=4, nm=6, grid_e=(3, 3, 2), grid_p=(3, 3, 3), nk=nk, nq=nq, cfg_id=87)
    gW_np, Re, Rp, ks = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    Uks = np.stack([wl.U_k(w, ik) for ik in range(nk)])
    ins = [wl.q_inputs(w, ik) for ik in range(nk)]
    ctx = harness.make_context(w, torch.from_numpy(gW_np).cuda(), nq_max=nk * nq, nk_max=nk)
    for key, val in knob.items():
        ctx.set_tuning(key, val)
    ctx.set_k_batch(ks, harness.to_device([Uks])[0])
    stacked = harness.to_device([np.stack([ins[ik][j] for ik in range(nk)]) for j in range(4)])
    out = ctx.q_batch_multi(*stacked)
    assert out.shape == (nk, nq, 4, 4, 6)
    got = out.cpu().numpy()
    for ik in range(nk):
        ref = oracle.elph(gW_np, Re, Rp, None, None, ks[ik], Uks[ik], *ins[ik])
        assert _relerr(got[ik], ref) <= TOL
        ctx.select_k(ik)
        one = ctx.q_batch(*harness.to_device(list(ins[ik]))).cpu().numpy()
        if "nq_sub" not in knob:
            assert _relerr(one, got[ik]) <= 1e-12        # equal up to the rounding order (the two may take different a4 kernels)
    # fewer slots than the batch holds; errors
    part = ctx.q_batch_multi(*[t[:2].contiguous() for t in stacked]).cpu().numpy()
    assert _relerr(part, got[:2]) <= 1e-12
    for bad in ([t[:, :100].contiguous() for t in stacked],):            # nq not a multiple of 64
        with pytest.raises(binding.PhoebeElphError) as e:
            ctx.q_batch_multi(*bad)
        assert e.value.code == -2
    ctx.close()


def test_two_contexts_on_two_threads(env):
    """Two contexts, each on its own host thread and CUDA stream, through the whole path at the same time (different
    shapes, so different kernel instantiations and shared-memory opt-ins race for the per-device attribute table):
    both against the oracle, repeated so that first-use initialisation overlaps."""
    import threading
    wl, oracle, torch, harness = env["wl"], env["oracle"], env["torch"], env["harness"]
    shapes = [dict(nw=6, nb1=5, nb2=6, nm=9, grid_e=(3, 2, 2), grid_p=(3, 3, 2), nq=300, cfg_id=181),
              dict(nw=16, nb1=16, nb2=16, nm=12, grid_e=(2, 2, 1), grid_p=(3, 3, 1), nq=200, cfg_id=182)]
    cases = []
    for sh in shapes:
        w = wl.custom(**sh)
        a = _inputs(wl, w)
        a["w"] = w
        a["ref"] = oracle.elph(a["gW"], a["Re"], a["Rp"], None, None, a["k"], a["Uk"], a["q"], a["Ukq"], a["ev"], a["om"])
        cases.append(a)
    errs, excs = [None, None], []
    start = threading.Barrier(2)

    def worker(i):
        try:
            a = cases[i]
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                gW = torch.from_numpy(a["gW"]).cuda()
                d = harness.to_device([a["q"], a["Ukq"], a["ev"], a["om"]])
                (Uk_d,) = harness.to_device([a["Uk"]])
                st.synchronize()
                start.wait()
                worst = 0.0
                for rep in range(5):
                    ctx = harness.make_context(a["w"], gW, nq_max=a["w"].nq)      # binds torch's current stream (st)
                    ctx.set_k(a["k"], Uk_d)
                    out = ctx.q_batch(*d)
                    st.synchronize()
                    worst = max(worst, _relerr(out.cpu().numpy(), a["ref"]))
                    ctx.close()
                errs[i] = worst
        except Exception as exc:          # surfaced in the main thread
            excs.append(exc)
            try:
                start.abort()
            except Exception:
                pass

    ts = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join(120)
    assert not excs, excs
    assert errs[0] is not None and errs[0] <= TOL and errs[1] is not None and errs[1] <= TOL, errs
