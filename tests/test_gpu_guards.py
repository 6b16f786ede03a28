"""Memory-safety checks of the CUDA path that need no external tool (compute-sanitizer is closed on this pool, see
profiles/r2_sanitizers.md):

  * POISONED WORKSPACE: the caller-allocated workspace starts as all-NaN bytes (0xFF).  Any kernel that reads workspace
    memory it (or an earlier kernel) did not write -- ring padding, C-layout padding, staging slack -- and lets it reach
    a result turns `out` into NaN and fails the oracle comparison.
  * CANARIES: `out`, `rate` and the g1' copy sit inside larger buffers whose surroundings hold a bit pattern; after the
    calls the surroundings must be bit-identical (no out-of-bounds write by any kernel of the path).
  * REPEATS: the same call again, and on a second poisoned context, is bit-identical (no dependence on stale
    shared-memory or workspace contents, no race between the producer's bulk copies and the consumers' loads).

Shapes cover every staging form of the rotation kernel (whole q-points per stage with block and with row copies,
b1 groups on two rings), the three contraction kernels, the stacked forms and the fused linewidths / polar term.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10
PAT = 0x7FF8DEADBEEF0BAD            # a quiet NaN with a recognisable payload


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


def _guarded(torch, shape, pad=4096):
    """A float64 CUDA tensor of `shape` inside a larger buffer filled with PAT -> (view, whole buffer, slice)."""
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * pad,), PAT, dtype=torch.int64, device="cuda")
    view = buf[pad:pad + n].view(torch.float64).view(*shape)
    return view, buf, (pad, pad + n)


def _canaries_intact(buf, sl):
    lo, hi = sl
    return bool((buf[:lo] == PAT).all().item()) and bool((buf[hi:] == PAT).all().item())


#        nw nb1 nb2 nm  grid_e     grid_p     nq   knobs
CASES = [(8, 4, 4, 6, (3, 2, 2), (3, 3, 3), 1000, {}),                       # band-window shape: block copies, 12 q per stage
         (8, 4, 4, 6, (3, 2, 2), (3, 3, 3), 1000, {"rot_blk": 1}),           # the same through row copies
         (16, 16, 16, 12, (2, 2, 1), (3, 3, 1), 150, {}),                    # 4-atom shape: padded C rows, b1 pairs
         (12, 7, 12, 30, (2, 1, 1), (3, 1, 1), 60, {"rot_gb1": 2}),          # b1 groups: two rings, ragged last group
         (5, 3, 4, 9, (2, 2, 1), (2, 3, 1), 257, {"pair": 0}),               # planar contraction, ragged everything
         (5, 3, 4, 9, (2, 2, 1), (2, 3, 1), 257, {"tile": 32}),              # interleaved 32x32 contraction
         (3, 3, 3, 51, (2, 1, 1), (2, 1, 1), 40, {})]                        # nm > 48: plain rotation kernel


@pytest.mark.parametrize("case", CASES, ids=lambda c: "nw%d_nb%d_%d_nm%d_%s" % (c[0], c[1], c[2], c[3], "_".join(c[7]) or "auto"))
def test_poisoned_workspace_and_canaries(env, case):
    wl, oracle, torch, binding, harness = env["wl"], env["oracle"], env["torch"], env["binding"], env["harness"]
    nw, nb1, nb2, nm, ge, gp, nq, knobs = case
    w = wl.custom(nw=nw, nb1=nb1, nb2=nb2, nm=nm, grid_e=ge, grid_p=gp, nq=nq, cfg_id=150 + nm)
    gW_np, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
    k, Uk = wl.k_points(w)[0], wl.U_k(w)
    q, Ukq, ev, om = wl.q_inputs(w)
    eps_k, eps_kq = wl.band_energies(w)
    P = dict(wl.RATE_PARAMS)
    ref = oracle.elph(gW_np, Re, Rp, None, None, k, Uk, q, Ukq, ev, om)
    rate_ref = oracle.rates(ref, eps_k, eps_kq, om, P["kT"], P["mu"], P["sigma"], P["pref"])
    gW = torch.from_numpy(gW_np).cuda()
    d = harness.to_device([q, Ukq, ev, om])
    de = harness.to_device([eps_k, eps_kq])
    results = []
    for _ in range(2):                                   # two independent poisoned contexts
        ctx = binding.ElphContext(gW, Re, Rp, None, None, nb1_max=nb1, nb2_max=nb2, nq_max=nq, poison_workspace=True)
        for key, val in knobs.items():
            ctx.set_tuning(key, val)
        ctx.set_k(k, harness.to_device([Uk])[0])
        out, obuf, osl = _guarded(torch, (nq, nb1, nb2, nm))
        ctx.q_batch(*d, out)
        first = out.clone()
        ctx.q_batch(*d, out)
        assert torch.equal(out, first), "q_batch is not reproducible"
        rate, rbuf, rsl = _guarded(torch, (nb1,), pad=64)
        rate.zero_()
        out2, o2buf, o2sl = _guarded(torch, (nq, nb1, nb2, nm))
        ctx.q_batch_rates(*d, *de, rate, out=out2, **P)
        rate_only, r2buf, r2sl = _guarded(torch, (nb1,), pad=64)
        rate_only.zero_()
        ctx.q_batch_rates(*d, *de, rate_only, **P)
        torch.cuda.synchronize()
        assert _canaries_intact(obuf, osl) and _canaries_intact(o2buf, o2sl), "out-of-bounds write around out"
        assert _canaries_intact(rbuf, rsl) and _canaries_intact(r2buf, r2sl), "out-of-bounds write around rate"
        o = out.cpu().numpy()
        assert np.isfinite(o).all(), "uninitialised workspace memory reached out"
        assert _relerr(o, ref) <= TOL and _relerr(out2.cpu().numpy(), ref) <= TOL
        assert _relerr(rate.cpu().numpy(), rate_ref) <= TOL
        assert torch.equal(rate, rate_only)
        results.append(first.cpu().numpy())
        ctx.close()
    assert np.array_equal(results[0], results[1]), "result depends on what the workspace held before"


def test_poisoned_workspace_stacked_and_polar(env):
    """set_k_batch + q_batch_multi / q_batch_rates_multi and the polar term on poisoned workspaces, with canaries."""
    wl, oracle, torch, binding, harness = env["wl"], env["oracle"], env["torch"], env["binding"], env["harness"]
    nk = 3
    w = wl.custom(nw=6, nb1=4, nb2=5, nm=6, grid_e=(2, 2, 1), grid_p=(3, 3, 1), nk=nk, nq=192, cfg_id=171)
    gW_np, Re, Rp, ks = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    Uks = np.stack([wl.U_k(w, i) for i in range(nk)])
    ins = [wl.q_inputs(w, i) for i in range(nk)]
    st = harness.to_device([np.ascontiguousarray(np.stack([x[j] for x in ins])) for j in range(4)])
    refs = [oracle.elph(gW_np, Re, Rp, None, None, ks[i], Uks[i], *ins[i]) for i in range(nk)]
    ctx = binding.ElphContext(torch.from_numpy(gW_np).cuda(), Re, Rp, None, None, nb1_max=w.nb1, nb2_max=w.nb2,
                              nq_max=nk * w.nq, nk_max=nk, poison_workspace=True)
    ctx.set_k_batch(ks, harness.to_device([Uks])[0])
    out, obuf, osl = _guarded(torch, (nk, w.nq, w.nb1, w.nb2, w.nm))
    ctx.q_batch_multi(*st, out)
    torch.cuda.synchronize()
    assert _canaries_intact(obuf, osl)
    got = out.cpu().numpy()
    for i in range(nk):
        assert _relerr(got[i], refs[i]) <= TOL
    # polar term on the same (poisoned) context
    pol = wl.polar_inputs(w)
    ctx.set_polar(**pol)
    ctx.select_k(1)
    q, Ukq, ev, om = ins[1]
    Pq = oracle.polar_amplitude(q, ev, pol["recip"], pol["G"], pol["Zstar"], pol["eps_inf"], pol["coeff"])
    g1_ref = oracle.setk(gW_np, Re, None, ks[1], Uks[1])
    ref = oracle.qbatch_polar(g1_ref, Rp, None, q, Ukq, ev, om, Uks[1], Pq)
    o1, o1buf, o1sl = _guarded(torch, (w.nq, w.nb1, w.nb2, w.nm))
    ctx.q_batch(*harness.to_device([q, Ukq, ev, om]), o1)
    torch.cuda.synchronize()
    assert _canaries_intact(o1buf, o1sl)
    assert _relerr(o1.cpu().numpy(), ref) <= TOL
    ctx.close()
