"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(set_k_batch over the workload's k-points, pair-form contraction, whole q batch per launch; the 4-atom and band-window
workloads through the stacked launch of all k slots of a batch, phoebe_elph_q_batch_multi):

  * 4-atom  (configs[2]): g_W 26.1 GB resident, 16 k in one pass, 8192 q per k
  * large   (configs[4]): g_W 57.8 GB resident,  4 k in one pass, 16384 q per k
  * band-window (configs[3]): 32 k per pass, 32 x 4096 q stacked; every q of 33 k-points

The oracle cannot do every (k,q) of these in seconds, so -- as the task statement allows -- it
computes SAMPLED outputs one by one: for EVERY k-point the full g1' (Eq. 71; the slabs of g_W
are regenerated on the host one at a time and never exist at once) and, on one seeded q out of every
64-row tile of every k-point's q list (`_one_row_per_tile`), `out` (Eq. 70 + Eq. 7).  The properties that hold at any
size (Eq. 87 periodicity) are checked on the full batch.  Same bar as everywhere: 1e-10 relative.
"""
import concurrent.futures as cf
import os

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


def _upload_and_oracle_setk(env, w, k_ids):
    """One pass over the host-generated slabs of g_W: each slab is copied to the device AND fed to the
    oracle's Eq. 71 routine for the k-points in k_ids.  -> (gW on device, {ik: g1_ref[nRp][nb1][nw][nm]})."""
    torch, oracle, wl = env["torch"], env["oracle"], env["wl"]
    gW = torch.empty((w.nRp, w.nRe, w.nw, w.nw, w.nm), dtype=torch.complex128, device="cuda")
    Re, ks = wl.Re_vectors(w), wl.k_points(w)
    Uks = {ik: wl.U_k(w, ik) for ik in k_ids}
    g1_ref = {ik: np.empty((w.nRp, w.nb1, w.nw, w.nm), dtype=np.complex128) for ik in k_ids}
    threads = min(32, os.cpu_count() or 8)
    # a slab is at most 168.6 MB ("large"); at most `threads` of them are alive at once
    bufs = [torch.empty((w.nRe, w.nw, w.nw, w.nm), dtype=torch.complex128).pin_memory() for _ in range(threads)]
    free = list(range(threads))

    def work(p, slot):
        slab = bufs[slot].numpy()
        wl.gW_slab(w, p, slab)
        gW[p].copy_(bufs[slot])                      # synchronous pinned -> device copy
        for ik in k_ids:
            g1_ref[ik][p] = oracle.setk_slab(slab, Re, None, ks[ik], Uks[ik])
        return slot

    with cf.ThreadPoolExecutor(threads) as pool:
        pending = set()
        for p in range(w.nRp):
            if not free:
                done, pending = cf.wait(pending, return_when=cf.FIRST_COMPLETED)
                free.extend(f.result() for f in done)
            pending.add(pool.submit(work, p, free.pop()))
        for f in pending:
            f.result()
    torch.cuda.synchronize()
    return gW, g1_ref


def _one_row_per_tile(nq, tile=64, seed=777):
    """Sampling rule of the full-size tests: ONE seeded row out of every `tile` consecutive rows of a q list (the
    contraction's row tile is 64, the rotation takes 1..16 consecutive q per CTA), plus the first and the last row.
    Every row tile of every persistent-kernel round therefore has at least one row compared with the oracle."""
    rng = np.random.default_rng(seed)
    idx = np.arange(0, nq, tile) + rng.integers(0, tile, size=(nq + tile - 1) // tile)
    idx = np.minimum(idx, nq - 1)
    return np.unique(np.concatenate([[0], idx, [nq - 1]]))


def _full_size_case(env, name, k_props, stacked=False):
    """Every k-point of the workload, one q per 64-row tile (`_one_row_per_tile`), compared with the oracle at 1e-10 --
    through the launch bench.py times (stacked: all k slots in one launch; else one q_batch per k after one
    set_k_batch).  k_props: the k-points that additionally get the whole-batch property checks (bit-identical repeat,
    q -> q+G, stacked == per-k)."""
    torch, oracle, wl, harness = env["torch"], env["oracle"], env["wl"], env["harness"]
    w = wl.CONFIGS[name]
    free, _ = torch.cuda.mem_get_info()
    if free < w.gW_bytes + (24 << 30):
        pytest.skip("not enough free device memory for %s" % name)
    kb = min(16, w.nk)
    assert kb == w.nk                                 # every k-point of the workload sits in one set_k_batch
    k_all = tuple(range(kb))
    gW, g1_ref = _upload_and_oracle_setk(env, w, k_all)
    Rp, ks = wl.Rp_vectors(w), wl.k_points(w)
    # stacked: bench.py runs the q lists of all kb k slots through ONE phase / contraction / rotation launch
    # (phoebe_elph_q_batch_multi) when the stacked C fits 8 GB -- the 4-atom workload
    ctx = harness.make_context(w, gW, nk_max=kb, nq_max=kb * w.nq if stacked else None)
    assert ctx.nq_batch == (kb * w.nq if stacked else w.nq)      # the whole q list is one batch (L576 sizing)
    Uks = np.stack([wl.U_k(w, ik) for ik in range(kb)])
    ctx.set_k_batch(ks[:kb], harness.to_device([Uks])[0])
    idx = _one_row_per_tile(w.nq)
    assert len(idx) >= w.nq // 64
    idx_d = torch.from_numpy(idx).cuda()
    ins = [wl.q_inputs(w, ik) for ik in range(kb)]
    # the oracle on the sampled rows of EVERY k-point
    refs = [oracle.qbatch(g1_ref[ik], Rp, None, ins[ik][0][idx], np.ascontiguousarray(ins[ik][1][idx]),
                          np.ascontiguousarray(ins[ik][2][idx]), ins[ik][3][idx]) for ik in range(kb)]
    worst_g1 = max(_relerr(_g1_of(ctx, ik), g1_ref[ik]) for ik in k_all)
    gots, scale, bases = [], 0.0, {}
    out = torch.empty((w.nq, w.nb1, w.nb2, w.nm), dtype=torch.float64, device="cuda")
    if stacked:
        st = [torch.from_numpy(np.ascontiguousarray(np.stack([ins[ik][j] for ik in range(kb)]))).cuda() for j in range(4)]
        outm = ctx.q_batch_multi(*st)
        assert outm.shape == (kb, w.nq, w.nb1, w.nb2, w.nm)
        scale = float(outm.max().item())             # R10: the maximum is over the whole compared config
        gots = [outm[ik][idx_d].cpu().numpy() for ik in range(kb)]
        n_multi = 1
    else:
        for ik in range(kb):
            ctx.select_k(ik)
            ctx.q_batch(*harness.to_device(ins[ik]), out)
            scale = max(scale, float(out.max().item()))
            gots.append(out[idx_d].cpu().numpy())
            if ik in k_props:
                bases[ik] = out.clone()
        n_multi = 0
    assert scale > 0 and np.isfinite(scale)
    worst_out = max(float(np.max(np.abs(g - r))) / max(scale, float(r.max())) for g, r in zip(gots, refs))
    # whole-batch properties on a few k-points (they compare the CUDA path with itself on EVERY row)
    n_single = 0 if stacked else kb
    for ik in k_props:
        ctx.select_k(ik)
        q_d, Ukq_d, ev_d, om_d = harness.to_device(ins[ik])
        if ik not in bases:
            ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)
            bases[ik] = out.clone()
            n_single += 1
        base = bases[ik]
        # the path has a fixed summation order: the same call again is bit-identical (this is what exposed a
        # shared-memory ring race in the contraction: an early stage release let a bulk copy overwrite fragments
        # still being loaded, on the first, cold call only)
        ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)
        assert bool(torch.equal(out, base)), "q_batch is not reproducible"
        if stacked:
            assert float((outm[ik] - base).abs().max().item()) <= 1e-12 * scale, "stacked form differs from the per-k call"
        # Eq. 87 on the whole batch: q -> q + G leaves out unchanged
        (q2_d,) = harness.to_device([ins[ik][0] + np.array([2.0, -1.0, 1.0])])
        ctx.q_batch(q2_d, Ukq_d, ev_d, om_d, out)
        out.sub_(base)
        shift_err = float(out.abs().max().item())
        n_single += 2
        del bases[ik]
        assert shift_err <= 1e-10 * scale, (shift_err, scale)
    n = ctx.launch_counts()
    assert n["setk_gemm"] == 1 and n["contract"] == n_single + n_multi       # one contraction launch per q batch
    ctx.close()
    del gW, out
    torch.cuda.empty_cache()
    assert worst_g1 < 1e-12, worst_g1
    assert worst_out <= TOL, worst_out


def _g1_of(ctx, ik):
    ctx.select_k(ik)
    return ctx.copy_g1().cpu().numpy()


def test_4atom_full_size_every_k_every_tile(env):
    """BASELINE.json configs[2] through the stacked launch bench.py times (set_k_batch(16) + q_batch_multi over
    16 x 8192 q): EVERY one of the 16 k slots, one q out of every 64-row tile of its 8192 (130 q per k; SURVEY 8(d)
    "all 16 k x 256 q ... cover every q-tile position"), g1' of every k element-wise; k = 0, 15 also per k with the
    whole-batch property checks."""
    _full_size_case(env, "4-atom", k_props=(0, 15), stacked=True)


def test_large_full_size_every_k_every_tile(env):
    """BASELINE.json configs[4]: the 57.8 GB g_W, set_k_batch(4) + one q_batch of 16384 q per k (bench.py's launch for
    this workload): ALL 4 k-points, one q out of every 64-row tile (258 q per k), g1' of every k element-wise; k = 3
    also with the whole-batch property checks."""
    _full_size_case(env, "large", k_props=(3,))


def test_band_window_full_size_stacked_batches(env):
    """BASELINE.json configs[3] in the launch shape bench.py times: set_k_batch(32) + q_batch_multi (and
    q_batch_rates_multi) over 32 x 4096 stacked q.  The whole first batch (k = 0..31, ALL 4096 q of each) and the last
    batch's k = 255 (all 4096 q) against the oracle at 1e-10; the fused linewidths of every checked k against
    oracle.rates of the oracle's own |g|^2."""
    torch, oracle, wl, harness = env["torch"], env["oracle"], env["wl"], env["harness"]
    w = wl.CONFIGS["band-window"]
    kb = 32
    gW_np = wl.gW_full(w)
    gW = torch.from_numpy(gW_np).cuda()
    Re, Rp, ks = wl.Re_vectors(w), wl.Rp_vectors(w), wl.k_points(w)
    ctx = harness.make_context(w, gW, nk_max=kb, nq_max=kb * w.nq)
    assert ctx.nq_batch == kb * w.nq
    P = wl.RATE_PARAMS
    worst = worst_rate = 0.0
    for batch, check in ((0, range(kb)), (w.nk // kb - 1, (kb - 1,))):
        kid = list(range(batch * kb, (batch + 1) * kb))
        Uks = np.stack([wl.U_k(w, ik) for ik in kid])
        ctx.set_k_batch(ks[kid], harness.to_device([Uks])[0])
        ins = [wl.q_inputs(w, ik) for ik in kid]
        eps = [wl.band_energies(w, ik) for ik in kid]
        st = [torch.from_numpy(np.ascontiguousarray(np.stack([x[j] for x in ins]))).cuda() for j in range(4)]
        outm = ctx.q_batch_multi(*st)
        eps_k = torch.from_numpy(np.stack([e[0] for e in eps])).cuda()
        eps_kq = torch.from_numpy(np.ascontiguousarray(np.stack([e[1] for e in eps]))).cuda()
        rate = torch.zeros((kb, w.nb1), dtype=torch.float64, device="cuda")
        ctx.q_batch_rates_multi(*st, eps_k, eps_kq, rate, **P)
        got, rate = outm.cpu().numpy(), rate.cpu().numpy()
        scale = float(got.max())
        for j in check:
            ik = kid[j]
            g1_ref = oracle.setk(gW_np, Re, None, ks[ik], Uks[j])
            ref = oracle.qbatch(g1_ref, Rp, None, *ins[j])
            worst = max(worst, float(np.max(np.abs(got[j] - ref))) / max(scale, float(ref.max())))
            r_ref = oracle.rates(ref, eps[j][0], eps[j][1], ins[j][3], P["kT"], P["mu"], P["sigma"], P["pref"])
            worst_rate = max(worst_rate, float(np.max(np.abs(rate[j] - r_ref)) / np.max(np.abs(r_ref))))
    n = ctx.launch_counts()
    assert n["setk_gemm"] == 2 and n["contract"] == 4         # one stacked contraction per (batch, call)
    ctx.close()
    assert worst <= TOL, worst
    assert worst_rate <= TOL, worst_rate
