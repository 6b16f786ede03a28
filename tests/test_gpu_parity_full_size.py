"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(set_k_batch over the workload's k-points, pair-form contraction, whole q batch per launch; the 4-atom workload also
through the stacked launch of all its k slots, phoebe_elph_q_batch_multi):

  * 4-atom  (configs[2]): g_W 26.1 GB resident, 16 k in one pass, 8192 q per k
  * large   (configs[4]): g_W 57.8 GB resident,  4 k in one pass, 16384 q per k

The oracle cannot do every (k,q) of these in seconds, so -- as the task statement allows -- it
computes SAMPLED outputs one by one: for the chosen k-points the full g1' (Eq. 71; the slabs of g_W
are regenerated on the host one at a time and never exist at once) and, on a seeded sample of the
q list that covers every tile position, `out` (Eq. 70 + Eq. 7).  The properties that hold at any
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


def _full_size_case(env, name, k_check, n_sample, stacked=False):
    torch, oracle, wl, harness = env["torch"], env["oracle"], env["wl"], env["harness"]
    w = wl.CONFIGS[name]
    free, _ = torch.cuda.mem_get_info()
    if free < w.gW_bytes + (24 << 30):
        pytest.skip("not enough free device memory for %s" % name)
    gW, g1_ref = _upload_and_oracle_setk(env, w, k_check)
    Rp, ks = wl.Rp_vectors(w), wl.k_points(w)
    kb = min(16, w.nk)
    # stacked: bench.py runs the q lists of all kb k slots through ONE phase / contraction / rotation launch
    # (phoebe_elph_q_batch_multi) when the stacked C fits 8 GB -- the 4-atom workload
    ctx = harness.make_context(w, gW, nk_max=kb, nq_max=kb * w.nq if stacked else None)
    assert ctx.nq_batch == (kb * w.nq if stacked else w.nq)      # the whole q list is one batch (L576 sizing)
    refs, bases = {}, {}
    Uks = np.stack([wl.U_k(w, ik) for ik in range(kb)])
    ctx.set_k_batch(ks[:kb], harness.to_device([Uks])[0])
    out = torch.empty((w.nq, w.nb1, w.nb2, w.nm), dtype=torch.float64, device="cuda")
    idx = wl.sample_indices(w.nq, n_sample)
    idx[0], idx[-1] = 0, w.nq - 1                    # first and last tile rows always in the sample
    worst_g1 = worst_out = 0.0
    for ik in k_check:
        ctx.select_k(ik)
        g1 = ctx.copy_g1().cpu().numpy()
        worst_g1 = max(worst_g1, _relerr(g1, g1_ref[ik]))
        q, Ukq, ev, om = wl.q_inputs(w, ik)
        q_d, Ukq_d, ev_d, om_d = harness.to_device([q, Ukq, ev, om])
        ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)
        got = out[torch.from_numpy(idx).cuda()].cpu().numpy()
        ref = oracle.qbatch(g1_ref[ik], Rp, None, q[idx], np.ascontiguousarray(Ukq[idx]),
                            np.ascontiguousarray(ev[idx]), om[idx])
        scale = float(out.max().item())              # R10: the maximum is over the whole compared config
        assert scale > 0 and np.isfinite(scale)
        worst_out = max(worst_out, float(np.max(np.abs(got - ref))) / max(scale, float(ref.max())))
        # Eq. 87 on the whole batch: q -> q + G leaves out unchanged
        base = out.clone()
        # the path has a fixed summation order: the same call again is bit-identical (this is what exposed a
        # shared-memory ring race in the contraction: an early stage release let a bulk copy overwrite fragments
        # still being loaded, on the first, cold call only)
        ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)
        assert bool(torch.equal(out, base)), "q_batch is not reproducible"
        (q2_d,) = harness.to_device([q + np.array([2.0, -1.0, 1.0])])
        ctx.q_batch(q2_d, Ukq_d, ev_d, om_d, out)
        out.sub_(base)
        shift_err = float(out.abs().max().item())
        if stacked:
            refs[ik], bases[ik] = (ref, scale), base
        del base
        assert shift_err <= 1e-10 * scale, (shift_err, scale)
    if stacked:
        # the launch configuration of bench.py: all kb q lists stacked, one launch of each kernel
        ins = [wl.q_inputs(w, ik) for ik in range(kb)]
        st = [torch.from_numpy(np.ascontiguousarray(np.stack([ins[ik][j] for ik in range(kb)]))).cuda() for j in range(4)]
        del ins
        outm = ctx.q_batch_multi(*st)
        assert outm.shape == (kb, w.nq, w.nb1, w.nb2, w.nm)
        for ik in k_check:
            ref, scale = refs[ik]
            got = outm[ik][torch.from_numpy(idx).cuda()].cpu().numpy()
            worst_out = max(worst_out, float(np.max(np.abs(got - ref))) / max(scale, float(ref.max())))
            assert bool(torch.equal(outm[ik], bases[ik])), "stacked form differs from the per-k call"
        del outm, st, bases
    n = ctx.launch_counts()
    assert n["setk_gemm"] == 1 and n["contract"] == 3 * len(k_check) + (1 if stacked else 0)   # one launch per q batch
    ctx.close()
    del gW, out
    torch.cuda.empty_cache()
    assert worst_g1 < 1e-12, worst_g1
    assert worst_out <= TOL, worst_out


def test_4atom_full_size_sampled(env):
    """BASELINE.json configs[2]: 16 k in one pass over the 26.1 GB g_W; k-points 0 and 15, 96 sampled q of 8192 -- per k
    and through the stacked launch of all 16 x 8192 q that bench.py times."""
    _full_size_case(env, "4-atom", k_check=(0, 15), n_sample=96, stacked=True)


def test_large_full_size_sampled(env):
    """BASELINE.json configs[4]: the 57.8 GB g_W, 4 k in one pass; k-point 3, 40 sampled q of 16384."""
    _full_size_case(env, "large", k_check=(3,), n_sample=40)
