#!/usr/bin/env python
"""bench.py -- throughput of the el-ph Wannier->Bloch |g|^2 hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A "step" is one pass of the whole hot path (set_k + q_batch for every k of the
workload: SURVEY.md 8(a) rows a1..a7) over one batch of seeded synthetic input.
Prints ONE JSON line.  `--impl reference` times the
CPU oracle (oracle/, as it stands) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2111_14999_b200 import workloads as wl  # noqa: E402

METRIC = "interpolated el-ph (k,q) pairs/sec"
UNIT = "pairs/s"
DEFAULT_WORKLOAD = "4-atom"

# FP64 "alu" peak derived from unit counts and clocks:
# 64 FP64 FMA / clk / SM  x 2 flop x 148 SMs x 1.965 GHz (clocks.max.sm)
FP64_PEAK_TFLOPS = 64 * 2 * 148 * 1.965e9 / 1e12
HBM_FALLBACK_GBS = 6650.0


# ----------------------------------------------------------------------------- utilities
def _measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": HBM_FALLBACK_GBS}, "fallback"


def _ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed ncu --set full
    summary profiles/traffic.csv (columns: workload,kernel,dram_bytes_per_launch,source); None if not captured."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    try:
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 3 and f[0] == workload and f[1] == kernel:
                return float(f[2])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        try:
            rows = [r.strip().split(",") for r in open(self.path) if r.strip()]
            os.unlink(self.path)
            sm = [float(r[0]) for r in rows if len(r) >= 7]
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            reasons = set()
            for r in rows:
                if len(r) >= 7:
                    for nme, v in zip(names, r[3:7]):
                        if v.strip().lower() == "active":
                            reasons.add(nme)
            if sm:
                out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(rows[0][1]), reasons=sorted(reasons),
                           samples=len(sm), power_w_max=max(float(r[2]) for r in rows if len(r) >= 7))
        except Exception:
            pass
        return out


from paper_2111_14999_b200.sharding import dist_env as _dist_env, max_over_ranks, shard_k  # noqa: E402


def _k_inputs(w, ik):
    """Inputs of k-point index ik; indices beyond the workload's own nk (other ranks' shards under weak
    scaling) reuse the recipe with a fresh seed index."""
    nk = w.nk
    ks = wl.k_points(w)
    k = ks[ik % nk] if ik < nk else np.random.default_rng([w.seed, w.cfg_id, 1, ik]).random(3)
    return k, wl.U_k(w, ik), wl.q_inputs(w, ik)


# ----------------------------------------------------------------------------- CPU oracle legs
def time_oracle(w, budget_s: float = 20.0):
    """The oracle as it stands, timed on the host cores on a bounded sample of workload w.
    Returns (pairs_per_s, cores, sample_description).  set_k is timed on a subset of the Rp slabs and
    scaled by nRp/slabs (it is a plain sum over independent slabs); q_batch is timed on a subset of the
    q list against a g1' of the right shape, and scaled by nq/sample."""
    import oracle
    cores = oracle.num_threads()
    Re, Rp = wl.Re_vectors(w), wl.Rp_vectors(w)
    k, Uk = wl.k_points(w)[0], wl.U_k(w, 0)
    slab_flop = 8.0 * w.nRe * w.X
    # assume >= 0.3 GFLOP/s/core for sizing; the measured time is what is reported
    n_slab = int(max(cores, min(w.nRp, (0.3 * budget_s * 0.3e9 * cores) / slab_flop)))
    n_slab = max(1, min(w.nRp, n_slab, int(2e9 // (16 * w.nRe * w.X))))      # <= 2 GB of g_W on the host
    slabs = np.empty((n_slab, w.nRe, w.nw, w.nw, w.nm), dtype=np.complex128)
    import concurrent.futures as cf
    with cf.ThreadPoolExecutor(min(16, os.cpu_count() or 4)) as pool:
        list(pool.map(lambda p: wl.gW_slab(w, p, slabs[p]), range(n_slab)))
    t0 = time.perf_counter()
    g1_part = oracle.setk(slabs, Re, None, k, Uk)
    t_setk = (time.perf_counter() - t0) * (w.nRp / n_slab)
    # q part: g1' of the right shape (values are irrelevant for timing): tile what set_k produced
    reps = -(-w.nRp // n_slab)
    g1 = np.ascontiguousarray(np.concatenate([g1_part] * reps)[: w.nRp])
    q_flop = 8.0 * w.nRp * w.N + 8.0 * w.nb1 * w.nb2 * w.nm * (w.nw + w.nm)
    nq_s = int(max(cores, min(w.nq, (0.7 * budget_s * 0.4e9 * cores) / q_flop)))
    nq_s = min(w.nq, nq_s)
    q, Ukq, ev, om = wl.q_inputs(w, 0)
    idx = wl.sample_indices(w.nq, nq_s)
    qa, Ua, ea, oa = q[idx], np.ascontiguousarray(Ukq[idx]), np.ascontiguousarray(ev[idx]), om[idx]
    t0 = time.perf_counter()
    oracle.qbatch(g1, Rp, None, qa, Ua, ea, oa)
    t_q = (time.perf_counter() - t0) * (w.nq / nq_s)
    pairs_per_s = w.nq / (t_setk + t_q)
    sample = (f"1 k-point of {w.nk}: set_k on {n_slab}/{w.nRp} Rp slabs (scaled x{w.nRp / n_slab:.2f}), "
              f"q_batch on {nq_s}/{w.nq} q (scaled x{w.nq / nq_s:.2f}); gcc -O2 -fopenmp, {cores} threads")
    return pairs_per_s, cores, sample, (t_setk, t_q)


def run_reference(args):
    rank, world, _ = _dist_env()
    if rank != 0:
        return
    w = wl.CONFIGS[args.workload]
    vals = []
    sample = ""
    cores = 0
    budget = max(2.0, min(20.0, 90.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        v, cores, sample, _ = time_oracle(w, budget)
        if i >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    ms_per_step = 1e3 * (w.nk * w.nq) / value
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(w, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def _config_dict(w, n_gpus):
    return {"workload": w.name, "nw": w.nw, "nb1": w.nb1, "nb2": w.nb2, "nmodes": w.nm, "nRe": w.nRe, "nRp": w.nRp,
            "nk": w.nk, "nq_per_k": w.nq, "gW_GB": round(w.gW_bytes / 1e9, 3),
            "cache": "inputs larger than L2 (g_W is streamed from HBM every step)",
            "parallelism": f"k-sharded x{n_gpus}, g_W replicated, no collective"}


def _with_kbatch(cfg, kb):
    cfg = dict(cfg)
    cfg["set_k_batch"] = kb
    return cfg


def _with_multi(cfg, multi):
    cfg = dict(cfg)
    cfg["q_batch_multi"] = bool(multi)
    return cfg


# ----------------------------------------------------------------------------- GPU leg
def run_ours(args):
    import torch
    from paper_2111_14999_b200 import binding, build, harness

    rank, world, local = _dist_env()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    binding.load_library()

    w = wl.CONFIGS[args.workload]
    t_gen = time.perf_counter()
    gW = harness.upload_gW(w, dev)
    k_ids = shard_k(w.nk, rank, world, "weak")
    host_inputs = [_k_inputs(w, ik) for ik in k_ids]
    dev_inputs = []
    for k, Uk, (q, Ukq, ev, om) in host_inputs:
        dev_inputs.append((k, harness.to_device([Uk], dev)[0], harness.to_device([q, Ukq, ev, om], dev)))
    t_gen = time.perf_counter() - t_gen
    kb = max(1, min(args.k_batch, 32, len(host_inputs)))
    # the q lists of all k slots of a batch go through ONE phase / contraction / rotation launch
    # (phoebe_elph_q_batch_multi) whenever the stacked C fits 8 GB: for band windows one k-point's list alone is too
    # small a GEMM for 148 SMs (57 % -> 92 % of peak), for the 4-atom cell it removes the ragged last round of tiles and
    # the launch gaps (93.8 % -> 95.1 %)
    multi = (kb > 1 and args.q_multi != 0 and w.nq % 64 == 0 and len(host_inputs) % kb == 0
             and (args.q_multi == 1 or kb * w.nq * w.N * 16 <= (8 << 30)))
    ctx = harness.make_context(w, gW, nk_max=kb if kb > 1 else 0, nq_max=kb * w.nq if multi else None)
    ctx.set_tuning("m3", args.m3)
    if args.tile:
        ctx.set_tuning("tile", args.tile)
    for kv in args.tune:                      # kernel-variant experiments: --tune rot_qg=4 (see include/phoebe_elph.h, set_tuning)
        key, val = kv.split("=")
        ctx.set_tuning(key, int(val))
    out = torch.empty((w.nq, w.nb1, w.nb2, w.nm), dtype=torch.float64, device=dev)
    # k-points grouped into batches of kb: one pass over g_W per batch (set_k_batch)
    groups = [list(range(i, min(i + kb, len(host_inputs)))) for i in range(0, len(host_inputs), kb)]
    ks_np = [np.stack([host_inputs[i][0] for i in g]) for g in groups]
    Uks_np = [np.ascontiguousarray(np.stack([host_inputs[i][1] for i in g])) for g in groups]
    Uks_d = [harness.to_device([u], dev)[0] for u in Uks_np]

    if multi:
        stacks = [[torch.stack([dev_inputs[i][2][j] for i in g]).contiguous() for j in range(4)] for g in groups]
        out_multi = torch.empty((kb, w.nq, w.nb1, w.nb2, w.nm), dtype=torch.float64, device=dev)

    def step():
        if multi:
            for ks, Uk_d, (q_s, Ukq_s, ev_s, om_s) in zip(ks_np, Uks_d, stacks):
                ctx.set_k_batch(ks, Uk_d)
                ctx.q_batch_multi(q_s, Ukq_s, ev_s, om_s, out_multi)
            return
        if kb == 1:
            for k, Uk_d, (q_d, Ukq_d, ev_d, om_d) in dev_inputs:
                ctx.set_k(k, Uk_d)
                ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)
            return
        for g, ks, Uk_d in zip(groups, ks_np, Uks_d):
            ctx.set_k_batch(ks, Uk_d)
            for j, i in enumerate(g):
                ctx.select_k(j)
                q_d, Ukq_d, ev_d, om_d = dev_inputs[i][2]
                ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def maxreduce(x):
        return max_over_ranks(x, dist, dev)

    # ---- device-resident timing ------------------------------------------------
    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = sum(ctx.launch_counts().values())
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = maxreduce(e0.elapsed_time(e1))
    clocks = sampler.stop() if rank == 0 else {}
    gpu_launches = sum(ctx.launch_counts().values()) - launches0
    pairs_per_step_all = world * w.nk * w.nq
    value = pairs_per_step_all * args.steps / (ms_total * 1e-3)

    # ---- per-kernel durations (CUDA events inside the library, on its stream) ---
    ctx.profile(True)
    prof_steps = max(1, min(args.steps, 3))
    for _ in range(prof_steps):
        step()
    prof = ctx.profile_read()
    ctx.profile(False)
    m3 = bool(ctx.get_tuning("m3"))
    pair_rows = ctx.get_tuning("pair_rows")     # > 0: a4 runs the +R / -R pair form (4 real flop per MAC)
    counts = harness.algorithmic_counts(w, m3=m3, pair_rows=pair_rows)
    peaks, peak_src = _measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", HBM_FALLBACK_GBS))
    kernels = {}
    for kind, (ms, n) in prof.items():
        if n == 0:
            continue
        kernels[kind] = {"ms_total": ms / prof_steps, "launches_per_step": n // prof_steps, "avg_ms": ms / n}
    n_k = len(dev_inputs)
    # algorithmic work per LAUNCH of each kernel
    gemm_launches = max(1, kernels.get("setk_gemm", {}).get("launches_per_step", 1))
    gemm_flop = counts["setk_gemm_flop"] * n_k / gemm_launches
    gemm_alu = gemm_flop / (FP64_PEAK_TFLOPS * 1e12) > counts["setk_stream_bytes"] / (hbm_peak * 1e9)
    per_launch = {
        "setk_stream": ("hbm", counts["setk_stream_bytes"]),
        # multi-k a1: g_W read once per launch, nk_b x the flops; bound = whichever floor is higher
        "setk_gemm": ("alu", gemm_flop) if gemm_alu else ("hbm", counts["setk_stream_bytes"]),
        "contract": ("alu", counts["contract_flop"] * n_k / max(1, kernels.get("contract", {}).get("launches_per_step", 1))),
    }
    # a5-a7: HBM-bound for small cells, FP64-bound for 4-atom / large: report against the higher floor.
    # Its flops are the ALGORITHMIC four-multiply count of SURVEY 8(d) (the kernel executes fewer: three-multiply product)
    rot_launches = max(1, kernels.get("rotate_epilogue", {}).get("launches_per_step", 1))
    rot_flop, rot_bytes = counts["rotate_flop"] * n_k / rot_launches, counts["rotate_bytes"] * n_k / rot_launches
    rot_alu = rot_flop / (FP64_PEAK_TFLOPS * 1e12) > rot_bytes / (hbm_peak * 1e9)
    per_launch["rotate_epilogue"] = ("alu", rot_flop) if rot_alu else ("hbm", rot_bytes)
    for kind, (bound, work) in per_launch.items():
        if kind in kernels:
            dur = kernels[kind]["avg_ms"] * 1e-3
            if bound == "hbm":
                kernels[kind].update(bound="hbm", achieved=work / dur / 1e9, peak=hbm_peak, unit="GB/s")
            else:
                kernels[kind].update(bound="alu", achieved=work / dur / 1e12, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s")
            kernels[kind]["frac"] = kernels[kind]["achieved"] / kernels[kind]["peak"]
    dominant = max(kernels, key=lambda kk: kernels[kk]["ms_total"])
    dk = kernels[dominant]
    traffic = _ncu_traffic(w.name, dominant)
    roofline = {"kernel": dominant, "bound": dk.get("bound"), "achieved": dk.get("achieved"), "peak": dk.get("peak"),
                "unit": dk.get("unit"), "frac": dk.get("frac"), "traffic": traffic,
                "peak_source": ("MEASURED_PEAKS.json hbm_gbs (%s)" % peak_src) if dk.get("bound") == "hbm"
                else "derived: 64 FP64 FMA/clk/SM x 148 SMs x 1.965 GHz x 2 = 37.24 TFLOP/s",
                "share_of_step": dk["ms_total"] / sum(v["ms_total"] for v in kernels.values()),
                "flop_per_complex_mac": counts["contract_flop_per_mac"] if dominant == "contract" else counts["flop_per_complex_mac"],
                "note": "achieved counts EXECUTED flops: 4 per complex MAC in a4's +R/-R pair form (real phases x complex "
                        "pair rows), 6 with the three-multiply product, 8 with the plain one; the algorithmic count of "
                        "SURVEY 8(d) is 8"}
    fp64_probe = None
    if rank == 0:
        try:
            fp64_probe = {"dmma_tflops": binding.probe_fp64("dmma", 4000), "dfma_tflops": binding.probe_fp64("dfma", 4000)}
        except Exception:
            fp64_probe = None

    # ---- end to end: host buffers through the C ABI, copies inside the timed region ----
    pinned = []
    for k, Uk, (q, Ukq, ev, om) in host_inputs:
        pin = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (Uk, q, Ukq, ev, om)]
        pinned.append((k, pin))
    Uks_pin = [torch.from_numpy(u).pin_memory() for u in Uks_np]
    out_hosts = [torch.empty((w.nq, w.nb1, w.nb2, w.nm), dtype=torch.float64).pin_memory() for _ in range(2)]
    out_host = out_hosts[0]
    h2d = sum(sum(t.numel() * t.element_size() for t in pin) + 24 for _, pin in pinned)
    d2h = len(pinned) * out_host.numel() * 8

    def step_e2e():
        # every k-point: inputs host->device, |g|^2 device->host (into two alternating pinned buffers, as a consumer
        # that reads batch n while batch n+1 is computed would hold them); phoebe_elph_q_batch_host_async overlaps the
        # copies with the kernels; the step ends when the last result is on the host (phoebe_elph_wait)
        n = 0
        for g, ks, Uk_p in zip(groups, ks_np, Uks_pin):
            if kb == 1:
                ctx.set_k_host(ks[0], Uk_p.numpy()[0])
            else:
                ctx.set_k_batch_host(ks, Uk_p.numpy())
            for j, i in enumerate(g):
                ctx.select_k(j)
                _, (_, q_p, Ukq_p, ev_p, om_p) = pinned[i]
                if args.e2e_sync:
                    ctx.q_batch_host(q_p.numpy(), Ukq_p.numpy(), ev_p.numpy(), om_p.numpy(), out_host.numpy())
                else:
                    ctx.q_batch_host_async(q_p.numpy(), Ukq_p.numpy(), ev_p.numpy(), om_p.numpy(),
                                           out_hosts[n & 1].numpy())
                n += 1
        ctx.wait()

    e2e_steps = max(1, min(args.steps, 3))
    step_e2e()
    barrier()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(e2e_steps):
        step_e2e()
    e1.record()
    barrier()
    ms_e2e = maxreduce(max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3))
    e2e_value = pairs_per_step_all * e2e_steps / (ms_e2e * 1e-3)

    # ---- the same pass with the linewidth sum (Eq. 29) fused in, |g|^2 never stored ----
    rates = None
    if not args.no_rates:
        P = wl.RATE_PARAMS
        eps_np = [wl.band_energies(w, ik) for ik in k_ids]
        eps_d = [harness.to_device([e1, e2], dev) for e1, e2 in eps_np]
        rate_d = torch.zeros((len(dev_inputs), w.nb1), dtype=torch.float64, device=dev)

        if multi:       # stacked form: eps / rate arrays of a k batch side by side
            eps_k_s = [torch.stack([eps_d[i][0] for i in g]).contiguous() for g in groups]
            eps_kq_s = [torch.stack([eps_d[i][1] for i in g]).contiguous() for g in groups]
            rate_s = [torch.zeros((len(g), w.nb1), dtype=torch.float64, device=dev) for g in groups]

        def step_rates():
            if multi:
                for ig, (ks, Uk_d, (q_s, Ukq_s, ev_s, om_s)) in enumerate(zip(ks_np, Uks_d, stacks)):
                    ctx.set_k_batch(ks, Uk_d)
                    ctx.q_batch_rates_multi(q_s, Ukq_s, ev_s, om_s, eps_k_s[ig], eps_kq_s[ig], rate_s[ig], **P)
                return
            for g, ks, Uk_d in zip(groups, ks_np, Uks_d):
                if kb == 1:
                    ctx.set_k(ks[0], Uk_d[0])
                else:
                    ctx.set_k_batch(ks, Uk_d)
                for j, i in enumerate(g):
                    ctx.select_k(j)
                    q_d, Ukq_d, ev_d, om_d = dev_inputs[i][2]
                    ctx.q_batch_rates(q_d, Ukq_d, ev_d, om_d, eps_d[i][0], eps_d[i][1], rate_d[i], **P)

        step_rates()
        barrier()
        e0.record()
        for _ in range(args.steps):
            step_rates()
        e1.record()
        barrier()
        ms_r = maxreduce(e0.elapsed_time(e1))
        eps_pin = [[torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in e] for e in eps_np]
        rate_h = torch.zeros((len(dev_inputs), w.nb1), dtype=torch.float64).pin_memory().numpy()

        def step_rates_e2e():
            for g, ks, Uk_p in zip(groups, ks_np, Uks_pin):
                if kb == 1:
                    ctx.set_k_host(ks[0], Uk_p.numpy()[0])
                else:
                    ctx.set_k_batch_host(ks, Uk_p.numpy())
                for j, i in enumerate(g):
                    ctx.select_k(j)
                    _, (_, q_p, Ukq_p, ev_p, om_p) = pinned[i]
                    ctx.q_batch_rates_host_async(q_p.numpy(), Ukq_p.numpy(), ev_p.numpy(), om_p.numpy(),
                                                 eps_pin[i][0].numpy(), eps_pin[i][1].numpy(), rate_h[i], **P)
            ctx.wait()

        step_rates_e2e()
        barrier()
        t0 = time.perf_counter()
        e0.record()
        for _ in range(e2e_steps):
            step_rates_e2e()
        e1.record()
        barrier()
        ms_re = maxreduce(max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3))
        rates = {"what": "same pass with phoebe_elph_q_batch_rates%s: Eq. 29 linewidth sum fused into the |g|^2 epilogue, "
                         "|g|^2 not stored; the result per k-point is nb1 doubles" % ("_multi (k batch stacked)" if multi else ""),
                 "value": pairs_per_step_all * args.steps / (ms_r * 1e-3), "unit": UNIT,
                 "e2e": {"value": pairs_per_step_all * e2e_steps / (ms_re * 1e-3), "unit": UNIT,
                         "h2d_bytes_per_step": int(h2d + sum(a.numel() * 8 for e in eps_pin for a in e)),
                         "d2h_bytes_per_step": int(len(pinned) * w.nb1 * 8)}}

    # ---- CPU baseline: the oracle on the host cores (rank 0, N=1 only) ----------
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, sample, _ = time_oracle(w, 20.0)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _with_multi(_with_kbatch(_config_dict(w, world), kb), multi),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "steps": e2e_steps, "api": "q_batch_host" if args.e2e_sync else "q_batch_host_async + wait"},
            "gpu_launches": int(gpu_launches),
            "roofline": roofline,
            "kernels": kernels,
            "fp64_probe": fp64_probe,
            "cpu_baseline": cpu_baseline,
            "rates_fused": rates,
            "fp64_tflops_whole_path_4m_equivalent": (counts["setk_flop"] + counts["contract_flop_4m"] + counts["rotate_flop"]) * w.nk * world
            * args.steps / (ms_total * 1e-3) / 1e12,
            "input_gen_s": round(t_gen, 1),
        }
        print(json.dumps(line))
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=list(wl.CONFIGS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--q-multi", type=int, default=-1,
                    help="phoebe_elph_q_batch_multi over the k slots of a batch: -1 = automatic (small cells), 0 = off, 1 = force")
    ap.add_argument("--e2e-sync", action="store_true", help="end-to-end leg with the synchronous q_batch_host (no copy/compute overlap)")
    ap.add_argument("--no-rates", action="store_true", help="skip the extra fused-linewidth (f2) measurement")
    ap.add_argument("--m3", type=int, default=1, help="1 = three-multiply complex product in the GEMMs (default), 0 = four")
    ap.add_argument("--tile", type=int, default=0, help="force the contraction CTA tile (0 = automatic)")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="phoebe_elph_set_tuning knob for kernel-variant experiments (repeatable)")
    ap.add_argument("--k-batch", type=int, default=32,
                    help="k-points per pass over g_W (phoebe_elph_set_k_batch); 1 = one set_k per k")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
