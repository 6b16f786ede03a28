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
BF16_FALLBACK_TFLOPS = 1590.0      # the profiling recipe's fallback (B200_PROFILING.md), used only without MEASURED_PEAKS.json


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

    def single(self, out):
        """One query right now (timed regions shorter than the sampling period leave no sample)."""
        try:
            r = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=10).stdout.strip().split(",")
            if len(r) >= 7:
                names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
                out.update(sm_mhz=float(r[0]), sm_max_mhz=float(r[1]), power_w_max=float(r[2]), samples=1,
                           reasons=sorted(n for n, v in zip(names, r[3:7]) if v.strip().lower() == "active"),
                           note="timed region shorter than the 100 ms sampling period: one query right after it")
        except Exception:
            pass
        return out

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return self.single(out)
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
        if not out["samples"]:
            return self.single(out)
        return out


from paper_2111_14999_b200.sharding import (allreduce_g1, dist_env as _dist_env, max_over_ranks, pool_set_k,  # noqa: E402
                                            pool_set_k_batch, shard_k, shard_range)


def _k_inputs(w, ik):
    """Inputs of k-point index ik; indices beyond the workload's own nk (other ranks' shards under weak
    scaling) reuse the recipe with a fresh seed index."""
    nk = w.nk
    ks = wl.k_points(w)
    k = ks[ik % nk] if ik < nk else np.random.default_rng([w.seed, w.cfg_id, 1, ik]).random(3)
    return k, wl.U_k(w, ik), wl.q_inputs(w, ik)


# ----------------------------------------------------------------------------- CPU oracle legs
def time_oracle(w, budget_s: float = 20.0):
    """The oracle as it stands, timed on the host cores on a bounded sample of workload w (SURVEY 8(d) "Oracle timed
    beside it": every k-point of the workload x min(256, nq) of its q-points; set_k on as many Rp slabs of g_W as the
    budget allows).  Returns (pairs_per_s, cores, sample_description, (t_setk, t_q)) for the WHOLE workload:
    set_k is a plain sum over independent slabs and is scaled by nRp/slabs, q_batch is linear in nq and is scaled by
    nq/sample -- the value is an EXTRAPOLATION from the sample, and says so."""
    import oracle
    cores = oracle.num_threads()
    Re, Rp = wl.Re_vectors(w), wl.Rp_vectors(w)
    ks = wl.k_points(w)
    nk_s = min(w.nk, 16)                                   # k-points actually run (band-window: 16 of its 256)
    slab_flop = 8.0 * w.nRe * w.X * nk_s
    # assume >= 0.3 GFLOP/s/core for sizing; the measured time is what is reported
    n_slab = int(max(1, min(w.nRp, (0.4 * budget_s * 0.3e9 * cores) / slab_flop)))
    n_slab = max(1, min(w.nRp, n_slab, int(2e9 // (16 * w.nRe * w.X))))      # <= 2 GB of g_W on the host
    slabs = np.empty((n_slab, w.nRe, w.nw, w.nw, w.nm), dtype=np.complex128)
    import concurrent.futures as cf
    with cf.ThreadPoolExecutor(min(16, os.cpu_count() or 4)) as pool:
        list(pool.map(lambda p: wl.gW_slab(w, p, slabs[p]), range(n_slab)))
    t0 = time.perf_counter()
    g1_part = None
    for ik in range(nk_s):
        g1_part = oracle.setk(slabs, Re, None, ks[ik], wl.U_k(w, ik))
    t_setk = (time.perf_counter() - t0) * (w.nRp / n_slab) * (w.nk / nk_s)
    # q part: g1' of the right shape (values are irrelevant for timing): tile what set_k produced
    reps = -(-w.nRp // n_slab)
    g1 = np.ascontiguousarray(np.concatenate([g1_part] * reps)[: w.nRp])
    nq_s = min(w.nq, 256)
    ws = w.with_(nq=nq_s)                                  # same recipe and distributions, nq_s q-points per k
    t_q = 0.0
    for ik in range(nk_s):
        qa, Ua, ea, oa = wl.q_inputs(ws, ik)
        t0 = time.perf_counter()
        oracle.qbatch(g1, Rp, None, qa, Ua, ea, oa)
        t_q += time.perf_counter() - t0
    t_q *= (w.nq / nq_s) * (w.nk / nk_s)
    pairs_per_s = w.nk * w.nq / (t_setk + t_q)
    sample = (f"{nk_s} of {w.nk} k-points: set_k on {n_slab}/{w.nRp} Rp slabs (scaled x{w.nRp / n_slab:.2f}), "
              f"q_batch on {nq_s}/{w.nq} q per k (scaled x{w.nq / nq_s:.2f}); EXTRAPOLATED to the whole workload; "
              f"gcc -O2 -fopenmp, {cores} threads")
    return pairs_per_s, cores, sample, (t_setk, t_q)


def run_reference(args):
    rank, world, _ = _dist_env()
    if rank != 0:
        return
    w = wl.CONFIGS[args.workload]
    vals = []
    sample = ""
    cores = 0
    budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        v, cores, sample, _ = time_oracle(w, budget)
        if i >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    ms_per_step = 1e3 * (w.nk * w.nq) / value
    line = {
        "impl": "reference", "extrapolated": True, "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(w, world),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "extrapolated": True},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def _config_dict(w, n_gpus, scaling="weak", pool=1):
    if pool > 1:
        par = (f"{max(1, n_gpus // pool)} Re-pools of {pool} ranks: g_W sharded over Re inside a pool, one NCCL all-reduce of g1' per "
               f"set_k_batch, q lists shared out inside the pool, k-points {scaling}-sharded over the pools")
    else:
        par = f"k-sharded x{n_gpus} ({scaling}), g_W replicated, no collective"
    return {"workload": w.name, "nw": w.nw, "nb1": w.nb1, "nb2": w.nb2, "nmodes": w.nm, "nRe": w.nRe, "nRp": w.nRp,
            "nk": w.nk, "nq_per_k": w.nq, "gW_GB": round(w.gW_bytes / 1e9, 3),
            "cache": "inputs larger than L2 (g_W is streamed from HBM every step)",
            "parallelism": par}


def cublas_ceilings(torch, dev, M, N, K):
    """cuBLAS FP64 GEMM throughput at the contraction's shape [M x K].[K x N] (through torch.matmul), as CEILINGS for
    the roofline: DGEMM in real flops (2 M N K), ZGEMM in the four-multiply convention (8 M N K)."""
    out = {}
    for name, dt, fl in (("cublas_dgemm_tflops", torch.float64, 2.0), ("cublas_zgemm_8flop_tflops", torch.complex128, 8.0)):
        a = torch.randn((M, K), dtype=dt, device=dev)
        b = torch.randn((K, N), dtype=dt, device=dev)
        c = torch.empty((M, N), dtype=dt, device=dev)
        for _ in range(2):
            torch.matmul(a, b, out=c)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        best = 1e30
        for _ in range(4):
            e0.record()
            torch.matmul(a, b, out=c)
            e1.record()
            e1.synchronize()
            best = min(best, e0.elapsed_time(e1))
        out[name] = fl * M * N * K / (best * 1e-3) / 1e12
        del a, b, c
    out["cublas_shape"] = [M, N, K]
    return out


def _with_kbatch(cfg, kb):
    cfg = dict(cfg)
    cfg["set_k_batch"] = kb
    return cfg


def _with_multi(cfg, multi):
    cfg = dict(cfg)
    cfg["q_batch_multi"] = bool(multi)
    return cfg


# ----------------------------------------------------------------------------- N ranks on one node
def _free_port():
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        return so.getsockname()[1]


def spawn_ranks(args, argv):
    """`python bench.py --gpus N` started WITHOUT torchrun: re-exec under torch.distributed.run with one process per
    GPU (the launch line the driver itself uses), relay its output, return its exit code."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")         # the communicator line ("... nranks N ...") shows every rank joined
    env.setdefault("OMP_NUM_THREADS", "4")
    return subprocess.call(cmd, env=env)


def rank_plan(w, rank, world, scaling, pool):
    """What one rank does (no arithmetic of the method): its pool, its k-points, its slice of the Re list (Re-pool,
    PAPER.md L576) and of every q list.  pool = P > 1: ranks [j*P, (j+1)*P) form pool j; the pools share out the
    k-points (weak: nk per pool; strong: the workload's nk dealt over the pools), the ranks of a pool share out Re for
    step 1 (one all-reduce of g1') and the q list for step 2."""
    assert pool >= 1 and world % pool == 0, "--pool must divide the number of ranks"
    npools, ipool, prank = world // pool, rank // pool, rank % pool
    k_ids = shard_k(w.nk, ipool, npools, scaling)
    re_lo, re_hi = shard_range(w.nRe, prank, pool)
    # q slices in multiples of 64 rows (the contraction's row tile), the last rank takes the ragged rest
    per = -(-w.nq // pool)
    per = -(-per // 64) * 64
    q_lo, q_hi = min(w.nq, prank * per), min(w.nq, (prank + 1) * per)
    return dict(rank=rank, pool=ipool, pool_rank=prank, pool_size=pool, k_ids=k_ids, re=(re_lo, re_hi), q=(q_lo, q_hi),
                pairs=len(k_ids) * (q_hi - q_lo))


def run_dry(args):
    """--dry-run: the N-rank plumbing without a GPU (the world-2 gloo test drives the spawn path through this): process
    group, pool sub-groups, the plan of every rank, one all-reduce over the pool through the same helper the Re-pool
    uses, barrier + max-over-ranks of a per-rank time.  No CUDA, no kernels, no oracle."""
    import torch
    import torch.distributed as dist
    rank, world, local = _dist_env()
    if world > 1:
        dist.init_process_group(args.backend if args.backend != "nccl" else "gloo")
    w = wl.CONFIGS[args.workload]
    plan = rank_plan(w, rank, world, args.scaling, args.pool)
    group = None
    if world > 1 and args.pool > 1:
        for j in range(world // args.pool):
            g = dist.new_group(list(range(j * args.pool, (j + 1) * args.pool)))
            if j == plan["pool"]:
                group = g
    t = torch.full((4,), float(rank + 1), dtype=torch.float64)
    if world > 1:
        from paper_2111_14999_b200.sharding import allreduce_g1
        allreduce_g1(t, dist, group)
        dist.barrier()
    plan["pool_sum"] = float(t[0])
    ms = max_over_ranks(10.0 + rank, dist if world > 1 else None)
    plans = [plan]
    if world > 1:
        plans = [None] * world
        dist.all_gather_object(plans, plan)
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"dry_run": True, "metric": METRIC, "n_gpus": world, "scaling": args.scaling, "pool": args.pool,
                          "ms_max_over_ranks": ms, "pairs_per_step": sum(p_["pairs"] for p_ in plans), "plans": plans}))


# ----------------------------------------------------------------------------- GPU leg
def run_ours(args):
    import torch
    from paper_2111_14999_b200 import binding, build, harness

    rank, world, local = _dist_env()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    w = wl.CONFIGS[args.workload]
    if args.pool_emulate:     # one GPU plays rank 0 of a pool of --pool ranks; nothing is summed over the pool
        assert world == 1, "--pool-emulate is a single-GPU smoke test of the Re-pool code path"
        plan = rank_plan(w, 0, args.pool, args.scaling, args.pool)
    else:
        plan = rank_plan(w, rank, world, args.scaling, args.pool)
    pool_group = None
    if dist is not None and args.pool > 1:
        for j in range(world // args.pool):      # every rank creates every group (collective call), keeps its own
            g_ = dist.new_group(list(range(j * args.pool, (j + 1) * args.pool)))
            if j == plan["pool"]:
                pool_group = g_
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    binding.load_library()

    t_gen = time.perf_counter()
    pooled = args.pool > 1
    re_lo, re_hi = plan["re"]
    q_lo, q_hi = plan["q"]
    nq_l = q_hi - q_lo                           # q-points per k on this rank (the whole list unless pooled)
    gW = harness.upload_gW(w, dev, re_range=(re_lo, re_hi) if pooled else None)
    k_ids = plan["k_ids"]
    host_inputs = []
    for ik in k_ids:
        k_, Uk_, qin = _k_inputs(w, ik)
        host_inputs.append((k_, Uk_, tuple(np.ascontiguousarray(x[q_lo:q_hi]) for x in qin)))
    dev_inputs = []
    for k, Uk, (q, Ukq, ev, om) in host_inputs:
        dev_inputs.append((k, harness.to_device([Uk], dev)[0], harness.to_device([q, Ukq, ev, om], dev)))
    t_gen = time.perf_counter() - t_gen
    kb = max(1, min(args.k_batch, 32, len(host_inputs)))
    # the q lists of all k slots of a batch go through ONE phase / contraction / rotation launch
    # (phoebe_elph_q_batch_multi) whenever the stacked C fits 8 GB: for band windows one k-point's list alone is too
    # small a GEMM for 148 SMs (57 % -> 92 % of peak), for the 4-atom cell it removes the ragged last round of tiles and
    # the launch gaps (93.8 % -> 95.1 %)
    multi = (kb > 1 and args.q_multi != 0 and nq_l % 64 == 0 and len(host_inputs) % kb == 0
             and (args.q_multi == 1 or kb * nq_l * w.N * 16 <= (8 << 30)))
    ctx = harness.make_context(w, gW, nk_max=kb if kb > 1 else 0, nq_max=kb * nq_l if multi else nq_l,
                               re_range=(re_lo, re_hi) if pooled else None)
    ctx.set_tuning("m3", args.m3)
    if args.tile:
        ctx.set_tuning("tile", args.tile)
    for kv in args.tune:                      # kernel-variant experiments: --tune rot_qg=4 (see include/phoebe_elph.h, set_tuning)
        key, val = kv.split("=")
        ctx.set_tuning(key, int(val))
    out = torch.empty((nq_l, w.nb1, w.nb2, w.nm), dtype=torch.float64, device=dev)
    # k-points grouped into batches of kb: one pass over g_W per batch (set_k_batch)
    groups = [list(range(i, min(i + kb, len(host_inputs)))) for i in range(0, len(host_inputs), kb)]
    ks_np = [np.stack([host_inputs[i][0] for i in g]) for g in groups]
    Uks_np = [np.ascontiguousarray(np.stack([host_inputs[i][1] for i in g])) for g in groups]
    Uks_d = [harness.to_device([u], dev)[0] for u in Uks_np]

    if multi:
        stacks = [[torch.stack([dev_inputs[i][2][j] for i in g]).contiguous() for j in range(4)] for g in groups]
        out_multi = torch.empty((kb, nq_l, w.nb1, w.nb2, w.nm), dtype=torch.float64, device=dev)

    def set_k_batch(ks, Uk_d):
        # Re-pool: every rank of the pool holds the partial g1' of its Re shard; ONE in-place all-reduce completes it
        # (sharding.pool_set_k_batch).  NCCL runs on torch's current stream = the library's stream.
        if pooled:
            pool_set_k_batch(ctx, ks, Uk_d, dist, pool_group)
        else:
            ctx.set_k_batch(ks, Uk_d)

    def step_three_call():
        # north_star's boundary as it stands: set_k, then q_batch, for every k-point
        for k, Uk_d, (q_d, Ukq_d, ev_d, om_d) in dev_inputs:
            if pooled:
                pool_set_k(ctx, k, Uk_d, dist, pool_group)
            else:
                ctx.set_k(k, Uk_d)
            ctx.q_batch(q_d, Ukq_d, ev_d, om_d, out)

    def step():
        if multi:
            for ks, Uk_d, (q_s, Ukq_s, ev_s, om_s) in zip(ks_np, Uks_d, stacks):
                set_k_batch(ks, Uk_d)
                ctx.q_batch_multi(q_s, Ukq_s, ev_s, om_s, out_multi)
            return
        if kb == 1:
            step_three_call()
            return
        for g, ks, Uk_d in zip(groups, ks_np, Uks_d):
            set_k_batch(ks, Uk_d)
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
    pairs_per_step_all = plan["pairs"]
    if dist is not None:
        t_pairs = torch.tensor([plan["pairs"]], dtype=torch.int64, device=dev)
        dist.all_reduce(t_pairs)
        pairs_per_step_all = int(t_pairs.item())
    value = pairs_per_step_all * args.steps / (ms_total * 1e-3)

    # ---- per-kernel durations (CUDA events inside the library, on its stream) ---
    ctx.profile(True)
    prof_steps = max(1, min(args.steps, 3))
    ep0, ep1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ep0.record()
    for _ in range(prof_steps):
        step()
    ep1.record()
    prof = ctx.profile_read()
    ctx.profile(False)
    profiled_step_ms = ep0.elapsed_time(ep1) / prof_steps      # the same steps, end to end, with the per-kernel events in
    m3 = bool(ctx.get_tuning("m3"))
    pair_rows = ctx.get_tuning("pair_rows")     # > 0: a4 runs the +R / -R pair form (4 real flop per MAC)
    counts = harness.algorithmic_counts(w, nq=nq_l, m3=m3, pair_rows=pair_rows)
    if pooled:       # a rank of a Re-pool streams only its share of g_W
        for key in ("setk_bytes", "setk_stream_bytes", "setk_flop", "setk_stream_flop", "setk_gemm_flop"):
            counts[key] = counts[key] * (re_hi - re_lo) // w.nRe
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
    setk_rows = ctx.get_tuning("setk_pair_rows")     # > 0: a1 GEMM in the +R / -R pair form: 4 real flop per (k, ring row, x)
    if setk_rows:
        counts["setk_gemm_flop"] = 4 * setk_rows * w.nRp * w.X        # (rows of THIS context: a Re shard when pooled)
    gemm_flop = counts["setk_gemm_flop"] * n_k / gemm_launches
    gemm_alu = gemm_flop / (FP64_PEAK_TFLOPS * 1e12) > counts["setk_stream_bytes"] / (hbm_peak * 1e9)
    # a4 on the INT8 tensor cores (contract_i8.cuh): 21 digit-pair products of the real pair-form GEMM, 2 ops per INT8 MAC
    i8_on = bool(ctx.get_tuning("i8")) and pair_rows > 0
    contract_launches = max(1, kernels.get("contract", {}).get("launches_per_step", 1))
    i8_ops = 21 * 2 * nq_l * (2 * w.N) * pair_rows * n_k / contract_launches if i8_on else 0
    int8_peak_tops = 2.0 * float(peaks.get("bf16_tflops", BF16_FALLBACK_TFLOPS))
    per_launch = {
        "setk_stream": ("hbm", counts["setk_stream_bytes"]),
        # multi-k a1: g_W read once per launch, nk_b x the flops; bound = whichever floor is higher
        "setk_gemm": ("alu", gemm_flop) if gemm_alu else ("hbm", counts["setk_stream_bytes"]),
        "contract": ("tensor", i8_ops) if i8_on else ("alu", counts["contract_flop"] * n_k / contract_launches),
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
            elif bound == "tensor":
                f64_flop = counts["contract_flop_4m"] * n_k / contract_launches
                kernels[kind].update(bound="tensor", achieved=work / dur / 1e12, peak=int8_peak_tops, unit="TOP/s", dtype="s8",
                                     grid_ctas=ctx.get_tuning("i8_grid"), cluster=ctx.get_tuning("i8_cluster"),
                                     int8_nominal_peak_tops=4500.0, frac_of_nominal=work / dur / 1e12 / 4500.0,
                                     fp64_equivalent_tflops=f64_flop / dur / 1e12,
                                     fp64_equivalent_over_fp64_peak=f64_flop / dur / 1e12 / FP64_PEAK_TFLOPS)
            else:
                kernels[kind].update(bound="alu", achieved=work / dur / 1e12, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s")
            kernels[kind]["frac"] = kernels[kind]["achieved"] / kernels[kind]["peak"]
    # the small kernels of the step, against the HBM floor of their ALGORITHMIC bytes per step:
    #   a2 k_setk_rotate: T read once (16 nRp X per k), g1' written (16 nRp N per k)
    #   a3 phases: the A operand written once (INT8: 6 digit planes of Kr real rows per q; FP64 pair form: 8 Kr per q)
    #   pack: g1' read once, the operand copy written (INT8: 6 planes x 2 real columns of Kr rows; FP64 pair rows: 16 Kr N)
    nb1_l = w.nb1
    small = {"setk_rotate": 16.0 * w.nRp * (w.X + nb1_l * w.nw * w.nm) * n_k,
             "qphase": (6.0 if i8_on else 8.0) * max(pair_rows, 1) * nq_l * n_k if pair_rows else 16.0 * w.nRp * nq_l * n_k,
             "pack": (16.0 * w.nRp * w.N + (12.0 if i8_on else 16.0) * max(pair_rows, 1) * w.N) * n_k if pair_rows else 0.0}
    for kind, bytes_step in small.items():
        if kind in kernels and bytes_step > 0 and "bound" not in kernels[kind]:
            dur = kernels[kind]["ms_total"] * 1e-3
            kernels[kind].update(bound="hbm", achieved=bytes_step / dur / 1e9, peak=hbm_peak, unit="GB/s",
                                 frac=bytes_step / dur / 1e9 / hbm_peak, per="step (all launches of the kind)")
    dominant = max(kernels, key=lambda kk: kernels[kk]["ms_total"])
    dk = kernels[dominant]
    traffic = _ncu_traffic(w.name, dominant)
    roofline = {"kernel": dominant, "bound": dk.get("bound"), "achieved": dk.get("achieved"), "peak": dk.get("peak"),
                "unit": dk.get("unit"), "frac": dk.get("frac"), "traffic": traffic,
                "peak_source": ("MEASURED_PEAKS.json hbm_gbs (%s)" % peak_src) if dk.get("bound") == "hbm"
                else ("INT8 dense = 2 x MEASURED_PEAKS.json bf16_tflops (%s; burst figure: the kernel is timed alone; the "
                      "guide's nominal INT8 : bf16 ratio is 4.5 : 2.25); nominal 4500 TOP/s" % peak_src) if dk.get("bound") == "tensor"
                else "derived: 64 FP64 FMA/clk/SM x 148 SMs x 1.965 GHz x 2 = 37.24 TFLOP/s",
                "share_of_step": dk["ms_total"] / sum(v["ms_total"] for v in kernels.values()),
                "flop_per_complex_mac": counts["contract_flop_per_mac"] if dominant == "contract" else counts["flop_per_complex_mac"],
                "note": ("a4 runs on the INT8 tensor cores by exact digit splitting (Ozaki scheme): every FP64 operand of the "
                         "+R/-R pair form is six signed base-256 digits, 21 digit-pair INT8 GEMMs (tcgen05.mma kind::i8, INT32 "
                         "accumulation in TMEM, exact) are recombined in the FP64 epilogue; achieved = 21 x 2 x q rows x 2 N x "
                         "pair rows INT8 ops per launch / duration; fp64_equivalent_tflops (kernels.contract) divides SURVEY "
                         "8(d)'s 8 real flop per complex MAC by the same duration") if dk.get("bound") == "tensor" else
                        ("achieved counts EXECUTED flops: 4 per complex MAC in a4's +R/-R pair form (real phases x complex "
                         "pair rows), 6 with the three-multiply product, 8 with the plain one; the algorithmic count of "
                         "SURVEY 8(d) is 8")}
    fp64_probe = None
    if rank == 0:
        try:
            fp64_probe = {"dmma_tflops": binding.probe_fp64("dmma", 4000), "dfma_tflops": binding.probe_fp64("dfma", 4000)}
        except Exception:
            fp64_probe = None

    # ---- FP64 ceilings measured in the same run (SURVEY 8(d) "Peaks"): the two in-library probes above and cuBLAS
    # (through torch.matmul: the product library links no cuBLAS) at the contraction's own shape -- ceilings only ----
    ceilings = None
    if rank == 0:
        ceilings = {"derived_tflops": FP64_PEAK_TFLOPS}
        if fp64_probe:
            ceilings.update(dmma_probe_tflops=fp64_probe["dmma_tflops"], dfma_probe_tflops=fp64_probe["dfma_tflops"])
        try:
            ceilings.update(cublas_ceilings(torch, dev, min(16384, max(1024, len(dev_inputs) * nq_l)), w.N, w.nRp))
        except Exception as exc:          # a ceiling that cannot be measured is reported as such, never guessed
            ceilings["cublas_error"] = str(exc)[:200]
        best = max(v for k_, v in ceilings.items() if k_ in ("derived_tflops", "dmma_probe_tflops", "cublas_dgemm_tflops"))
        ceilings["max_tflops"] = best
        for kk in kernels.values():
            if kk.get("bound") == "alu":
                kk["frac_of_max_ceiling"] = kk["achieved"] / best

    # ---- Re-pool check (f3): g1' of the pooled path against the unsharded path, element by element, on this rank ----
    pool_check = None
    if pooled:
        free_b, _ = torch.cuda.mem_get_info()
        if free_b > w.gW_bytes + (16 << 30):
            gW_full = harness.upload_gW(w, dev)
            ctx_full = harness.make_context(w, gW_full, nk_max=kb if kb > 1 else 0, nq_max=64)
            worst = 0.0
            ks0, Uk0 = ks_np[0], Uks_d[0]
            if kb > 1:
                ctx_full.set_k_batch(ks0, Uk0)
                set_k_batch(ks0, Uk0)
            else:
                ctx_full.set_k(ks0[0], Uk0[0])
                pool_set_k(ctx, ks0[0], Uk0[0], dist, pool_group)
            for j in range(len(groups[0])):
                a_ = ctx.g1_view(j)
                b_ = ctx_full.g1_view(j)
                worst = max(worst, float(((a_ - b_).abs().max() / b_.abs().max()).item()))
            ctx_full.close()
            del gW_full
            torch.cuda.empty_cache()
            pool_check = {"what": "max |g1'(Re-pool, all-reduced) - g1'(unsharded)| / max |g1'| over the first k batch, "
                                  "worst rank", "max_rel_err": maxreduce(worst), "ok": maxreduce(worst) < 1e-12}
        else:
            pool_check = {"skipped": "not enough free device memory for the unsharded g_W beside the shard"}

    # ---- the north-star boundary as it stands: set_k + q_batch per k-point (no set_k_batch, no stacking) ----
    three_call = None
    if not args.no_three_call and kb > 1:
        for _ in range(2):
            step_three_call()
        barrier()
        n3 = max(1, min(args.steps, 3))
        e0.record()
        for _ in range(n3):
            step_three_call()
        e1.record()
        barrier()
        ms3 = maxreduce(e0.elapsed_time(e1))
        ctx.profile(True)
        step_three_call()
        prof3 = ctx.profile_read()
        ctx.profile(False)
        c1 = harness.algorithmic_counts(w, nq=nq_l, m3=m3, pair_rows=ctx.get_tuning("pair_rows"))
        k3 = {kind: {"ms_total": ms_, "launches_per_step": n_, "avg_ms": ms_ / n_} for kind, (ms_, n_) in prof3.items() if n_}
        share = (re_hi - re_lo) / w.nRe if pooled else 1.0
        i8_3 = bool(ctx.get_tuning("i8")) and ctx.get_tuning("pair_rows") > 0
        for kind, bound, work in (("setk_stream", "hbm", c1["setk_stream_bytes"] * share),
                                  ("contract", "tensor", 21 * 2 * nq_l * (2 * w.N) * ctx.get_tuning("pair_rows")) if i8_3
                                  else ("contract", "alu", c1["contract_flop"]),
                                  ("rotate_epilogue", "alu" if rot_alu else "hbm", c1["rotate_flop"] if rot_alu else c1["rotate_bytes"])):
            if kind in k3:
                dur = k3[kind]["avg_ms"] * 1e-3
                peak_ = {"alu": FP64_PEAK_TFLOPS, "tensor": int8_peak_tops, "hbm": hbm_peak}[bound]
                ach = work / dur / (1e9 if bound == "hbm" else 1e12)
                k3[kind].update(bound=bound, achieved=ach, peak=peak_, unit={"alu": "TFLOP/s", "tensor": "TOP/s", "hbm": "GB/s"}[bound],
                                frac=ach / peak_)
        three_call = {"what": "phoebe_elph_set_k + phoebe_elph_q_batch per k-point (north_star's three-call boundary; g_W is "
                              "re-read for every k-point)", "value": pairs_per_step_all * n3 / (ms3 * 1e-3), "unit": UNIT,
                      "ms_per_step": ms3 / n3, "kernels": k3}

    # ---- end to end: host buffers through the C ABI, copies inside the timed region ----
    pinned = []
    for k, Uk, (q, Ukq, ev, om) in host_inputs:
        pin = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (Uk, q, Ukq, ev, om)]
        pinned.append((k, pin))
    Uks_pin = [torch.from_numpy(u).pin_memory() for u in Uks_np]
    out_hosts = [torch.empty((nq_l, w.nb1, w.nb2, w.nm), dtype=torch.float64).pin_memory() for _ in range(2)]
    out_host = out_hosts[0]
    h2d = sum(sum(t.numel() * t.element_size() for t in pin) + 24 for _, pin in pinned)
    d2h = len(pinned) * out_host.numel() * 8

    def set_k_host(ks, Uk_p):
        if kb == 1:
            ctx.set_k_host(ks[0], Uk_p.numpy()[0])
        else:
            ctx.set_k_batch_host(ks, Uk_p.numpy())
        if pooled:
            allreduce_g1(ctx.g1_view(-1), dist, pool_group)

    if multi:     # k-stacked pinned arrays of every k batch (the layout of phoebe_elph_q_batch_multi_host_async)
        stacks_pin = [[torch.from_numpy(np.ascontiguousarray(np.stack([host_inputs[i][2][j] for i in g]))).pin_memory()
                       for j in range(4)] for g in groups]
        out_multi_hosts = [torch.empty((kb, nq_l, w.nb1, w.nb2, w.nm), dtype=torch.float64).pin_memory() for _ in range(2)]

    def step_e2e_multi():
        # one call per k batch: the stacked inputs host->device, the stacked |g|^2 device->host (two alternating pinned
        # buffers); copies of neighbouring batches and the next set_k_batch overlap this batch's kernels
        for n, (ks, Uk_p, st_p) in enumerate(zip(ks_np, Uks_pin, stacks_pin)):
            set_k_host(ks, Uk_p)
            ctx.q_batch_multi_host_async(*[t.numpy() for t in st_p], out_multi_hosts[n & 1].numpy())
        ctx.wait()

    def step_e2e():
        if multi and not args.e2e_sync:
            return step_e2e_multi()
        # every k-point: inputs host->device, |g|^2 device->host (into two alternating pinned buffers, as a consumer
        # that reads batch n while batch n+1 is computed would hold them); phoebe_elph_q_batch_host_async overlaps the
        # copies with the kernels; the step ends when the last result is on the host (phoebe_elph_wait)
        n = 0
        for g, ks, Uk_p in zip(groups, ks_np, Uks_pin):
            set_k_host(ks, Uk_p)
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
        eps_np = [(e1_, np.ascontiguousarray(e2_[q_lo:q_hi])) for e1_, e2_ in (wl.band_energies(w, ik) for ik in k_ids)]
        eps_d = [harness.to_device([e1, e2], dev) for e1, e2 in eps_np]
        rate_d = torch.zeros((len(dev_inputs), w.nb1), dtype=torch.float64, device=dev)

        if multi:       # stacked form: eps / rate arrays of a k batch side by side
            eps_k_s = [torch.stack([eps_d[i][0] for i in g]).contiguous() for g in groups]
            eps_kq_s = [torch.stack([eps_d[i][1] for i in g]).contiguous() for g in groups]
            rate_s = [torch.zeros((len(g), w.nb1), dtype=torch.float64, device=dev) for g in groups]

        def step_rates():
            if multi:
                for ig, (ks, Uk_d, (q_s, Ukq_s, ev_s, om_s)) in enumerate(zip(ks_np, Uks_d, stacks)):
                    set_k_batch(ks, Uk_d)
                    ctx.q_batch_rates_multi(q_s, Ukq_s, ev_s, om_s, eps_k_s[ig], eps_kq_s[ig], rate_s[ig], **P)
                return
            for g, ks, Uk_d in zip(groups, ks_np, Uks_d):
                if kb == 1:
                    if pooled:
                        pool_set_k(ctx, ks[0], Uk_d[0], dist, pool_group)
                    else:
                        ctx.set_k(ks[0], Uk_d[0])
                else:
                    set_k_batch(ks, Uk_d)
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

        if multi:
            eps_k_pin = [torch.from_numpy(np.stack([eps_np[i][0] for i in g])).pin_memory() for g in groups]
            eps_kq_pin = [torch.from_numpy(np.ascontiguousarray(np.stack([eps_np[i][1] for i in g]))).pin_memory() for g in groups]
            rate_hm = [torch.zeros((len(g), w.nb1), dtype=torch.float64).pin_memory() for g in groups]

        def step_rates_e2e():
            if multi:
                for n, (ks, Uk_p, st_p) in enumerate(zip(ks_np, Uks_pin, stacks_pin)):
                    set_k_host(ks, Uk_p)
                    ctx.q_batch_rates_multi_host_async(*[t.numpy() for t in st_p], eps_k_pin[n].numpy(), eps_kq_pin[n].numpy(),
                                                       rate_hm[n].numpy(), **P)
                ctx.wait()
                return
            for g, ks, Uk_p in zip(groups, ks_np, Uks_pin):
                set_k_host(ks, Uk_p)
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
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "extrapolated": True}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": _with_multi(_with_kbatch(_config_dict(w, world, args.scaling, args.pool), kb), multi),
            "clocks": clocks,
            # inputs, outputs and every step but a4 are FP64; a4 (default path) = exact s8 digit products with s32 accumulation
            # that reproduce the FP64 contraction to 3-5e-13 of max |g|^2 (tests/test_gpu_i8.py; --tune i8=0: FP64 DMMA)
            "arithmetic": {"a1_a2_a3_a5_a6_a7": "f64", "a4": "s8 x s8 -> s32 digit products of 48-bit operands (exact), f64 epilogue"
                           if i8_on else "f64"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "steps": e2e_steps, "api": "q_batch_host" if args.e2e_sync else
                    ("set_k_batch_host + q_batch_multi_host_async + wait" if multi else "q_batch_host_async + wait")},
            "gpu_launches": int(gpu_launches),
            "roofline": roofline,
            "kernels": kernels,
            # sum of the kernels' own durations vs the step they were measured in (gaps between launches) vs the timed loop
            "kernel_sum_ms": sum(v["ms_total"] for v in kernels.values()), "profiled_step_ms": profiled_step_ms,
            "fp64_probe": fp64_probe,
            "fp64_ceilings": ceilings,
            "three_call": three_call,
            "pool_check": pool_check,
            "cpu_baseline": cpu_baseline,
            "rates_fused": rates,
            "fp64_tflops_whole_path_4m_equivalent": (counts["setk_flop"] + counts["contract_flop_4m"] + counts["rotate_flop"]) * w.nk * world
            * args.steps / (ms_total * 1e-3) / 1e12,
            "input_gen_s": round(t_gen, 1),
        }
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)     # the last thing on stdout, behind NCCL's shutdown messages


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
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank (pool) runs the workload's nk k-points of its own; strong = the workload's "
                         "nk k-points are dealt over the ranks (the paper's axis: MPI loop over k, PAPER.md L556, L705)")
    ap.add_argument("--pool", type=int, default=1,
                    help="Re-pool size P (PAPER.md L576): P ranks share one g_W, sharded over Re; one all-reduce of g1' per "
                         "set_k_batch, then the q lists are shared out.  Must divide the number of ranks")
    ap.add_argument("--pool-emulate", action="store_true",
                    help="single-GPU smoke test of the Re-pool code path: this rank acts as rank 0 of a pool of --pool ranks "
                         "and the all-reduce is skipped, so g1' stays partial and pool_check must report the mismatch")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="process-group backend (gloo: --dry-run only)")
    ap.add_argument("--dry-run", action="store_true", help="N-rank plumbing only (no GPU): prints every rank's plan")
    ap.add_argument("--no-three-call", action="store_true", help="skip the extra set_k + q_batch per k measurement")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args, sys.argv[1:]))
    if args.dry_run:
        run_dry(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
