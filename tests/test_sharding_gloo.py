"""N>1 path on CPU: world_size-2 `gloo` processes run the same sharding / timing-reduction code as bench.py
(paper_2111_14999_b200/sharding.py).  The per-rank "device work" is stood in for by the oracle on a tiny workload, so
the test also checks that the union of the shards reproduces the unsharded result exactly (no collective on the data
path: PAPER.md L556)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2111_14999_b200 import sharding, workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, scaling, nk, q):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert sharding.dist_env() == (rank, world, rank)
        w = wl.custom(nw=3, nb1=2, nb2=3, nm=3, grid_e=(3, 2, 1), grid_p=(2, 2, 2), nk=nk, nq=6, cfg_id=90)
        gW, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
        ks = np.random.default_rng(5).random((world * nk, 3))
        mine = sharding.shard_k(nk, rank, world, scaling)
        local = {}
        for ik in mine:
            qq, Ukq, ev, om = wl.q_inputs(w, ik)
            local[ik] = oracle.elph(gW, Re, Rp, None, None, ks[ik], wl.U_k(w, ik), qq, Ukq, ev, om)
        dist.barrier()
        t = sharding.max_over_ranks(10.0 + rank, dist)
        merged = sharding.gather_by_k(local, dist)
        if rank == 0:
            q.put((t, sorted(merged), {k: v.copy() for k, v in merged.items()}))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_world2_gloo_sharding(scaling):
    import oracle
    world, nk = 2, 4
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, scaling, nk, q)) for r in range(world)]
    for p in procs:
        p.start()
    t, keys, merged = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert t == 11.0                                       # max over ranks
    expect = list(range(world * nk)) if scaling == "weak" else list(range(nk))
    assert keys == expect                                  # disjoint cover, nothing twice, nothing missing
    w = wl.custom(nw=3, nb1=2, nb2=3, nm=3, grid_e=(3, 2, 1), grid_p=(2, 2, 2), nk=nk, nq=6, cfg_id=90)
    gW, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
    ks = np.random.default_rng(5).random((world * nk, 3))
    for ik in expect:
        qq, Ukq, ev, om = wl.q_inputs(w, ik)
        ref = oracle.elph(gW, Re, Rp, None, None, ks[ik], wl.U_k(w, ik), qq, Ukq, ev, om)
        assert np.array_equal(merged[ik], ref)


def test_shard_k_properties():
    for world in (1, 2, 3, 8):
        for nk in (1, 4, 16, 7):
            weak = [sharding.shard_k(nk, r, world, "weak") for r in range(world)]
            assert sorted(sum(weak, [])) == list(range(world * nk)) and all(len(s) == nk for s in weak)
            strong = [sharding.shard_k(nk, r, world, "strong") for r in range(world)]
            assert sorted(sum(strong, [])) == list(range(nk))
            assert max(map(len, strong)) - min(map(len, strong)) <= 1
    with pytest.raises(ValueError):
        sharding.shard_k(4, 0, 2, "other")
    assert sharding.max_over_ranks(3.5) == 3.5 and sharding.gather_by_k({1: 2}) == {1: 2}


# ---- the Re-pool ------------------------------------------------------------------
def _pool_worker(rank, world, port, q):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.custom(nw=3, nb1=2, nb2=3, nm=3, grid_e=(3, 3, 1), grid_p=(2, 2, 2), nk=1, nq=7, cfg_id=91)
        gW, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
        deg_e = np.random.default_rng(3).integers(1, 4, w.nRe).astype(np.float64)
        k, Uk = wl.k_points(w)[0], wl.U_k(w, 0)
        lo, hi = sharding.shard_range(w.nRe, rank, world)
        # this rank's slab of g_W and its Re vectors: the partial g1' of Eq. 71 (stood in for by the oracle on CPU)
        part = oracle.setk(np.ascontiguousarray(gW[:, lo:hi]), Re[lo:hi], deg_e[lo:hi], k, Uk)
        g1 = torch.from_numpy(part)
        sharding.allreduce_g1(g1, dist)                  # the one collective of the path
        # step 2 shards over q, no collective
        qq, Ukq, ev, om = wl.q_inputs(w, 0)
        qlo, qhi = sharding.shard_range(w.nq, rank, world)
        out = oracle.qbatch(g1.numpy(), Rp, None, qq[qlo:qhi], np.ascontiguousarray(Ukq[qlo:qhi]),
                            np.ascontiguousarray(ev[qlo:qhi]), om[qlo:qhi])
        merged = sharding.gather_by_k({rank: (qlo, qhi, out, g1.numpy().copy())}, dist)
        if rank == 0:
            q.put(merged)
    finally:
        dist.destroy_process_group()


def test_world2_gloo_re_pool():
    import oracle
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_pool_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    merged = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    w = wl.custom(nw=3, nb1=2, nb2=3, nm=3, grid_e=(3, 3, 1), grid_p=(2, 2, 2), nk=1, nq=7, cfg_id=91)
    gW, Re, Rp = wl.gW_full(w), wl.Re_vectors(w), wl.Rp_vectors(w)
    deg_e = np.random.default_rng(3).integers(1, 4, w.nRe).astype(np.float64)
    g1_ref = oracle.setk(gW, Re, deg_e, wl.k_points(w)[0], wl.U_k(w, 0))
    qq, Ukq, ev, om = wl.q_inputs(w, 0)
    ref = oracle.qbatch(g1_ref, Rp, None, qq, Ukq, ev, om)
    got = np.empty_like(ref)
    for r in range(world):
        qlo, qhi, out, g1 = merged[r]
        assert np.max(np.abs(g1 - g1_ref)) <= 1e-13 * np.max(np.abs(g1_ref))      # sum of the shards == Eq. 71
        got[qlo:qhi] = out
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(ref)


def test_shard_range_properties():
    for world in (1, 2, 3, 8):
        for n in (1, 5, 27, 343, 729):
            parts = [sharding.shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    t = torch.ones(3, dtype=torch.complex128)
    assert sharding.allreduce_g1(t) is t


def _run_bench_dry(*flags):
    """bench.py --gpus 2 started WITHOUT torchrun: it must re-exec itself under torch.distributed.run with two ranks
    (the launch line the driver uses) and rank 0 must print ONE JSON line for the whole job."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-run", "--backend", "gloo",
                        *flags], capture_output=True, text=True, timeout=300, env=env, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    return json.loads(lines[0])


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_bench_gpus2_spawns_two_ranks(scaling):
    d = _run_bench_dry("--workload", "4-atom", "--scaling", scaling)
    w = wl.CONFIGS["4-atom"]
    assert d["n_gpus"] == 2 and d["scaling"] == scaling and d["ms_max_over_ranks"] == 11.0
    ks = sorted(sum((p["k_ids"] for p in d["plans"]), []))
    assert ks == (list(range(2 * w.nk)) if scaling == "weak" else list(range(w.nk)))
    assert d["pairs_per_step"] == (2 if scaling == "weak" else 1) * w.nk * w.nq
    assert all(p["re"] == [0, w.nRe] and p["q"] == [0, w.nq] for p in d["plans"])      # no pool: g_W replicated


def test_bench_gpus2_re_pool_plan():
    """--pool 2: the two ranks form one Re-pool: same k-points, disjoint Re shards that cover the list, disjoint q
    slices in multiples of the contraction's 64-row tile, and the pool's all-reduce (through sharding.allreduce_g1,
    the helper the GPU path uses) sums over both ranks."""
    d = _run_bench_dry("--workload", "band-window", "--pool", "2", "--scaling", "strong")
    w = wl.CONFIGS["band-window"]
    p0, p1 = d["plans"]
    assert p0["k_ids"] == p1["k_ids"] == list(range(w.nk)) and p0["pool"] == p1["pool"] == 0
    assert p0["re"][0] == 0 and p0["re"][1] == p1["re"][0] and p1["re"][1] == w.nRe
    assert p0["q"][0] == 0 and p0["q"][1] == p1["q"][0] and p1["q"][1] == w.nq and p0["q"][1] % 64 == 0
    assert p0["pool_sum"] == p1["pool_sum"] == 3.0
    assert d["pairs_per_step"] == w.nk * w.nq
