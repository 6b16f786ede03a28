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
