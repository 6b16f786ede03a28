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
