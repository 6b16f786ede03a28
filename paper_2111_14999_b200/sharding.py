"""Multi-GPU plumbing of the path: (k,q) pairs are independent ("MPI loop over k"), so the path
shards over k-points with g_W replicated and NO data-path collective.  The only communication is the
barrier / max-over-ranks of the timing and (optionally) a gather of per-rank results.  Backend-agnostic
(`nccl` on GPUs, `gloo` in the CPU tests).  No arithmetic of the method lives here.
"""
from __future__ import annotations

import os


def dist_env():
    """(rank, world_size, local_rank) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def shard_k(nk: int, rank: int, world: int, scaling: str = "weak"):
    """k-point indices a rank processes.
    weak:   every rank runs nk k-points of its own (global indices rank*nk .. rank*nk+nk-1);
    strong: the nk k-points of the workload are dealt round-robin (rank, rank+world, ...)."""
    if scaling == "weak":
        return list(range(rank * nk, (rank + 1) * nk))
    if scaling == "strong":
        return list(range(rank, nk, world))
    raise ValueError(scaling)


def max_over_ranks(x: float, dist=None, device="cpu") -> float:
    """max of a per-rank scalar (the device-timed milliseconds) over all ranks."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_by_k(local: dict, dist=None):
    """Merge {k_index: result} dicts of all ranks on every rank (test / validation helper; not on the timed path)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return dict(local)
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, local)
    merged = {}
    for p in parts:
        for k, v in p.items():
            assert k not in merged, f"k-point {k} computed by two ranks"
            merged[k] = v
    return merged
