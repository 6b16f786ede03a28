"""Multi-GPU plumbing of the path: (k,q) pairs are independent ("MPI loop over k"), so the path
shards over k-points with g_W replicated and NO data-path collective.  The only communication is the
barrier / max-over-ranks of the timing and (optionally) a gather of per-rank results.  Backend-agnostic
(`nccl` on GPUs, `gloo` in the CPU tests).  No arithmetic of the method lives here.

Re-pool (when g(Re,Rp) is too large for one GPU's memory the coupling "can be
distributed over the index R_e across a 'pool' of MPI processes"): every rank of a pool holds the slab g_W[nRp][Re shard][...] and the Re
vectors of its shard, computes the partial g1' of Eq. 71 for them (set_k / set_k_batch on its own context; Eq. 71
is linear in g_W), and ONE all-reduce (sum) of g1' -- 2*nRp*N doubles per k, <= 169 MB -- completes it on every rank;
step 2 then shards over q with no further collective.  This is the path's only real exchange step.
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


def shard_range(n: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) of range(n) for `rank` (the first n % world ranks get one more)."""
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def allreduce_g1(g1, dist=None, group=None):
    """In-place sum over the pool of a g1' tensor (complex128, or its float64 view): the one collective of the
    Re-pool.  Works on CUDA tensors with nccl (enqueued on torch's current stream, i.e. stream-ordered with the
    library's kernels) and on CPU tensors with gloo."""
    if dist is None or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return g1
    import torch
    buf = torch.view_as_real(g1) if g1.is_complex() else g1
    dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
    return g1


def pool_set_k_batch(ctx, ks, Uks, dist=None, group=None):
    """Eq. 71 on a Re-pool: `ctx` was set up with this rank's Re shard (its Re vectors, its slab of g_W).
    Partial g1' for all k of the batch on every rank, then one in-place all-reduce over the pool."""
    ctx.set_k_batch(ks, Uks)
    allreduce_g1(ctx.g1_view(-1), dist, group)


def pool_set_k(ctx, k, Uk, dist=None, group=None):
    ctx.set_k(k, Uk)
    allreduce_g1(ctx.g1_view(0), dist, group)
