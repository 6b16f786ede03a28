"""Plumbing shared by tests, bench.py and smoke(): move a synthetic workload to the
device and drive the C ABI over it.  No arithmetic of the method lives here, and
this module never imports ``oracle``.
"""
from __future__ import annotations

import concurrent.futures as cf
import os

import numpy as np

from . import binding
from . import workloads as wl


def upload_gW(w: wl.Workload, device="cuda:0", threads: int | None = None, re_range=None):
    """g_W as a CUDA complex128 tensor [nRp][nRe][nw][nw][nm], generated slab by slab
    on the host (bit-identical to workloads.gW_slab) and copied through a small ring
    of pinned buffers, so the 57.8 GB workload never exists on the host at once.
    re_range = (lo, hi): only the electron lattice vectors lo..hi-1 (the shard of one rank of a
    Re-pool): [nRp][hi-lo][nw][nw][nm]."""
    import torch

    lo, hi = (0, w.nRe) if re_range is None else re_range
    gW = torch.empty((w.nRp, hi - lo, w.nw, w.nw, w.nm), dtype=torch.complex128, device=device)
    threads = threads or min(32, os.cpu_count() or 8)
    slab_shape = (w.nRe, w.nw, w.nw, w.nm)
    nbuf = threads * 2
    pinned = [torch.empty(slab_shape, dtype=torch.complex128).pin_memory() for _ in range(min(nbuf, w.nRp))]
    events = [None] * len(pinned)
    stream = torch.cuda.Stream(device=device)

    def gen(p, slot):
        wl.gW_slab(w, p, pinned[slot].numpy())
        return p, slot

    with cf.ThreadPoolExecutor(threads) as pool:
        pending = {}
        next_p = 0
        free_slots = list(range(len(pinned)))
        done = 0
        while done < w.nRp:
            while free_slots and next_p < w.nRp:
                slot = free_slots.pop()
                if events[slot] is not None:
                    events[slot].synchronize()
                fut = pool.submit(gen, next_p, slot)
                pending[fut] = slot
                next_p += 1
            finished, _ = cf.wait(list(pending), return_when=cf.FIRST_COMPLETED)
            for fut in finished:
                p, slot = fut.result()
                del pending[fut]
                with torch.cuda.stream(stream):
                    gW[p].copy_(pinned[slot][lo:hi], non_blocking=True)
                    ev = torch.cuda.Event()
                    ev.record(stream)
                events[slot] = ev
                free_slots.append(slot)
                done += 1
    stream.synchronize()
    return gW


def make_context(w: wl.Workload, gW, *, nq_max=None, deg_e=None, deg_p=None, hbm_budget_bytes=None,
                 nb1_max=None, nb2_max=None, nk_max=0, re_range=None) -> binding.ElphContext:
    """re_range = (lo, hi): gW holds only these electron lattice vectors (one rank of a Re-pool)."""
    Re = wl.Re_vectors(w)
    if re_range is not None:
        Re = np.ascontiguousarray(Re[re_range[0]:re_range[1]])
        deg_e = None if deg_e is None else np.ascontiguousarray(deg_e[re_range[0]:re_range[1]])
    return binding.ElphContext(gW, Re, wl.Rp_vectors(w), deg_e, deg_p,
                               nb1_max=nb1_max or w.nb1, nb2_max=nb2_max or w.nb2,
                               nq_max=nq_max or w.nq, nk_max=nk_max, hbm_budget_bytes=hbm_budget_bytes)


def to_device(arrs, device="cuda:0"):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in arrs]


def algorithmic_counts(w: wl.Workload, nq: int | None = None, m3: bool = False, pair_rows: int = 0):
    """Flop / byte counts of SURVEY 8(d), per k-point and per q-batch of nq.  The two GEMMs count the flops they
    EXECUTE: 8 real flop per complex MAC with the four-multiply product, 6 with the three-multiply product (m3;
    its few extra additions -- 2 per operand element loaded, 3 per output -- are not counted)."""
    nq = w.nq if nq is None else nq
    fpc = 6 if m3 else 8
    X, N, Y = w.X, w.N, w.nw * w.nm
    return {
        # a1+a2: bytes = |g_W| + |g1'| ; flop = Fourier sum + rotation
        "setk_bytes": 16 * w.nRp * (w.nRe * X + N),
        "setk_stream_bytes": 16 * w.nRp * w.nRe * X,
        "setk_flop": 8 * w.nRp * w.nRe * X + 8 * w.nRp * w.nw * w.nb1 * Y,
        "setk_stream_flop": 8 * w.nRp * w.nRe * X,
        "setk_gemm_flop": fpc * w.nRp * w.nRe * X,
        # a4: 8 flop per complex MAC
        # pair_rows > 0: the +R / -R pair form (contract_pair.cuh) -- real phases x complex rows, 4 flop per (q, row, n)
        "contract_flop": 4 * nq * pair_rows * N if pair_rows else fpc * nq * w.nRp * N,
        "contract_flop_per_mac": 4 if pair_rows else fpc,
        "contract_flop_4m": 8 * nq * w.nRp * N,
        "flop_per_complex_mac": fpc,
        # a5-a7 per batch
        "rotate_flop": nq * (8 * w.nb1 * w.nb2 * w.nm * (w.nw + w.nm) + 4 * w.nb1 * w.nb2 * w.nm),
        "rotate_bytes": nq * (16 * N + 8 * w.nb1 * w.nb2 * w.nm + 16 * w.nw * w.nb2 + 16 * w.nm * w.nm + 8 * w.nm),
        "qphase_evals": nq * w.nRp,
    }
