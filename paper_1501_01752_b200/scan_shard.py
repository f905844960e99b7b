"""Multi-GPU scan: the (k, omega) points of a scan are independent solves, so the list is
partitioned across ranks, every rank owns a replica of the plan, and the only exchange is a host-side gather of
the npts x 3 complex responses.  There is no data-path collective.

Works with any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests); holds none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np


def shard_bounds(npts: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous block [lo, hi) of rank `rank`: sizes differ by at most one, earlier ranks get the longer blocks.

    Contiguous blocks keep each rank's kappa values adjacent, so the solves of one lock-step batch have similar
    iteration counts (the count grows towards a pole)."""
    if world < 1 or not (0 <= rank < world) or npts < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(npts, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def sharded_scan(scan_fn, k_bloch, k0, pol, rank: int = 0, world: int = 1, group=None):
    """Run `scan_fn(k_bloch[lo:hi], k0[lo:hi], pol[lo:hi]) -> (resp[nloc,3] complex, iters[nloc], resid[nloc])` on this
    rank's block and gather the pieces on every rank (all_gather_object of small host arrays).

    Returns (resp[npts,3], iters[npts], resid[npts]) identical on all ranks."""
    k_bloch = np.asarray(k_bloch, dtype=np.float64)
    k0 = np.asarray(k0, dtype=np.float64)
    pol = np.asarray(pol)
    npts = k_bloch.shape[0]
    lo, hi = shard_bounds(npts, rank, world)
    if hi > lo:
        resp, iters, resid = scan_fn(k_bloch[lo:hi], k0[lo:hi], pol[lo:hi])
    else:
        resp, iters, resid = np.zeros((0, 3), np.complex128), np.zeros(0, np.int32), np.zeros(0)
    piece = (lo, np.asarray(resp, np.complex128), np.asarray(iters, np.int32), np.asarray(resid, np.float64))
    if world == 1:
        pieces = [piece]
    else:
        import torch.distributed as dist
        pieces = [None] * world
        dist.all_gather_object(pieces, piece, group=group)
    out_resp = np.zeros((npts, 3), np.complex128)
    out_iters = np.zeros(npts, np.int32)
    out_resid = np.zeros(npts)
    for plo, r, it, rs in pieces:
        out_resp[plo:plo + len(r)] = r
        out_iters[plo:plo + len(r)] = it
        out_resid[plo:plo + len(r)] = rs
    return out_resp, out_iters, out_resid
