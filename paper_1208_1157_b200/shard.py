"""Host-side sharding of an ensemble over ranks (one process per GPU).  DESIGN.md §10.

Systems are independent: there is no exchange step, so the data path has NO collective.  A rank
owns a contiguous range of system indices aligned to the 64-system granule of the SoA rows; the only
``torch.distributed`` traffic is control plane (max-over-ranks of a timing scalar, sums of a few summary
counters, an optional gather of final results to rank 0).  Works with any backend (``nccl`` on GPUs, ``gloo`` in
the CPU tests).  No arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np

GRANULE = 64  # systems; the padding granule of the SoA rows (csrc/ens_api.cu TILE)


def partition(n_sys: int, world: int, granule: int = GRANULE):
    """[(start, stop)] per rank: contiguous, disjoint, covering [0, n_sys), starts multiples of ``granule``,
    sizes differing by at most one granule plus the ragged tail (trailing ranks may be empty when n_sys < world * granule)."""
    if n_sys < 0 or world < 1 or granule < 1:
        raise ValueError("partition: need n_sys >= 0, world >= 1, granule >= 1")
    n_gran = -(-n_sys // granule)
    base, extra = divmod(n_gran, world)
    out, g0 = [], 0
    for r in range(world):
        g1 = g0 + base + (1 if r < extra else 0)
        out.append((min(g0 * granule, n_sys), min(g1 * granule, n_sys)))
        g0 = g1
    return out


def my_range(n_sys: int, rank: int, world: int, granule: int = GRANULE):
    return partition(n_sys, world, granule)[rank]


def weak_range(n_sys_per_rank: int, rank: int):
    """Weak scaling (bench.py): every rank integrates its own ``n_sys_per_rank`` systems of the seeded generator."""
    return rank * n_sys_per_rank, (rank + 1) * n_sys_per_rank


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def max_over_ranks(x: float, device="cpu") -> float:
    """Timing rule: a multi-GPU time is the max over ranks."""
    dist = _dist()
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_counters(counts, device="cpu"):
    """Element-wise sum over ranks of a short vector of integer counters (e.g. the status histogram)."""
    dist = _dist()
    c = np.asarray(counts, dtype=np.int64)
    if dist is None:
        return c
    import torch
    t = torch.from_numpy(c.copy()).to(device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()


def status_histogram(status) -> np.ndarray:
    """Counts of per-system status codes 0..5 (include/ens.h) on this rank."""
    return np.bincount(np.asarray(status, dtype=np.int64), minlength=6)[:6]


def gather_to_rank0(local: np.ndarray, n_sys: int, world: int, granule: int = GRANULE):
    """Concatenate per-rank result arrays (first axis = this rank's systems) on rank 0; others get None.
    Outside the timed path: results leave the GPUs once, after the run."""
    dist = _dist()
    if dist is None:
        return local
    parts = [None] * world if dist.get_rank() == 0 else None
    dist.gather_object(np.ascontiguousarray(local), parts, dst=0)
    if dist.get_rank() != 0:
        return None
    ranges = partition(n_sys, world, granule)
    for p, (a, b) in zip(parts, ranges):
        if p.shape[0] != b - a:
            raise RuntimeError("gather_to_rank0: a rank returned the wrong number of systems")
    return np.concatenate(parts, axis=0)
