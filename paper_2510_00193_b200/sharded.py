"""Sharded evaluation over the ranks of a torch.distributed group (the
paper's full-node runs).  One process per GPU; positions and types are replicated; the atoms are cut into contiguous
ranges and every rank holds the CSR rows of its own range only.  The one exchange of the path is an all-reduce (sum) of
the partial forces (3 N doubles) and of the 7 scalars E, virial; neighbourhood grades need none, the configuration
grade one all-reduce of sum_i B (n_basis doubles).  This module is host logic only: partitioning, the window's CSR,
the two collectives.  The arithmetic runs in mtp_compute_rows / mtp_grade_rows (or in whatever `compute_rows`
callable the caller supplies -- the CPU tests run it with the oracle over gloo)."""
from __future__ import annotations

import numpy as np


def row_range(n_atoms: int, rank: int, world: int):
    """Contiguous, near-equal atom ranges: the first n_atoms % world ranks get one atom more."""
    base, extra = divmod(int(n_atoms), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def balanced_row_range(off, rank: int, world: int):
    """Contiguous ranges with near-equal PAIR counts (the work is per pair): cut where the CSR offsets cross
    k * nnz / world.  off: host array [N + 1]."""
    off = np.asarray(off)
    n, nnz = off.shape[0] - 1, int(off[-1])
    cuts = [int(np.searchsorted(off, (k * nnz) // world, side="left")) for k in range(world + 1)]
    cuts[0], cuts[-1] = 0, n
    for k in range(1, world + 1):
        cuts[k] = max(cuts[k], cuts[k - 1])
    return cuts[rank], cuts[rank + 1]


def window_list(off, idx, shift, lo: int, hi: int):
    """The CSR rows [lo, hi) as a list of their own: offsets from 0, global neighbour indices."""
    off = np.asarray(off)
    a, b = int(off[lo]), int(off[hi])
    return (np.ascontiguousarray(off[lo:hi + 1] - a), np.ascontiguousarray(idx[a:b]),
            None if shift is None else np.ascontiguousarray(shift[a:b]))


def all_reduce_sum(dist, *tensors):
    """One collective for several tensors: packed into a single buffer (launch latency, not bandwidth, is what a
    25 MB all-reduce over NVSwitch costs)."""
    import torch
    flat = torch.cat([t.reshape(-1) for t in tensors])
    dist.all_reduce(flat, op=dist.ReduceOp.SUM)
    o = 0
    for t in tensors:
        k = t.numel()
        t.copy_(flat[o:o + k].reshape(t.shape))
        o += k


def sharded_compute(compute_rows, dist, n_atoms, lo, hi):
    """compute_rows(lo, hi) -> dict(E[1], Ei[N], F[N,3], virial[6]) of PARTIAL sums (torch tensors, any device
    the group's backend reduces).  Returns the same dict with E, F, virial summed over the ranks and Ei complete
    (every rank wrote its window into a zeroed array)."""
    out = compute_rows(lo, hi)
    all_reduce_sum(dist, out["F"], out["E"], out["virial"], out["Ei"])
    return out


def sharded_grade(grade_rows, cfg_from_sum, dist, lo, hi):
    """grade_rows(lo, hi) -> dict(gamma_atom[N] window entries, Bsum[n_basis] window sum); cfg_from_sum(Bsum) -> the
    configuration grade.  Returns dict(gamma_atom (complete), Bsum (all atoms), gamma_cfg)."""
    out = grade_rows(lo, hi)
    all_reduce_sum(dist, out["Bsum"], out["gamma_atom"])
    out["gamma_cfg"] = cfg_from_sum(out["Bsum"])
    return out
