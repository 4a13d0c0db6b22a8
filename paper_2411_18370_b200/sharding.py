"""Multi-GPU sharding of a template bank.

Templates are independent (PAPER.md:213 `vmap s`), so the bank is split along its outermost
non-trivial grid axis in contiguous blocks, one block per rank; the spectrogram is replicated.
Because every axis before the sharded one has length 1, a rank's local canonical index maps to the
global one by adding a constant.  Each rank selects its own per-band top-k; the records of all ranks
are all-gathered (KBs, no data-path collective) and merged under the same total order
(ranking value descending, global canonical index ascending; PAPER.md:330 loudest per region).
Host logic only: no statistic is computed here.
"""
from __future__ import annotations

import copy

import numpy as np

AXES = ("sky", "a_p", "P_orb", "tasc_frac")  # canonical order, slowest first (then f1, f0)
PAD = np.uint64(2 ** 64 - 1)                 # idx of an empty candidate slot (fasttracks_b200.h)


def shard_grid(grid, rank: int, world: int):
    """Return (local grid, index offset).  Splits the first axis with more than one entry;
    ranks beyond the axis length get an empty shard (local grid None)."""
    sizes = [len(getattr(grid, a)) for a in AXES]
    per_outer = int(grid.n_f1) * int(grid.n_f0)
    for i, (name, n) in enumerate(zip(AXES, sizes)):
        if n > 1 or i == len(AXES) - 1:
            inner = per_outer
            for m in sizes[i + 1:]:
                inner *= m
            bounds = [(n * r) // world for r in range(world + 1)]
            lo, hi = bounds[rank], bounds[rank + 1]
            if hi <= lo:
                return None, 0
            g = copy.copy(grid)
            setattr(g, name, np.ascontiguousarray(getattr(grid, name)[lo:hi]))
            return g, lo * inner
    raise AssertionError("unreachable")


def merge_candidates(per_rank, k: int, by_count: bool = False):
    """per_rank: list of structured arrays [n_bands][k] (binding.CAND_DTYPE) whose idx is already
    GLOBAL.  Returns [n_bands][k] under (value desc, idx asc), padded with idx = 2^64-1."""
    per_rank = [c for c in per_rank if c is not None and c.size]
    n_bands = per_rank[0].shape[0]
    out = np.zeros((n_bands, k), dtype=per_rank[0].dtype)
    out["idx"] = PAD
    for b in range(n_bands):
        rows = np.concatenate([c[b] for c in per_rank])
        rows = rows[rows["idx"] != PAD]
        val = rows["count"].astype(np.float64) if by_count else rows["power"]
        order = np.lexsort((rows["idx"], -val))[:k]
        out[b, :order.size] = rows[order]
        out["band"][b] = b
    return out


def to_global(cands, offset: int):
    """Shift the local canonical indices of a rank's candidates by its shard offset."""
    c = cands.copy()
    live = c["idx"] != PAD
    c["idx"][live] += np.uint64(offset)
    return c


def all_gather_candidates(cands, device=None):
    """all_gather the candidate records of every rank (torch.distributed must be initialised;
    gloo with CPU tensors, nccl with device tensors).  Returns a list of arrays, rank order."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size()
    flat = torch.from_numpy(np.ascontiguousarray(cands).view(np.uint8).reshape(-1).copy())
    if device is not None:
        flat = flat.to(device)
    bufs = [torch.empty_like(flat) for _ in range(world)]
    dist.all_gather(bufs, flat)
    return [b.cpu().numpy().view(cands.dtype).reshape(cands.shape) for b in bufs]
