"""Sector-sharded multi-GPU use of the tracker ("sector-sharded multi-GPU").

The tracking path has no link, tracklet or claim that crosses a sector (reading A16: 36 sectors, each in its own local
frame), so ONE time frame can be cut by sector: rank r gets the clusters of a contiguous range of sectors, tracks them
with the unchanged `tpc_track_timeframe`, and the frame's tracks are the concatenation of the ranks' tracks.  There is no
collective inside the tracking; the only exchanges are the initial routing of the clusters (here every rank selects its
own clusters from the frame) and a final gather of the tracks for the steps that look across sectors (C7 / C10 merging,
C8 / C12 refits), which run on the gathered tracks.

This module holds the host logic only (index arithmetic and the ragged gather; no tracker arithmetic), so that `bench.py
--shard sectors`, the world_size-2 gloo test and the single-GPU union test share it.

Why the shard's result is bit-identical to the whole frame's: a shard keeps its clusters in their original relative order,
so every tie that breaks on the original cluster index breaks the same way, and `global_index()` maps the shard's indices
back (the map is increasing).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


def sector_ranges(n_sectors: int, world: int, clusters_per_sector: Sequence[int] | None = None) -> List[Tuple[int, int]]:
    """`world` contiguous sector ranges [lo, hi) covering [0, n_sectors), every rank at least one sector when
    world <= n_sectors (else the surplus ranks get empty ranges).  With `clusters_per_sector` the cuts balance the cluster
    counts (greedy on the prefix sums), otherwise the sector counts."""
    if n_sectors < 1 or world < 1:
        raise ValueError("n_sectors and world must be positive")
    w = np.ones(n_sectors, np.float64) if clusters_per_sector is None else np.asarray(clusters_per_sector, np.float64)
    if w.shape != (n_sectors,) or np.any(w < 0):
        raise ValueError("clusters_per_sector must hold one non-negative count per sector")
    used = min(world, n_sectors)
    prefix = np.concatenate([[0.0], np.cumsum(w)])
    cuts = [0]
    for k in range(1, used):
        target = prefix[-1] * k / used
        c = int(np.searchsorted(prefix, target, side="left"))
        if c > 0 and abs(prefix[c - 1] - target) <= abs(prefix[min(c, n_sectors)] - target):
            c -= 1
        c = max(c, cuts[-1] + 1)                      # at least one sector per used rank ...
        c = min(c, n_sectors - (used - k))            # ... and enough sectors left for the ranks behind
        cuts.append(c)
    cuts.append(n_sectors)
    ranges = [(cuts[k], cuts[k + 1]) for k in range(used)]
    return ranges + [(n_sectors, n_sectors)] * (world - used)


def sector_histogram(row: np.ndarray, n_sectors: int, n_rows: int) -> np.ndarray:
    """Clusters per sector from the `row` input array (row = sector * n_rows + pad row, reading R2); clusters whose row is
    not an integer inside the geometry are not counted."""
    r = np.asarray(row)
    ok = (r >= 0) & (r < n_sectors * n_rows) & (r == np.floor(r))
    return np.bincount((r[ok].astype(np.int64) // n_rows), minlength=n_sectors)[:n_sectors]


def shard_indices(row: np.ndarray, n_rows: int, lo: int, hi: int) -> np.ndarray:
    """Ascending original indices of the clusters of sectors [lo, hi).  Clusters outside the geometry (invalid rows)
    belong to no shard: they are dropped here, where the whole-frame call would flag them."""
    r = np.asarray(row)
    sel = (r >= lo * n_rows) & (r < hi * n_rows) & (r == np.floor(r))
    return np.nonzero(sel)[0].astype(np.int64)


def global_index(sel: np.ndarray, local: np.ndarray) -> np.ndarray:
    """Maps cluster indices of a shard (-1 = none) back to indices of the whole frame."""
    local = np.asarray(local)
    return np.where(local >= 0, np.asarray(sel)[np.maximum(local, 0)], -1)


def all_gather_ragged(t, world: int):
    """Concatenation over ranks (in rank order) of a tensor whose first dimension differs per rank; every rank gets the
    result and the per-rank lengths.  One all_gather of the lengths, one of the data padded to the longest.
    `world` > 1 needs an initialised `torch.distributed` process group (nccl on GPUs, gloo in the CPU test)."""
    import torch
    if world <= 1:
        return t, [int(t.shape[0])]
    import torch.distributed as dist
    n = torch.tensor([int(t.shape[0])], dtype=torch.int64, device=t.device)
    lens = [torch.zeros_like(n) for _ in range(world)]
    dist.all_gather(lens, n)
    lens = [int(x[0]) for x in lens]
    m = max(max(lens), 1)
    pad = torch.zeros((m,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
    pad[: t.shape[0]] = t
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([p[:k] for p, k in zip(parts, lens)], dim=0), lens
