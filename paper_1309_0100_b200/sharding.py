"""Host logic for running the scan on several GPUs (one process per GPU).

The path has no exchange step: grid frequencies are independent fits (eq. 10),
so ranks take disjoint contiguous ranges of the grid and every rank holds the whole series
(<= 1 MB).  The only communication is the final gather of k (z, index) pairs per rank to
merge the peak lists.  A rank scans one halo point on each side of its range so that the
local-maximum test at the range boundary sees the true neighbours.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from fractions import Fraction


@dataclass(frozen=True)
class GridShard:
    k_lo: int        # first grid index this rank owns
    k_hi: int        # one past the last index it owns
    halo_lo: int     # 1 if a halo point precedes k_lo in the scanned range, else 0
    halo_hi: int
    f0: float        # frequency of the first SCANNED point (halo included)
    K: int           # number of scanned points = k_hi - k_lo + halo_lo + halo_hi


def grid_frequency(f0: float, df: float, k: int) -> float:
    """The double nearest to f0 + k*df (reading S1)."""
    return float(Fraction(k) * Fraction(df) + Fraction(f0))


def shard_grid(f0: float, df: float, K: int, world: int, rank: int) -> GridShard:
    """Strong split: contiguous ranges of ceil(K/world) grid points (the last may be short or empty)."""
    per = math.ceil(K / world)
    lo, hi = min(K, rank * per), min(K, (rank + 1) * per)
    return _with_halo(f0, df, K, lo, hi)


def weak_grid(f0: float, df: float, K: int, world: int, rank: int) -> GridShard:
    """Weak scaling: every rank owns K points; the job is the grid of world*K points."""
    return _with_halo(f0, df, world * K, rank * K, (rank + 1) * K)


def _with_halo(f0, df, K_total, lo, hi) -> GridShard:
    hl = 1 if lo > 0 and hi > lo else 0
    hh = 1 if hi < K_total and hi > lo else 0
    return GridShard(lo, hi, hl, hh, grid_frequency(f0, df, lo - hl), hi - lo + hl + hh)


def local_candidates(shard: GridShard, z_local, idx_local):
    """Turn the top-(k+2) peak indices of the SCANNED range into global (z, index) pairs,
    dropping peaks that sit on a halo point.  z_local/idx_local are indexable host sequences."""
    out = []
    for i in idx_local:
        i = int(i)
        if i < 0:
            continue
        g = shard.k_lo - shard.halo_lo + i
        if shard.k_lo <= g < shard.k_hi:
            out.append((float(z_local[i]), g))
    return out


def merge_candidates(lists, k: int):
    """Global top-k under the total order (z descending, index ascending); -1 padded."""
    allc = [c for lst in lists for c in lst]
    allc.sort(key=lambda c: (-c[0], c[1]))
    idx = [c[1] for c in allc[:k]]
    return idx + [-1] * (k - len(idx))


def gather_topk(shard: GridShard, z_local, idx_local, k: int):
    """All ranks call this; returns the merged global top-k index list on every rank.
    Uses torch.distributed (NCCL or gloo) only for the small gather of candidate pairs."""
    import torch.distributed as dist
    mine = local_candidates(shard, z_local, idx_local)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return merge_candidates([mine], k)
    gathered = [None] * dist.get_world_size()
    dist.all_gather_object(gathered, mine)
    return merge_candidates(gathered, k)
