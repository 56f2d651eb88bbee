"""Host-side partition logic for more than one GPU.  Index arithmetic only.

The path shards with NO collective:

* a T-P table ("repeat this calculation for multiple combinations of temperature and pressure") is a list of
  independent opacity functions over the same resident line list  ->  `shard_pairs`;
* one opacity function splits along the wavenumber grid: kappa_j depends only on the lines within +-cutoff of nu_j, and
  k-distribution bins are independent, so a rank owns a contiguous, bin-aligned range of grid points plus the lines whose
  window touches it (a read-only halo of lines, duplicated between neighbours)  ->  `shard_grid`.

Results are concatenated in rank order (an all-gather only if every rank needs the whole table).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


def shard_pairs(n_pairs: int, rank: int, world: int) -> range:
    """Contiguous, balanced slice of the (T, P) pair indices 0..n_pairs-1 owned by `rank` (sizes differ by at most 1)."""
    if not (0 <= rank < world) or n_pairs < 0:
        raise ValueError("bad rank/world/n_pairs")
    base, extra = divmod(n_pairs, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


@dataclass(frozen=True)
class GridShard:
    rank: int
    j_lo: int          # first grid point owned (a multiple of bin_pts)
    j_hi: int          # one past the last grid point owned
    line_lo: int       # lines [line_lo, line_hi) of the nu0-ordered list can reach the owned points
    line_hi: int
    nu_min: float      # wavenumber of grid point j_lo: the rank calls hk_opacity(nu_min, nu_max, dnu) on its own range
    nu_max: float
    evals: int         # line-point evaluations inside the owned range (the balance criterion)


def _windows(nu0, nu_min, N, dnu, cutoff):
    # the index window of include/hk.h, rounded exactly as the library and the oracle do (sub, sub, divide, ceil/floor)
    lo = np.ceil(((nu0 - cutoff) - nu_min) / dnu)
    hi = np.floor(((nu0 + cutoff) - nu_min) / dnu)
    lo = np.clip(lo, 0, None)
    hi = np.clip(hi, None, N - 1)
    return lo.astype(np.int64), hi.astype(np.int64)


def shard_grid(nu0_sorted, nu_min: float, N: int, dnu: float, cutoff: float, bin_pts: int, world: int) -> list:
    """Splits grid points 0..N-1 into `world` contiguous ranges aligned to k-distribution bins (`bin_pts` points) and
    balanced by line-point evaluations (not by width: config 3's line density is a ramp).  Returns one GridShard per rank."""
    nu0 = np.ascontiguousarray(nu0_sorted, dtype=np.float64)
    if N < 1 or bin_pts < 1 or N % bin_pts or world < 1:
        raise ValueError("N must be a positive multiple of bin_pts")
    n_bins = N // bin_pts
    if world > n_bins:
        raise ValueError("more ranks than bins")
    jl, jh = _windows(nu0, nu_min, N, dnu, cutoff)
    live = jh >= jl
    # evaluations per grid point = number of windows covering it (difference array), then per bin
    diff = np.zeros(N + 1, dtype=np.int64)
    np.add.at(diff, jl[live], 1)
    np.add.at(diff, jh[live] + 1, -1)
    per_bin = np.cumsum(diff[:N]).reshape(n_bins, bin_pts).sum(axis=1)
    cum = np.concatenate(([0], np.cumsum(per_bin)))
    total = int(cum[-1])
    cuts = [0]
    for r in range(1, world):
        target = total * r / world
        b = int(np.searchsorted(cum, target, side="left"))
        if b > 0 and abs(cum[b - 1] - target) <= abs(cum[min(b, n_bins)] - target):
            b -= 1                                                # the nearer of the two bin edges
        b = min(max(b, cuts[-1] + 1), n_bins - (world - r))      # every rank keeps at least one bin
        cuts.append(b)
    cuts.append(n_bins)
    out = []
    for r in range(world):
        j_lo, j_hi = cuts[r] * bin_pts, cuts[r + 1] * bin_pts
        touch = live & (jh >= j_lo) & (jl <= j_hi - 1)
        idx = np.flatnonzero(touch)
        l_lo, l_hi = (int(idx[0]), int(idx[-1]) + 1) if idx.size else (0, 0)
        out.append(GridShard(r, j_lo, j_hi, l_lo, l_hi, nu_min + j_lo * dnu, nu_min + j_hi * dnu,
                             int(cum[cuts[r + 1]] - cum[cuts[r]])))
    return out
