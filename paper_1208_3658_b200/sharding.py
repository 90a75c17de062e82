"""Row sharding of one pair count over the ranks of a torch.distributed job.

Pair counts are additive over any partition of the pair matrix (the paper's sub-matrix loop,
PAPER.md:84, 101; "clusters of independent GPUs").  A rank counts rows
[i_begin, i_end) of catalogue A against all of B with acf_pair_count_rows; the only exchange is
a sum of nbins u64 (and f64) at the end.  This module is host logic only: the ranges and the
final reduction.  The counting itself is the library's kernels.
"""
from __future__ import annotations

import math


def pairs_before_row(i: int, n_a: int, n_b: int, is_auto: bool) -> int:
    """Number of pairs held by rows [0, i): i * n_b (cross), or sum_{r<i} (n_a - 1 - r) (auto: row r pairs with j > r)."""
    if not is_auto:
        return i * n_b
    return i * (n_a - 1) - i * (i - 1) // 2


def row_ranges(n_a: int, n_b: int, is_auto: bool, world_size: int):
    """world_size contiguous row ranges [(begin, end), ...] covering [0, n_a) with near-equal pair
    counts.  Auto-counts get triangle-balanced slices (early rows hold more pairs)."""
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    total = pairs_before_row(n_a, n_a, n_b, is_auto)
    cuts = [0]
    for r in range(1, world_size):
        target = total * r // world_size
        if not is_auto:
            i = 0 if n_b == 0 else min(n_a, -(-target // n_b))
        else:
            # smallest i with pairs_before_row(i) >= target: i^2 - (2n - 1) i + 2 target <= 0
            b = 2 * n_a - 1
            disc = max(0, b * b - 8 * target)
            i = max(0, min(n_a, int((b - math.isqrt(disc)) // 2)))
            while i < n_a and pairs_before_row(i, n_a, n_b, True) < target:
                i += 1
            while i > 0 and pairs_before_row(i - 1, n_a, n_b, True) >= target:
                i -= 1
        cuts.append(max(cuts[-1], i))
    cuts.append(n_a)
    return [(cuts[r], cuts[r + 1]) for r in range(world_size)]


def all_reduce_counts(counts, wsums=None, group=None):
    """Sum the per-rank histograms in place over the process group (counts: int64 tensor holding
    the u64 tallies; wsums: float64 tensor or None).  Integer sums are exact whatever the order."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
        if wsums is not None:
            dist.all_reduce(wsums, op=dist.ReduceOp.SUM, group=group)
    return counts, wsums


def sharded_pair_count(ctx, d_a, d_wa, d_b, d_wb, cos_edges, is_auto, rank: int, world_size: int, group=None):
    """One pair count split by rows over the ranks: every rank holds both catalogues, counts its
    row range on its own GPU and the histograms are summed.  -> (counts, wsums or None)."""
    from . import binding as B
    n_a = d_a.numel() // 3
    n_b = n_a if is_auto else d_b.numel() // 3
    lo, hi = row_ranges(n_a, n_b, bool(is_auto), world_size)[rank]
    out = B.acf_pair_count_rows(ctx, d_a, d_wa, lo, hi, d_b, d_wb, cos_edges, is_auto)
    counts, wsums = out if d_wa is not None else (out, None)
    return all_reduce_counts(counts, wsums, group)


def sharded_pair_count_prepared(ctx, cat_a, cat_b, cos_edges, rank: int, world_size: int, weighted=None, group=None):
    """The same on prepared catalogues (acf_prepare on every rank): rank r counts part r of world_size interleaved
    slices of the pair matrix -- the i-tiles of the sorted catalogue dealt out in turn, so that the slices are
    balanced whatever the pruning leaves of them -- and the histograms are summed.  Nothing is prepared again."""
    from . import binding as B
    out = B.acf_pair_count_prepared(ctx, cat_a, cat_b, cos_edges, part=rank, n_parts=world_size, weighted=weighted)
    counts, wsums = out if isinstance(out, tuple) else (out, None)
    return all_reduce_counts(counts, wsums, group)
