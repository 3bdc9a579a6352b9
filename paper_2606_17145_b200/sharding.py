"""Host-side target sharding for N GPUs ("same-rank" targets first): once the
tree exists every active target is independent, so each rank holds the whole tree (built redundantly from the same
inputs) and walks a contiguous MORTON range of the active targets, balanced by the work each target took in the
previous pass (OG_F_WALK_COST).  No reduction: every target has one owner.  Range boundaries are multiples of 32
positions of the sorted active order, so that every rank's warps hold exactly the targets they would hold in a
single-GPU call and the concatenated results are bit-identical to it (og.h, og_shortrange_accel) -- provided every
rank walks with the grouping the full list would get: the library picks 32 or 8 targets per warp from each list's own
Morton span, so the ranks build their trees with OG_WALK_G32 / OG_WALK_G8 as og_stats.walk_targets_per_warp of a call
on the full list says (bench.py --scaling strong).

Pure NumPy index logic: no method arithmetic, no CUDA (the world-size-2 gloo test runs it on CPU)."""
from __future__ import annotations

import numpy as np

ALIGN = 32   # targets per warp of the dense walk; 8-target warps of the sparse walk divide it


def sorted_active_order(slot_of_active: np.ndarray) -> np.ndarray:
    """order[k] = position in the caller's active list of the k-th target in Morton (sorted-slot) order; ties
    (duplicates in the active list) keep the caller's order, as the library's stable sort does."""
    return np.argsort(np.asarray(slot_of_active), kind="stable")


def partition_by_cost(cost_sorted: np.ndarray, n_ranks: int, align: int = ALIGN) -> np.ndarray:
    """Boundaries b[0..n_ranks] of contiguous ranges of the sorted active order with about equal summed cost;
    b[0] = 0, b[n_ranks] = len(cost), every inner boundary a multiple of `align`.  Ranges may be empty."""
    n = int(len(cost_sorted))
    b = np.zeros(n_ranks + 1, dtype=np.int64)
    b[n_ranks] = n
    if n == 0 or n_ranks == 1:
        return b
    cum = np.cumsum(np.asarray(cost_sorted, dtype=np.float64))
    total = cum[-1] if cum[-1] > 0 else float(n)
    if cum[-1] <= 0:
        cum = np.arange(1, n + 1, dtype=np.float64)
    for r in range(1, n_ranks):
        k = int(np.searchsorted(cum, total * r / n_ranks, side="left")) + 1     # first position past the share
        k = int(round(k / align)) * align
        b[r] = min(max(k, b[r - 1]), n)
    return b


def rank_sublist(active_idx: np.ndarray | None, n: int, order: np.ndarray, bounds: np.ndarray, rank: int):
    """-> (positions in the caller's active list, original particle indices) of rank's share."""
    pos = order[int(bounds[rank]):int(bounds[rank + 1])]
    idx = pos.astype(np.uint32) if active_idx is None else np.asarray(active_idx)[pos]
    return pos, np.ascontiguousarray(idx, dtype=np.uint32)
