"""Host-side partition logic for more than one GPU (SURVEY.md §8(e)/(f) "NEXT-1"; Alg. 1-2).

The path shards over grid batches: K~ is a plain sum over batches.  Because batching is
lattice-anchored (R13), a subset made of WHOLE ROOT CELLS reproduces exactly the global batches, so dealing
root cells to ranks and summing the partial K with ONE all-reduce (Alg. 1 line 13) gives the
same kept-term set as the single-GPU build.  Costs for Alg. 2's greedy LPT are the primitive pair-points per root cell
that one screening pass of the library reports (snk_screen + snk_batch_costs: the work model W_j of PAPER.md:330 for this
path), or points per root cell when no costs are given.
No method arithmetic here; the K build of each rank is the same C-ABI call.
"""
from __future__ import annotations

import numpy as np


def root_cell_keys(points: np.ndarray, h0: float) -> np.ndarray:
    cell = np.floor(np.asarray(points) / h0).astype(np.int64)
    return (cell[:, 0] + (1 << 20)) << 42 | (cell[:, 1] + (1 << 20)) << 21 | (cell[:, 2] + (1 << 20))


def lpt_partition(costs, world: int) -> np.ndarray:
    """Alg. 2: sort tasks by cost W_j (descending), give each to the least-loaded rank.
    Replicated and deterministic: every rank computes the same assignment.  Returns the owner of each task."""
    costs = np.asarray(costs, dtype=np.float64)
    order = np.argsort(-costs, kind="stable")
    load = np.zeros(world)
    owner = np.zeros(len(costs), dtype=np.int64)
    for t in order:
        r = int(np.argmin(load))
        owner[t] = r
        load[r] += costs[t]
    return owner


def root_cell_costs(points: np.ndarray, h0: float, batch_off: np.ndarray, perm: np.ndarray, batch_costs: np.ndarray):
    """Per-root-cell work from per-batch costs (snk_batch_costs) and the batch lists (snk_export_lists): a batch lies in
    the root cell of any of its points (R13).  Returns (sorted unique cell keys of ALL points, cost per cell); cells whose
    batches were all dropped (empty B_j) cost 0."""
    key = root_cell_keys(points, h0)
    uniq = np.unique(key)
    cost = np.zeros(len(uniq))
    nb = len(batch_off) - 1
    if nb > 0:
        first = np.asarray(perm)[np.asarray(batch_off[:-1])]
        np.add.at(cost, np.searchsorted(uniq, key[first]), np.asarray(batch_costs, dtype=np.float64)[:nb])
    return uniq, cost


def shard_points(points: np.ndarray, h0: float, rank: int, world: int, cell_costs=None) -> np.ndarray:
    """Boolean mask of the points this rank owns (whole root cells).  ``cell_costs`` = (cell keys, cost per cell) from
    root_cell_costs; default: points per cell."""
    if world == 1:
        return np.ones(points.shape[0], dtype=bool)
    key = root_cell_keys(points, h0)
    uniq, inv, cnt = np.unique(key, return_inverse=True, return_counts=True)
    w = cnt.astype(np.float64)
    if cell_costs is not None:
        ck, cc = cell_costs
        assert np.array_equal(np.asarray(ck), uniq), "cell_costs were computed for another grid"
        w = np.asarray(cc, dtype=np.float64) + 1e-9 * cnt        # zero-cost cells still have to go somewhere, lightest last
    owner = lpt_partition(w, world)
    return owner[inv] == rank


def root_cell_sample(points: np.ndarray, h0: float, frac: float) -> np.ndarray:
    """Deterministic subset made of whole root cells (R13): cells ordered by a fixed integer hash of (ix,iy,iz)
    (ties by index), taken until the cumulative point count first reaches frac * N.  Boolean mask."""
    key = root_cell_keys(points, h0)
    uniq, inv, cnt = np.unique(key, return_inverse=True, return_counts=True)
    h = (uniq.astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15)) >> np.uint64(11)
    order = np.lexsort((uniq, h))
    csum = np.cumsum(cnt[order])
    k = min(len(uniq), int(np.searchsorted(csum, frac * points.shape[0])) + 1)
    chosen = np.zeros(len(uniq), dtype=bool)
    chosen[order[:k]] = True
    return chosen[inv]


def all_reduce_K(K, group=None):
    """Alg. 1 line 13: sum of the per-rank partial K (torch tensor on the rank's device; NCCL on GPUs, gloo on CPU)."""
    import torch.distributed as dist
    dist.all_reduce(K, op=dist.ReduceOp.SUM, group=group)
    return K
