"""Host-side logic of the N>1 path: root cells dealt to ranks by Alg. 2, every rank
builds the K of its own points, one all-reduce sums them (Alg. 1 line 13).  Runs on CPU with the gloo
backend, world_size 2; the per-rank builder here is the oracle (test infrastructure), so what is tested is the
partition (whole root cells, R13), the balance of Alg. 2 and the reduction -- not the kernels."""
import os
import socket

import numpy as np
import pytest

from paper_2303_14280_b200 import inputs
from paper_2303_14280_b200.dist import lpt_partition, root_cell_costs, root_cell_keys, root_cell_sample, shard_points


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_lpt_partition_is_greedy_and_balanced():
    """Alg. 2: tasks sorted by cost, each to the least-loaded rank; max load <= mean + largest task."""
    rng = np.random.default_rng(7)
    costs = rng.integers(1, 1000, 200).astype(float)
    for world in (1, 2, 3, 8):
        owner = lpt_partition(costs, world)
        load = np.bincount(owner, weights=costs, minlength=world)
        assert load.sum() == costs.sum()
        lower = max(costs.sum() / world, costs.max())          # OPT >= both
        assert load.max() <= lower + costs.max()                # greedy never exceeds mean + largest task
        # brute-force replay of the greedy rule
        ref_load = np.zeros(world)
        for t in np.argsort(-costs, kind="stable"):
            r = int(np.argmin(ref_load))
            assert owner[t] == r
            ref_load[r] += costs[t]


def test_shards_are_whole_root_cells_and_cover_the_grid():
    w = inputs.make_workload(2, grid=(8, 6, 8))
    key = root_cell_keys(w.points, w.batch_cell)
    for world in (2, 3, 5):
        masks = [shard_points(w.points, w.batch_cell, r, world) for r in range(world)]
        tot = np.zeros(len(key), dtype=int)
        for m in masks:
            tot += m
            assert not (set(key[m].tolist()) & set(key[~m].tolist()))      # a root cell is never split
        assert np.all(tot == 1)                                             # every point owned exactly once
    m = root_cell_sample(w.points, w.batch_cell, 0.2)
    assert 0 < m.sum() < len(key) and not (set(key[m].tolist()) & set(key[~m].tolist()))


def test_cost_based_partition_balances_work_not_points(oracle_mod):
    """Alg. 2 on a work model: per-batch costs (here the oracle's own pair counts times points, standing in for
    snk_batch_costs, which needs a GPU) are summed per root cell and balance the partition better than point counts do."""
    w = inputs.make_workload(2, grid=(8, 6, 8))
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=w.eps, batch_cell=w.batch_cell, batch_max=256)
    o.screen(w.P)
    off, perm, _ = o.batches()
    Voff, _ = o.V_lists()
    costs = np.diff(off) * np.diff(Voff).astype(float)           # pair-points per batch
    keys, cell_cost = root_cell_costs(w.points, w.batch_cell, off, perm, costs)
    assert np.array_equal(keys, np.unique(root_cell_keys(w.points, w.batch_cell)))
    assert abs(cell_cost.sum() - costs.sum()) <= 1e-9 * costs.sum()
    key = root_cell_keys(w.points, w.batch_cell)
    first = perm[off[:-1]]
    for world in (2, 4):
        def imbalance(cc):
            load = np.zeros(world)
            for r in range(world):
                m = shard_points(w.points, w.batch_cell, r, world, cell_costs=cc)
                assert not (set(key[m].tolist()) & set(key[~m].tolist()))                  # whole root cells
                load[r] = costs[m[first]].sum()
            assert abs(load.sum() - costs.sum()) <= 1e-9 * costs.sum()
            return load.max() / load.mean()
        by_cost, by_points = imbalance((keys, cell_cost)), imbalance(None)
        assert by_cost <= by_points + 1e-12, (world, by_cost, by_points)
        assert by_cost <= 1.0 + cell_cost.max() / (cell_cost.sum() / world)                # greedy bound: mean + largest task
    with pytest.raises(AssertionError):
        shard_points(w.points[:-7], w.batch_cell, 0, 2, cell_costs=(keys[:-1], cell_cost[:-1]))


def _rank_main(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from oracle import oracle as orc
    from paper_2303_14280_b200.dist import all_reduce_K
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = inputs.make_workload(2, grid=(8, 6, 8), lattice=1)
    mine = shard_points(w.points, w.batch_cell, rank, world)
    o = orc.Oracle(w.basis)
    o.set_grid(w.points[mine], w.weights[mine], eps=w.eps, batch_cell=w.batch_cell, batch_max=w.batch_max)
    K = torch.as_tensor(o.build_K(w.P).copy())
    all_reduce_K(K)
    if rank == 0:
        q.put((K.numpy(), int(mine.sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_world2_gloo_sharded_build_equals_single_build(oracle_mod):
    """K is a plain sum over batches and whole root cells reproduce the global batches (R13), so
    the all-reduced partial K of 2 ranks equals the single-rank K up to summation order."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    K2, n0 = q.get(timeout=300)
    for p in procs:
        p.join(timeout=300)
        assert p.exitcode == 0
    w = inputs.make_workload(2, grid=(8, 6, 8), lattice=1)
    assert 0 < n0 < w.points.shape[0]
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=w.eps, batch_cell=w.batch_cell, batch_max=w.batch_max)
    K1 = o.build_K(w.P)
    assert np.abs(K2 - K1).max() <= 1e-12 * max(1.0, np.abs(K1).max())


def test_bench_oracle_sample_is_spatially_compact():
    """bench.py sizes the timed oracle sample as a Morton-order prefix of whole root cells: a permutation whose prefixes are
    compact boxes (so the oracle's octree makes batches of the usual size out of them), never scattered points."""
    import bench
    w = inputs.make_workload(2, grid=(10, 6, 12))
    order = bench._morton_order(w.points, w.batch_cell)
    assert np.array_equal(np.sort(order), np.arange(len(order)))
    key = root_cell_keys(w.points[order], w.batch_cell)
    assert len(np.unique(key)) == 1 + int(np.count_nonzero(np.diff(key)))           # every root cell is one contiguous run
    # inside the most populated root cell a prefix is the lower octants (whole octree leaves), a strided sample spans the cell
    uk, cnt = np.unique(key, return_counts=True)
    cell = w.points[order][key == uk[np.argmax(cnt)]]            # Morton-ordered points of that cell
    n = len(cell) // 16
    vol = lambda p: float(np.prod(p.max(axis=0) - p.min(axis=0)))
    assert vol(cell[:n]) < 0.5 * vol(cell[::16][:n])
