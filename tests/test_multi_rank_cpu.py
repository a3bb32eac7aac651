"""The N>1 path on CPU: world_size-2 `gloo` processes exercise the sharding and the timing
reduction bench.py uses under torchrun (cells are sharded, there is no data-path collective), and
check that sharded oracle runs reproduce the unsharded run cell for cell."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as W
from oracle import npfem_oracle as O
from paper_2011_04332_b200.multi import (aggregate_throughput, cell_range, max_over_ranks,
                                         rank_seed, sum_over_ranks)


def test_cell_ranges_tile_the_suspension():
    for n_cells in (0, 1, 7, 100_000, 100_003):
        for world in (1, 2, 3, 8):
            ranges = [cell_range(n_cells, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == n_cells
            assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
            sizes = [hi - lo for lo, hi in ranges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        cell_range(10, 2, 2)
    assert rank_seed(4, 0) != rank_seed(4, 1) and rank_seed(4, 1) == rank_seed(4, 1)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # timing reduction: the job time is the slowest rank's, the job's units are everybody's
        ms = 10.0 + 5.0 * rank
        assert max_over_ranks(ms) == 10.0 + 5.0 * (world - 1)
        assert sum_over_ranks(100.0 * (rank + 1)) == 100.0 * world * (world + 1) / 2
        thr = aggregate_throughput(1000.0, ms)
        assert thr == pytest.approx(world * 1000.0 / ((10.0 + 5.0 * (world - 1)) * 1e-3))
        # sharded step: each rank advances its own cell range; no exchange is needed
        w = W.make_config(2, cells=6)
        g = w.groups[0]
        lo, hi = cell_range(6, rank, world)
        oc = O.OracleCell(g.tris, g.rest, g.material, w.dt)
        f = w.forces(0, 0)
        pos, vel = oc.step(g.pos0[lo:hi], g.vel0[lo:hi], f[lo:hi], 3)
        np.save(os.path.join(out_dir, f"pos_{rank}.npy"), pos)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_cells_and_reduce_times(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = W.make_config(2, cells=6)
    g = w.groups[0]
    oc = O.OracleCell(g.tris, g.rest, g.material, w.dt)
    pos_all, _ = oc.step(g.pos0, g.vel0, w.forces(0, 0), 3)
    got = np.concatenate([np.load(tmp_path / f"pos_{r}.npy") for r in range(world)])
    assert np.array_equal(got, pos_all)          # cells are independent: sharding changes nothing
