"""N > 1 path of bench.py on CPU: the path does not exchange data between GPUs (replicas only), so the only multi-rank
logic is the max-over-ranks time / sum-of-units aggregation.  Covered with a world-size-2 gloo group."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    elapsed = 1.0 + rank          # rank 1 is the slow one
    units = 100.0 * (rank + 1)
    t, u = bench.aggregate_over_ranks(elapsed, units, dist)
    out[rank] = (t, u)
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_over_two_ranks_gloo():
    mgr = mp.Manager()
    out = mgr.dict()
    port = 29500 + (os.getpid() % 1000)
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    for rank in (0, 1):
        t, u = out[rank]
        assert t == pytest.approx(2.0) and u == pytest.approx(300.0)   # max time, summed units -> value = 150 units/s


def test_single_process_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(0.5, 10.0, None) == (0.5, 10.0)


def test_iteration_byte_formula():
    sys.path.insert(0, ROOT)
    import bench
    # one iteration at j = 0, one column per pass over the basis: operator + dots 24 (1 + 1) + update 24 (1 + 2); one cycle end:
    # combine 8 (3 + 15) + true residual + norm 24
    assert bench.iteration_bytes_per_cell(1, operator=0) == 336 + 48 + 72 + 8 * 18 + 120 + 360 + 24
    assert bench.iteration_bytes_per_cell(1, operator=1, block=1) == 136 + 48 + 72 + 8 * 18 + 216 + 24
    # matrix-free default: blocks of five columns.  First block (j = 0) of a cycle that needs all five: five operator applications,
    # dots 24 (1 + 5), update 24 + 240 (the in-block solve rides on the update pass: predicted by the dot pass)
    assert bench.iteration_bytes_per_cell(5, operator=1, pair=False) == 5 * 136 + 144 + 264 + 8 * (15 + 15) + 216 + 24
    # ... and two operator applications per pass inside the block (periodic grids): 2 x 160 + 136
    assert bench.iteration_bytes_per_cell(5, operator=1) == 2 * 160 + 136 + 144 + 264 + 8 * (15 + 15) + 216 + 24
    # two columns per pass: two operator applications, dots 24 + 48, update 24 + 96, the W2 - gamma W1 pass 72
    assert bench.iteration_bytes_per_cell(2, operator=1, block=2, pair=False) == 2 * 136 + 72 + 120 + 72 + 8 * (6 + 15) + 216 + 24
    assert bench.iteration_bytes_per_cell(2, operator=1, block=2) == 160 + 72 + 120 + 72 + 8 * (6 + 15) + 216 + 24
    assert bench.iteration_bytes_per_cell(60) == 2 * bench.iteration_bytes_per_cell(30)
