"""Host-side logic of the slab decomposition (no GPU): the partition arithmetic of ark_m1_slab_range and the torch.distributed
transport behind ark_m1_group_create_host, exercised with two gloo ranks on the CPU."""
import os
import socket

import numpy as np
import pytest

import paper_2011_13926_b200 as ark


@pytest.mark.parametrize("ny,nranks", [(4096, 8), (4096, 3), (29, 3), (7, 7), (10, 4), (1, 1)])
def test_slab_ranges_tile_the_grid(ny, nranks):
    ranges = [ark.slab_range(ny, nranks, r) for r in range(nranks)]
    assert ranges[0][0] == 0 and ranges[-1][1] == ny
    for (a0, a1), (b0, b1) in zip(ranges, ranges[1:]):
        assert a1 == b0                               # contiguous, no overlap
    sizes = [b - a for a, b in ranges]
    assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
    assert ranges == [(ny * r // nranks, ny * (r + 1) // nranks) for r in range(nranks)]


def test_slab_range_rejects_bad_arguments():
    for args in ((10, 11, 0), (10, 2, 2), (10, 0, 0), (0, 1, 0), (10, 2, -1)):
        with pytest.raises(ValueError):
            ark.slab_range(*args)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _transport_worker(rank, world, port, periodic, out):
    import ctypes as C
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    tr, keep = ark.gloo_host_transport(dist, rank, world)
    n = 37
    dp = C.POINTER(C.c_double)
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else -1)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else -1)
    send_lo = np.full(n, 100.0 * rank + 1.0) + np.arange(n)        # "my first row"
    send_hi = np.full(n, 100.0 * rank + 2.0) + np.arange(n)        # "my last row"
    recv_lo, recv_hi = np.full(n, -1.0), np.full(n, -1.0)
    rc = tr.sendrecv(None, lo, hi, send_lo.ctypes.data_as(dp), send_hi.ctypes.data_as(dp), recv_lo.ctypes.data_as(dp), recv_hi.ctypes.data_as(dp), n)
    assert rc == 0
    # my lower halo is the LAST row of the rank below; my upper halo is the FIRST row of the rank above
    if lo >= 0:
        assert np.array_equal(recv_lo, np.full(n, 100.0 * lo + 2.0) + np.arange(n))
    else:
        assert np.all(recv_lo == -1.0)
    if hi >= 0:
        assert np.array_equal(recv_hi, np.full(n, 100.0 * hi + 1.0) + np.arange(n))
    else:
        assert np.all(recv_hi == -1.0)
    # the reduction of the Gram-Schmidt sums: every rank ends with the same bits
    buf = np.array([1.0 + rank, 0.1 * (rank + 1), 1e-17 * (rank + 1), -3.0])
    assert tr.allreduce_sum(None, buf.ctypes.data_as(dp), 4) == 0
    want = sum(np.array([1.0 + r, 0.1 * (r + 1), 1e-17 * (r + 1), -3.0]) for r in range(world))
    assert np.allclose(buf, want, rtol=1e-15)
    gathered = [None] * world
    dist.all_gather_object(gathered, buf.tobytes())
    assert all(g == gathered[0] for g in gathered)
    dist.barrier()
    dist.destroy_process_group()
    out.put(rank)


@pytest.mark.parametrize("periodic", [True, False])
def test_gloo_transport_two_ranks(periodic):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_transport_worker, args=(r, 2, port, periodic, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
    assert all(p.exitcode == 0 for p in procs), [p.exitcode for p in procs]
    assert sorted(out.get(timeout=5) for _ in range(2)) == [0, 1]
