"""N > 1 is replicas only (slices are independent): bench.py's only
cross-rank logic is the max-over-ranks of the timing and the job's voxel count.  Exercised here with two
CPU processes over gloo (127.0.0.1 rendezvous)."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 100.0 + 25.0 * rank                      # rank 1 is the slow one
        ms = bench.max_over_ranks(ms_local, world)
        nz, total = bench.replica_slices(100, 32, world)
        dist.barrier()
        out.put((rank, ms, nz, total))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_replica_count_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [125.0, 125.0]            # both ranks see the slowest rank's time
    assert all(r[2] == 96 and r[3] == 192 for r in res)     # 3 whole chunks of 32 per replica, 2 replicas


def _range_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import paper_2209_08450_b200 as tcp
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        z0, z1 = tcp.tcp_slice_range(2049, rank, world)      # host logic of the library: no GPU needed
        mine = torch.tensor([z0, z1], dtype=torch.int64)
        allr = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(allr, mine)                           # bookkeeping only: the data path has no collective
        out.put((rank, [tuple(int(v) for v in t) for t in allr]))
    finally:
        dist.destroy_process_group()


def test_slice_ranges_world2_tile_the_stack():
    """the volume shards by contiguous slice range, one process per GPU, no exchange.
    Two processes take their range from tcp_slice_range; together the ranges tile the stack in rank order."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_range_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1] == [(0, 1025), (1025, 2049)]


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.replica_slices(2048, 32, 1) == (2048, 2048)
