"""The N > 1 plumbing of bench.py on CPU: world_size-2 gloo, max-over-ranks step time, whole-job
aggregate (the path does not shard -- replicas only, no data-path collective)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local_ms = 2.0 + rank                      # rank 1 is the slow replica
        ms = bench.max_over_ranks(torch, local_ms, dist, "cpu")
        dist.barrier()
        out[rank] = (ms, bench.aggregate(1000.0, world, ms))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        ms, rate = res[rank]
        assert ms == 3.0                           # the slowest rank's time, on every rank
        assert abs(rate - 2 * 1000.0 / 3.0e-3) < 1e-6


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(torch, 1.25, None, "cpu") == 1.25
    assert bench.aggregate(10.0, 1, 2.0) == 5000.0
