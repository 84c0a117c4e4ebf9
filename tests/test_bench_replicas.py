"""bench.py's N > 1 host logic on CPU: world_size-2 gloo process group, max-over-ranks time, whole-job throughput
(DESIGN.md Sect. 9: the path does not shard -> N independent replicas, no data-path collective)."""
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
    ms_local = 10.0 if rank == 0 else 12.5          # rank 1 is the slow replica
    value, ms_max = bench.replicas_throughput(ms_local, cells=1000, steps=4, world=world)
    dist.barrier()
    out[rank] = (value, ms_max)
    dist.destroy_process_group()


def test_replicas_throughput_takes_the_slowest_rank():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29531 + os.getpid() % 200, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        value, ms_max = res[r]
        assert ms_max == 12.5
        assert value == pytest.approx(2 * 1000 * 4 / 12.5e-3)


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms_max = bench.replicas_throughput(5.0, cells=100, steps=2, world=1)
    assert ms_max == 5.0 and value == pytest.approx(100 * 2 / 5e-3)
