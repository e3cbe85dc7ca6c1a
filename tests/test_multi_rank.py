"""N > 1 path of bench.py on CPU: two gloo ranks stand in for two replicas.
The data path has no collective; what crosses ranks is the timing barrier, the max of the measured times and the
sum of the launch counts."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    dist.barrier()
    # rank r "measured" (100 + 10 r) ms of decode, (200 + r) ms in all, (2 + r) ms TTFT, 1000 + r launches
    res = bench.aggregate_over_ranks(dist, torch.device("cpu"), 100.0 + 10 * rank, 200.0 + rank, 2.0 + rank, 1000 + rank)
    out[rank] = res
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_aggregate_max_time_and_sum_launches():
    import torch.multiprocessing as mp
    import bench
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        dec, tot, ttft, launches = res[r]
        assert dec == pytest.approx(110.0) and tot == pytest.approx(201.0) and ttft == pytest.approx(3.0)
        assert launches == 2001
    # whole-job throughput = tokens of both replicas over the slowest replica's time
    v = bench.job_tokens_per_s(world, 5, 110.0)
    assert v == pytest.approx(2 * 5 * bench.DECODE_STEPS / 0.110)
    # single process: identity
    assert bench.aggregate_over_ranks(None, None, 1.0, 2.0, 3.0, 4) == (1.0, 2.0, 3.0, 4)
