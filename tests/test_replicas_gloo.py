"""Multi-GPU mode is "replicas only": N independent solves, no collective on the data path; the only
communication is the barrier and the MAX-over-ranks of the timed region in bench.py.  That host-side logic is covered
here with two CPU processes over gloo (rendezvous on 127.0.0.1)."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seconds = [0.5, 2.0][rank]                    # rank 1 is the slow replica
    dist.barrier()
    slowest = bench.max_over_ranks(seconds, dist)
    value = bench.aggregate_replicas(1000.0, seconds, world, dist)
    dist.barrier()
    out[rank] = (slowest, value)
    dist.destroy_process_group()


def test_two_replicas_report_the_slowest_rank_and_the_whole_job_rate():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1] == (2.0, 2 * 1000.0 / 2.0)


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(0.25, None) == 0.25
    assert bench.aggregate_replicas(10.0, 0.5, 1, None) == 20.0
