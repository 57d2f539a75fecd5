"""The N > 1 path of bench.py is "replicas only": no data-path collective, each
rank runs the same configuration, the job time is the max over ranks.  This checks that rule with
two gloo ranks on the CPU (no GPU, no libsph call)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = 10.0 + 5.0 * rank                     # rank 1 is the slow replica
    job_ms = bench.max_over_ranks(ms)
    rate = bench.whole_job_rate(1000 * 4, world, job_ms * 1e-3)
    dist.barrier()
    out[rank] = (job_ms, rate)
    dist.destroy_process_group()


def test_two_replicas_max_over_ranks_and_aggregate_rate():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    job_ms, rate = res[0]
    assert job_ms == 15.0
    assert abs(rate - 2 * 4000 / 0.015) < 1e-6


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_rate(10, 1, 2.0) == 5.0
