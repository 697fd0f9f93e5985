"""world_size-2 gloo test of the replica logic bench.py uses for N > 1."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1406_7635_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = 10.0 + 5.0 * rank                     # rank 1 is the slow one
        cells, steps = 4096, 7
        value, ms_max = replicas.aggregate_throughput(cells * steps, ms)
        jobs = replicas.shard_jobs(5, rank, world)
        out[rank] = (value, ms_max, replicas.replica_seed(100, rank), jobs)
    finally:
        dist.destroy_process_group()


def test_two_ranks_agree_on_whole_job_throughput():
    world, port = 2, _free_port()
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    v0, ms0, seed0, jobs0 = res[0]
    v1, ms1, seed1, jobs1 = res[1]
    assert ms0 == ms1 == 15.0                       # max over ranks
    expected = 2 * 4096 * 7 / 15e-3                 # all ranks' units / slowest rank's time
    assert abs(v0 - expected) < 1e-6 * expected and v0 == v1
    assert seed0 != seed1 and (seed0, seed1) == (100, 101)
    assert sorted(jobs0 + jobs1) == list(range(5)) and not set(jobs0) & set(jobs1)


def test_single_process_is_identity():
    v, ms = replicas.aggregate_throughput(1000, 2.0)
    assert ms == 2.0 and abs(v - 5e5) < 1e-9
    assert replicas.shard_jobs(3, 0, 1) == [0, 1, 2]
