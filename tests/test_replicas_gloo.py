"""Multi-rank host logic of bench.py --gpus N (replicas only) on the gloo backend,
world_size 2, CPU only."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2604_05867_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seconds_local = 2.0 if rank == 0 else 3.5          # rank 1 is the slow replica
        value, t = replicas.aggregate_throughput(1000.0, seconds_local, world)
        dist.barrier()
        out[rank] = (value, t, replicas.replica_d(rank, world, 0.70))
    finally:
        dist.destroy_process_group()


def test_replicas_world2_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        value, t, _ = res[r]
        assert t == 3.5                                     # max over ranks, identical on every rank
        assert value == 2 * 1000.0 / 3.5                    # units of ALL ranks / slowest rank's time
    assert res[0][2] == 0.70 and res[1][2] == 0.64          # one d of configs[2]'s sweep per rank


def test_single_rank_is_identity():
    assert replicas.replica_d(0, 1, 0.7) == 0.7
    assert replicas.aggregate_throughput(10.0, 2.0, 1) == (5.0, 2.0)
