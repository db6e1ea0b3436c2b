"""N > 1 host logic on the CPU: two gloo ranks, replicas only -- per-rank seeds differ, the reported times are
the maximum over ranks, and no rank needs data of another rank."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_09058_b200.replicas import max_over_ranks, replica_seed
from paper_2606_09058_b200.synth import make_config


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    prob = make_config(0, seed=replica_seed(rank))
    times = [10.0 + rank, 5.0 - rank, 1.0]            # rank-dependent "measurements"
    dist.barrier()
    red = max_over_ranks(times, dist)
    out[rank] = (red, float(np.abs(prob.H).sum()))
    dist.destroy_process_group()


def test_two_gloo_ranks_max_over_ranks_and_distinct_replicas():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == [11.0, 5.0, 1.0]          # element-wise max, identical on every rank
    assert res[0][1] != res[1][1]                              # different seeds: independent replicas


def test_single_process_is_identity():
    assert max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
