"""World-size-2 gloo test of the only cross-rank step of bench.py: the path
shards by independent problems, so ranks exchange nothing but the MAX of their timings."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2310_03568_b200 import benchlib as L
    from paper_2310_03568_b200 import workloads as W
    ms = L.max_over_ranks(10.0 + 5.0 * rank)           # rank 1 is the slow one
    d = W.c1_rbi_add(n=1000, w=16, seed=rank)            # every rank draws its own problem
    out[rank] = (ms, L.whole_job_throughput(1000, world, ms), int(d["is_"].sum()))
    dist.destroy_process_group()


def test_weak_scaling_aggregation_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0                # MAX over ranks on every rank
    assert res[0][1] == pytest.approx(2 * 1000 / 15e-3 / 1e9)
    assert res[0][2] != res[1][2]                        # different seeds: independent problems


def test_single_process_is_a_no_op():
    from paper_2310_03568_b200 import benchlib as L
    assert L.max_over_ranks(3.5) == 3.5
