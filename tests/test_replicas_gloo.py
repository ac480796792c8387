"""CPU, world_size 2, gloo: the N > 1 logic of bench.py (replicas only): max-over-ranks time,
whole-job sub-step count, per-rank seeds."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1111_5295_b200 import replicas
from paper_1111_5295_b200 import workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e = (10.0, 0.5) if rank == 0 else (12.0, 0.4)
    res = replicas.aggregate(ms, e2e, 1000 * (rank + 1), 100 * (rank + 1))
    cfg = W.config0(n=64, seed=replicas.rank_seed(7, rank))
    out.put((rank, res, float(cfg["species"][0]["x"][0])))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_two_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, res, _ in got:
        assert res == (12.0, 0.5, 3000.0, 300.0)     # max time, summed units, on every rank
    assert got[0][2] != got[1][2]                    # different seeds -> different particles


def test_aggregate_without_process_group():
    assert replicas.aggregate(1.0, 2.0, 3, 4) == (1.0, 2.0, 3.0, 4.0)
