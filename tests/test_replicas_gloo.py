"""N > 1 path (replicas only, row 8(e)): world_size-2 gloo run on CPU of the aggregation
bench.py uses — whole-job value = total updates / max-over-ranks time."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1006_0663_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    ms = 10.0 if rank == 0 else 12.5                 # rank 1 is the slow replica
    res = replicas.aggregate(ms, 1.0e6 * (rank + 1), dist)
    dist.barrier()
    if rank == 0:
        torch.save(res, out)
    dist.destroy_process_group()


def test_two_rank_aggregation_gloo(tmp_path):
    out = str(tmp_path / "res.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    ms_max, units, value = torch.load(out)
    assert ms_max == 12.5
    assert units == 3.0e6
    assert abs(value - 3.0e6 / 12.5e-3) < 1e-6


def test_single_process_is_identity():
    assert replicas.aggregate(4.0, 8.0) == (4.0, 8.0, 2000.0)
