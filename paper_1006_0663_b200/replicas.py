"""Multi-GPU host logic: the path does not shard across GPUs in this round (north_star: one GPU), so N > 1 means
N independent replicas of the same workload, one process per GPU, with NO data-path collective.  The only
communication is the bookkeeping below (barrier + max-over-ranks of the device time), which is what bench.py
uses and what tests/test_replicas_gloo.py runs with the gloo backend on CPU."""
from __future__ import annotations


def aggregate(ms_local: float, units_local: float, dist=None, device="cpu"):
    """Return (ms_max, units_total, value) with value = units_total / (ms_max * 1e-3).

    ms_local: this rank's device time for its replica (CUDA events); units_local: grid-point updates it performed."""
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    ms_max, units = float(t.item()), float(u.item())
    return ms_max, units, units / (ms_max * 1e-3)
