"""Multi-GPU plumbing of the bench: replicas only.

A batch-1 draft step is a strictly sequential chain of small-M GEMVs: it does
not shard, so N GPUs run N independent replicas (independent requests) with no data-path collective.
The only communication is the timing reduction below: the job's time is the MAX over ranks, the job's
work is the SUM over ranks. Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from typing import Tuple

import torch


def job_time_and_work(ms_local: float, units_local: float, device="cpu") -> Tuple[float, float]:
    """(max over ranks of the local elapsed milliseconds, sum over ranks of the local work units)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(ms_local: float, units_local: float, device="cpu") -> float:
    """Whole-job units per second: all ranks' work divided by the slowest rank's time."""
    ms, units = job_time_and_work(ms_local, units_local, device)
    return units / (ms * 1e-3)
