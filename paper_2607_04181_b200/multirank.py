"""N > 1: the path does not shard -- "replicas only".  Every rank runs its own
independent batch on its own GPU; nothing of the data path crosses ranks.  The only cross-rank operations are
the barrier around the timed region and the MAX over ranks of the device time, from which the whole-job
throughput is computed.  Kept here, backend-agnostic, so that the CPU suite can cover it with gloo."""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> int:
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def barrier() -> None:
    if world() > 1:
        dist.barrier()


def max_over_ranks(x: float, device="cpu") -> float:
    """MAX over ranks of a scalar (a device-timed duration)."""
    if world() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank_step: int, steps: int, local_ms_total: float, device="cpu"):
    """(whole-job units/s, ms per step): all ranks' units divided by the slowest rank's time."""
    ms = max_over_ranks(local_ms_total, device)
    return world() * units_per_rank_step * steps / (ms * 1e-3), ms / steps
