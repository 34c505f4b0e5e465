"""Multi-GPU = independent replicas: one process per GPU, each with its own weights and ring,
no data-path collective.  The only cross-rank logic is the timing contract of bench.py: a barrier on both sides of
the timed region and the MAX over ranks of the device-timed milliseconds; whole-job throughput is then
world * steps / max_ms.  This module holds that logic so it can be tested on CPU with the gloo backend."""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> int:
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def barrier() -> None:
    if world() > 1:
        dist.barrier()


def max_over_ranks(values, device=None) -> list:
    """Element-wise MAX over ranks of a list of floats (all ranks get the result)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_throughput(steps: int, ms_max: float) -> float:
    """Units (frames) per second of all replicas together: every rank ran `steps` steps within ms_max."""
    return world() * steps / (ms_max / 1e3)
