"""N > 1 is "replicas only": every rank runs the whole layer on its own GPU and its own batch; the data
path has no collective.  The only communication is the timing protocol: a barrier on both sides of the timed region
and the MAX of the per-rank step time."""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> int:
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def barrier() -> None:
    if world() > 1:
        dist.barrier()


def max_over_ranks(ms_local: float, device="cpu") -> float:
    """Slowest rank's step time: multi-GPU numbers are the max over ranks, never a wall clock."""
    if world() == 1:
        return float(ms_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tokens_per_s(tokens_per_rank: int, ms_step_max: float) -> float:
    """Weak scaling: every rank processes its own `tokens_per_rank` in the (max) step time."""
    return world() * tokens_per_rank / (ms_step_max / 1e3)
