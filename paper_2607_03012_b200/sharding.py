"""Multi-GPU plumbing of the operator: every (batch, head) is an independent instance of the whole pipeline
(SURVEY.md section 8(e)), so heads are sharded round-robin over ranks with NO collective on the data path.  The only
communication is the timing reduction of bench.py (max over ranks).  Backend-agnostic (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_heads(n_heads: int, rank: int, world: int) -> list[int]:
    """Heads owned by `rank`: round-robin, so that every rank gets floor or ceil of n_heads / world."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return list(range(rank, n_heads, world))


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (the timed region of bench.py is reported as the slowest rank's)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(ms_per_step_max: float, world: int) -> float:
    """bench.py's `value` for weak scaling of a time-like metric: every rank processes one full-size call per step, the
    job processes `world` calls in the slowest rank's time -> ms per call of the whole job."""
    return ms_per_step_max / world
