"""Host logic of the N > 1 path: the decode path shards by sequence with no data-path collective; every
rank decodes its own sequences over its own host link.  The only cross-rank step is the timing reduction: the step time
of the job is the MAX over ranks (device time), the whole-job value is all ranks' tokens over that time.  No method
arithmetic here; `bench.py` uses these helpers under NCCL, `tests/test_shard_gloo.py` under gloo with world size 2."""
from __future__ import annotations

import torch
import torch.distributed as dist


def rank_config(cfg, rank: int):
    """Per-rank workload: same shapes, its own sequences (a disjoint seed stream per rank)."""
    return cfg.with_(seed=cfg.seed + 1000 * rank)


def max_over_ranks(ms: float, device="cpu") -> float:
    """MAX over ranks of a per-rank device time in milliseconds (identity when not distributed)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(tokens_per_rank: int, world: int, ms_per_step_max: float) -> float:
    """Tokens decoded per second by all ranks together (weak scaling: per-rank work is fixed)."""
    return tokens_per_rank * world / (ms_per_step_max * 1e-3)
