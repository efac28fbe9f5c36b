"""Host-side plumbing of the N > 1 bench path ("replicas only"): one process per GPU, every rank
propagates its own seeded system, no data-path collective; the only exchanges are the barrier around the timed region
and a MAX reduction of the per-rank device times.  No method arithmetic here; works with the nccl and gloo backends
(the gloo path is what tests/test_replicas_gloo.py runs on CPU with world_size 2)."""
from __future__ import annotations

import dataclasses
import os


def rank_env():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_workload(w, rank: int):
    """Rank r propagates the same workload shape with its own seed (seed + 100 r): independent systems."""
    return dataclasses.replace(w, seed=w.seed + 100 * rank)


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX over ranks of a short list of floats (per-rank device times in ms)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_steps_per_s(steps_per_rank: int, world: int, ms_max: float) -> float:
    """Aggregate throughput: the steps all ranks advanced divided by the slowest rank's time (weak scaling)."""
    return world * steps_per_rank / (ms_max * 1e-3)
