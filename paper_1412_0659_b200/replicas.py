"""Multi-GPU plumbing of the benchmark: the force path partitions by independent problems
("replicas only"): every rank runs its own replica of the workload, there is no
data-path collective; only the timing / interaction totals are reduced (max / sum over ranks).
Host logic only, no CUDA: covered on CPU with the gloo backend (tests/test_replicas_gloo.py)."""
from __future__ import annotations

import torch
import torch.distributed as dist

SEED_STRIDE = 7919  # replica r draws its particles with seed + SEED_STRIDE * r


def replica_seed(seed: int, rank: int) -> int:
    return int(seed) + SEED_STRIDE * int(rank)


def reduce_max_sum(values, device="cpu"):
    """values: floats of this rank. Returns (max over ranks, sum over ranks) as lists of floats."""
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        mx = t.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        sm = t.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
        return mx.tolist(), sm.tolist()
    return t.tolist(), t.tolist()


def whole_job_rate(seconds: float, units: float, device="cpu") -> float:
    """Weak-scaling aggregate: units all ranks processed / the slowest rank's time."""
    mx, sm = reduce_max_sum([seconds, units], device)
    return sm[1] / mx[0]
