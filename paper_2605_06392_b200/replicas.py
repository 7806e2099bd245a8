"""Multi-GPU = independent replicas: the sweep over time blocks is sequential, so one gradient does
not shard; N GPUs evaluate N different theta points (line-search points, the 2d+1 stencil of the Hessian,
PAPER.md:189-194) with no data-path collective.  Only timings are reduced (max over ranks)."""
from __future__ import annotations

import numpy as np


def replica_thetas(theta, rank: int, count: int, h: float = 5e-3):
    """`count` evaluation points for replica `rank`: the central-difference stencil of Eq. 13 dealt round-robin
    over ranks -- point q of the global sequence is theta, theta + h e_0, theta - h e_0, theta + h e_1, ..."""
    theta = np.asarray(theta, dtype=np.float64)
    d = theta.shape[0]
    out = []
    q = rank
    while len(out) < count:
        p = q % (2 * d + 1)
        t = theta.copy()
        if p > 0:
            j, sign = (p - 1) // 2, 1.0 if (p - 1) % 2 == 0 else -1.0
            t[j] += sign * h
        out.append(t)
        q += max(1, world_size())
    return out


def world_size() -> int:
    import torch.distributed as dist
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def max_over_ranks(values, device="cpu"):
    """Element-wise max of a list of floats over all ranks (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def aggregate_throughput(units_per_rank: int, ms_max: float) -> float:
    """Whole-job units/s: every rank processed `units_per_rank` units within the slowest rank's time."""
    return world_size() * units_per_rank / (ms_max * 1e-3)
