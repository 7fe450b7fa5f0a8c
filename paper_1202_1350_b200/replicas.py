"""Multi-GPU = replicas only: every rank proves its own instance of the same circuit,
no data-path collective.  The only communication is the timing plumbing of bench.py: a barrier and a MAX over ranks.
Host logic only (torch.distributed; nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import numpy as np


def replica_input(base_input: np.ndarray, data_seed: int, rank: int) -> np.ndarray:
    """Rank r > 0 gets another seeded input of the same recipe: a seeded permutation of the base vector (same value
    distribution, same size); rank 0 keeps the base input, so N = 1 is exactly the BASELINE.json workload."""
    if rank == 0:
        return base_input
    return np.random.default_rng(data_seed + rank).permutation(base_input)


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_value(units_per_rank: int, world: int, ms_per_step: float) -> float:
    """Weak scaling: every rank processes `units_per_rank` per step; value = all ranks' units / max-over-ranks time."""
    return units_per_rank * world / (ms_per_step * 1e-3)
