"""Member sharding for multi-GPU runs: host logic only, no field arithmetic.

Ensemble members are independent (no cross-member term in eqs (2)-(6)), so
a multi-GPU run gives each rank a contiguous member range and there is NO data-path
collective; only the per-member diagnostic records are gathered at the end.
"""
from __future__ import annotations

import numpy as np


def member_range(rank: int, world: int, n_members: int):
    """Contiguous [lo, hi) of rank's members; the first n_members % world ranks get one more."""
    if not (0 <= rank < world) or n_members < 0:
        raise ValueError("bad rank/world/n_members")
    q, r = divmod(n_members, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def gather_diagnostics(local: np.ndarray, group=None) -> np.ndarray | None:
    """Concatenate the per-rank structured diagnostic arrays on rank 0 (None elsewhere).
    Works on any torch.distributed backend (object gather: the records are tiny)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return local
    world = dist.get_world_size(group)
    out = [None] * world if dist.get_rank(group) == 0 else None
    dist.gather_object(local, out, dst=0, group=group)
    if out is None:
        return None
    return np.concatenate(out)
