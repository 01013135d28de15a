"""Column sharding for multi-GPU runs.

Columns of the filter are independent (each output column depends only on H, its own input
column and its own degree), so N GPUs shard the COLUMNS and replicate H: no data-path
collective.  Columns arrive sorted by ascending degree (Alg. 1 l.15); dealing
them round-robin keeps every shard sorted and balances sum(deg) -- and therefore flops
(8 N^2 sum(deg)) -- to within one column per distinct degree.
"""
from __future__ import annotations

import numpy as np


def shard_columns(ncols: int, world: int, rank: int) -> np.ndarray:
    """Indices (ascending) of the columns owned by `rank`: rank, rank + world, ..."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("need 0 <= rank < world")
    return np.arange(rank, ncols, world, dtype=np.int64)


def unshard_columns(ncols: int, world: int) -> np.ndarray:
    """perm such that concat(shard_0, ..., shard_{world-1})[:, perm] is in the original order."""
    order = np.concatenate([shard_columns(ncols, world, r) for r in range(world)])
    perm = np.empty(ncols, dtype=np.int64)
    perm[order] = np.arange(ncols)
    return perm


def shard_balance(degrees, world: int):
    """sum(deg) per rank -- what each GPU's flop count is proportional to."""
    deg = np.asarray(degrees)
    return [int(deg[shard_columns(len(deg), world, r)].sum()) for r in range(world)]
