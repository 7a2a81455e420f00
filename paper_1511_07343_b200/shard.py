"""DM-trial sharding across ranks (one process per GPU).

DM trials are independent series "searched individually", so the path shards with no
exchange step: rank r searches the trials {dm : dm mod world == r} and the
candidate lists are concatenated on rank 0.  The only collective is that control-plane gather of the
(small) result lists; nothing on the data path crosses ranks.
"""
from __future__ import annotations

from typing import Dict, List, Sequence

import numpy as np


def dm_shard(n_dm: int, rank: int, world: int) -> List[int]:
    """DM-trial indices searched by `rank`: dm mod world == rank (round robin keeps ranks balanced when
    the per-trial cost drifts with DM)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    return list(range(rank, n_dm, world))


def gather_candidates(local: Dict[int, np.ndarray], n_dm: int, group=None, dst: int = 0):
    """Collect the per-DM candidate arrays of every rank on `dst`; returns {dm: array} there, None elsewhere.
    `local` maps each DM index this rank searched to its structured candidate array."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return dict(local)
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    gathered: Sequence = [None] * world if rank == dst else None
    dist.gather_object({int(k): np.asarray(v) for k, v in local.items()}, gathered, dst=dst, group=group)
    if rank != dst:
        return None
    merged: Dict[int, np.ndarray] = {}
    for r, part in enumerate(gathered):
        for dm, c in part.items():
            if dm in merged or dm % world != r:
                raise RuntimeError("DM trial %d reported by the wrong rank %d" % (dm, r))
            merged[dm] = c
    if sorted(merged) != list(range(n_dm)):
        raise RuntimeError("missing DM trials: %s" % sorted(set(range(n_dm)) - set(merged)))
    return merged
