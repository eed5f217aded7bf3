"""Replica sharding over ranks (one process per GPU).

The path shards over replicas with no data-path collective (every replica is an independent anneal,
PAPER.md:78,106); the only exchange is the best-replica reduction Eq.5 across ranks.
Works on any torch.distributed backend (NCCL on GPUs; gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def replica_seed(base_seed: int, rank: int) -> int:
    """Distinct, reproducible field seed per rank (the generator is keyed on (seed, replica, variable, state))."""
    return int(base_seed) * 1000003 + int(rank)


def best_over_ranks(best_energy: float, best_config: np.ndarray, device: torch.device):
    """argmin over ranks of each rank's best energy (lowest rank on ties), then that rank's configuration.

    Returns (energy, owner_rank, config) on every rank.  Traffic: 8 bytes per rank + n int32 from the owner."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    cfg = torch.tensor(np.asarray(best_config, dtype=np.int32), device=device)  # a copy: the broadcast is in place
    if not dist.is_initialized():
        return float(best_energy), 0, cfg.cpu().numpy()
    mine = torch.tensor([best_energy], dtype=torch.float64, device=device)
    allv = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(allv, mine)
    vals = torch.cat(allv).cpu().numpy()
    owner = int(np.argmin(vals))                      # numpy argmin returns the first minimum = lowest rank
    dist.broadcast(cfg, src=owner)
    return float(vals[owner]), owner, cfg.cpu().numpy()
