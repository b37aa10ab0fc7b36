"""Multi-GPU plumbing of the env step.  Economies are independent and every
random draw is keyed by the GLOBAL env id, so the path shards with no data-path collective:
rank r owns global envs [r * E_per_rank, (r + 1) * E_per_rank).  The only exchange is the timing
reduction of bench.py (max over ranks)."""
from __future__ import annotations


def shard_env_base(rank: int, world: int, envs_per_rank: int) -> int:
    """Global id of this rank's local env 0 (``ej_params.env_id_base``)."""
    if not (0 <= rank < world) or envs_per_rank < 1:
        raise ValueError("bad shard (rank %d of %d, %d envs)" % (rank, world, envs_per_rank))
    return rank * envs_per_rank


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """Max of a per-rank scalar (kernel time) over the process group; identity without a group."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def total_units(local_units: int, world: int) -> int:
    """Weak scaling: every rank advances the same number of agent-steps."""
    return int(local_units) * int(world)
