"""Multi-GPU host logic: replicas only.

The hot path runs on one GPU; with N GPUs every rank analyses its own independent stack and there is
no data-path collective.  The only cross-rank step is the measurement itself: the whole-job rate is
(units processed by all ranks) / (max over ranks of the device time).  These helpers hold that logic so
that it can be covered by world_size-2 gloo tests on CPU.
"""
from dataclasses import replace


def rank_config(cfg, rank: int):
    """Rank r analyses the same kind of stack with a different seed (rank 0 keeps the config's seed)."""
    return cfg if rank == 0 else replace(cfg, seed=cfg.seed + 100 * rank, fringes=[])


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a per-rank scalar (device time in ms); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, ms_per_step_max: float, world: int) -> float:
    """units/s over all ranks: world * units_per_rank / max-over-ranks time."""
    return world * units_per_rank / (ms_per_step_max * 1e-3)
