"""Multi-GPU host logic.  The path is built for ONE GPU (BASELINE.json north_star: "Everything
runs on one GPU").  Focal points are independent of one another (each trace of N_i depends on a single focal
point), so with N GPUs the job shards over focal points with R^ replicated and NO data-path
collective; when a workload has a single focal point (config 1) the ranks are independent replicas, each with its
own focal point.  torch.distributed is used only for the barrier and the max-over-ranks timing."""
from __future__ import annotations

from dataclasses import replace

from .configs import Config


def focal_slice(nfoc_total: int, rank: int, world: int) -> range:
    """Contiguous, balanced slice of focal-point indices owned by `rank` (sizes differ by at most 1)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(nfoc_total, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def replica_config(cfg: Config, rank: int, world: int) -> Config:
    """Weak scaling: every rank keeps the whole per-GPU workload of `cfg` (same R, same nfoc).  Ranks > 0 move
    their focal depth by 25 m per rank so that they do not all compute the same numbers."""
    if world == 1 or rank == 0:
        return cfg
    rule = cfg.focal.split(":")
    if rule[0] in ("single", "line", "line256", "fan"):
        rule[-1] = str(float(rule[-1]) + 25.0 * rank)
        return replace(cfg, focal=":".join(rule))
    return cfg


def max_over_ranks(value: float, dist=None) -> float:
    """max of a host float over all ranks (identity when torch.distributed is not initialised)."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None) -> float:
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
