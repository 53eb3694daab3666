"""Replica bookkeeping for N>1 runs ("replicas only").

The decode MoE layer of BASELINE.json runs on ONE GPU: no sharding, no data-path collective.  `bench.py --gpus N`
therefore runs N independent replicas of the same layer-step (weak scaling), and the only thing that crosses
ranks is the timing protocol of the bench contract: a barrier on both sides of the timed region and the MAX of
the per-rank device times.  That host logic lives here so that the world_size-2 `gloo` test can cover it
without a GPU.  There is no arithmetic of the method in this module.
"""
from __future__ import annotations


def max_over_ranks(ms: float, dist=None, device="cpu") -> float:
    """Device time of the slowest rank (all ranks get the same number).  `dist` is torch.distributed when a
    process group is up, else None (single process)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput_gbs(bytes_per_rank: float, world: int, ms: float) -> float:
    """Whole-job GB/s: every replica moves `bytes_per_rank` in the (max-over-ranks) `ms`."""
    return bytes_per_rank * world / (ms * 1e-3) / 1e9


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica draws its own batch (distinct hiddens, same layer weights)."""
    return int(base_seed) + 7919 * int(rank)
