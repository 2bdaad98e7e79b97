"""Multi-GPU plumbing of the exploration rollout (host logic only; no arithmetic of the path).

Every sequence (prompt g, seed k) is independent from the noise to the reward (PAPER.md:29 rollout is
"embarrassingly parallel"; :81 near-linear scaling with added GPUs), so sequences are sharded across ranks with
weights replicated and NO data-path collective.  The only exchange is an all-gather of the per-sequence fp32
rewards, after which the selection (top/bottom-k, sigma_g) runs redundantly on every rank.  Works with any
torch.distributed backend (NCCL over NVLink on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import List, Optional, Tuple

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous partition: unit b goes to rank floor(b * world / n_units), so a prompt group stays on as few
    GPUs as possible.  Returns [lo, hi) of this rank (possibly empty)."""
    assert 0 <= rank < world and n_units >= 0
    lo = -(-rank * n_units // world)
    hi = -(-(rank + 1) * n_units // world)
    return lo, hi


def shard_sizes(n_units: int, world: int) -> List[int]:
    return [shard_range(n_units, r, world)[1] - shard_range(n_units, r, world)[0] for r in range(world)]


def gather_rewards(local: torch.Tensor, n_units: int, group: Optional[dist.ProcessGroup] = None) -> torch.Tensor:
    """All-gather the ragged per-rank reward shards into the full [n_units] vector (same on every rank)."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        assert local.numel() == n_units
        return local
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    sizes = shard_sizes(n_units, world)
    assert local.numel() == sizes[rank], (local.numel(), sizes, rank)
    width = max(sizes)
    padded = torch.zeros(width, dtype=local.dtype, device=local.device)
    padded[:local.numel()] = local
    out = torch.empty(world * width, dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(out, padded, group=group)
    return torch.cat([out[r * width:r * width + sizes[r]] for r in range(world)])


def max_over_ranks(value: float, device: str | torch.device = "cpu", group: Optional[dist.ProcessGroup] = None) -> float:
    """Timing reduction of bench.py: a multi-GPU step takes as long as its slowest rank."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
