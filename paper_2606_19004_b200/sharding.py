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


def shard_prompt_index(lo: int, hi: int, seeds_per_prompt: int) -> List[int]:
    """Prompt of every sequence of the shard [lo, hi): sequence b belongs to prompt b // K (a shard may start and end
    inside a prompt group)."""
    return [b // seeds_per_prompt for b in range(lo, hi)]


def explore_shard(ctx, seeds: torch.Tensor, text_emb: torch.Tensor, timesteps, probe: torch.Tensor, n_prompts: int,
                  seeds_per_prompt: int, rank: int, world: int) -> dict:
    """This rank's slice of one exploration call (sequence b -> rank floor(b * world / B)): noise,
    T Euler steps and rewards of sequences [lo, hi) through the C ABI.  The slice runs as hi - lo one-seed prompt groups
    with the text rows gathered per sequence (a row copy; h_txt0 is then projected per sequence, 2 * N_txt * D^2 FLOP
    each), so it may cut through a prompt group; a sequence's result does not depend on its batch (spot.h "Determinism"),
    hence the shards together are bit-identical to the unsharded call.  Returns {"lo", "hi", "latents", "rewards"}."""
    from . import binding
    B = n_prompts * seeds_per_prompt
    assert seeds.numel() == B and text_emb.shape[0] == n_prompts
    lo, hi = shard_range(B, rank, world)
    s = ctx.shape
    if hi == lo:
        return {"lo": lo, "hi": hi, "latents": torch.empty((0, s.n_img, s.latent_ch), dtype=torch.float32, device=seeds.device),
                "rewards": torch.empty(0, dtype=torch.float32, device=seeds.device)}
    idx = torch.tensor(shard_prompt_index(lo, hi, seeds_per_prompt), dtype=torch.long, device=text_emb.device)
    local_text = text_emb.index_select(0, idx).contiguous()
    out = binding.spot_explore(ctx, seeds[lo:hi].contiguous(), local_text, timesteps, probe, hi - lo, 1, 0)
    return {"lo": lo, "hi": hi, "latents": out["latents"], "rewards": out["rewards"]}


def explore_sharded(ctx, seeds: torch.Tensor, text_emb: torch.Tensor, timesteps, probe: torch.Tensor, n_prompts: int,
                    seeds_per_prompt: int, k_select: int, group: Optional[dist.ProcessGroup] = None) -> dict:
    """One exploration call spread over the ranks of `group` (strong scaling of a fixed P x K batch): every rank holds
    the full seeds / text / probe and the replicated weights, computes its shard (explore_shard), the fp32 rewards are
    all-gathered (the path's only exchange: 4 B per sequence) and the selection runs redundantly on every rank.
    Returns rewards [P * K], stats, top, bottom (identical on all ranks) and this rank's latents with their range."""
    from . import binding
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    shard = explore_shard(ctx, seeds, text_emb, timesteps, probe, n_prompts, seeds_per_prompt, rank, world)
    rewards = gather_rewards(shard["rewards"], n_prompts * seeds_per_prompt, group)
    stats, top, bottom = binding.spot_select_seeds(rewards, n_prompts, seeds_per_prompt, k_select)
    return {"rewards": rewards, "stats": stats, "top": top, "bottom": bottom, "local_latents": shard["latents"],
            "local_range": (shard["lo"], shard["hi"])}
