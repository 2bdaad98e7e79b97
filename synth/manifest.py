"""Shapes of BASELINE.json's five configs and the manifest of synthetic tensors.

Input data only (see synth/__init__.py).  Shapes trace to the paper's workload:
Qwen-Image 20B, 512x512 and 1280x1280, 16 samples per
prompt up to 32 sequences, 10 denoising steps for Geneval
(PAPER.md:251), fewer effective steps during exploration.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Dict, Iterable, List, Optional

import torch

from .generators import hash_normal

STREAMS = ("img", "txt")
BLOCK_TENSORS = ("mod_w", "mod_b", "qkv_w", "qkv_b", "out_w", "out_b", "fc1_w", "fc1_b", "fc2_w", "fc2_b")
GLOBAL_IDS = {"time_w1": 1, "time_b1": 2, "time_w2": 3, "time_b2": 4, "img_in_w": 5, "img_in_b": 6,
              "txt_in_w": 7, "txt_in_b": 8, "final_mod_w": 9, "final_mod_b": 10, "proj_w": 11, "proj_b": 12,
              "probe": 13, "blk_h_txt": 14, "blk_temb": 15, "blk_h_img": 16}
TEXT_EMB_ID0 = 32
BLOCK_ID0 = 1024


@dataclass(frozen=True)
class SpotShape:
    name: str
    dtype: torch.dtype
    n_blocks: int
    hidden: int
    n_heads: int
    head_dim: int
    mlp_hidden: int
    grid_h: int
    grid_w: int
    n_txt: int
    n_prompts: int
    seeds_per_prompt: int
    n_steps: int
    latent_ch: int = 64
    rope_theta: float = 10000.0
    ln_eps: float = 1e-6
    rms_eps: float = 1e-6
    seeds: tuple = ()
    weight_family: int = 0     # configs 2-5 share one weight manifest; config 1 has its own

    @property
    def n_img(self) -> int:
        return self.grid_h * self.grid_w

    @property
    def seq(self) -> int:
        return self.n_txt + self.n_img

    @property
    def txt_dim(self) -> int:
        return self.hidden

    @property
    def n_seqs(self) -> int:
        return self.n_prompts * self.seeds_per_prompt

    @property
    def rope_pairs(self) -> tuple:
        half = self.head_dim // 2
        t = half // 8
        h = (half - t) // 2
        return (t, h, half - t - h)        # (8,28,28) for d_h=128; (4,14,14) for d_h=64

    @property
    def timesteps(self) -> List[float]:
        T = self.n_steps
        return [1.0 - i / T for i in range(T + 1)]   # linspace(1, 0, T+1)

    def flops_per_rollout(self) -> float:
        """Algorithmic FLOPs (2 per multiply-add), DESIGN.md 'Algorithmic work'."""
        S, D, F = self.seq, self.hidden, self.mlp_hidden
        per_seq_block = 2 * S * D * (3 * D + D + 2 * F) + 4 * S * S * D
        io = 2 * 2 * self.n_img * self.latent_ch * D
        per_step = self.n_seqs * (self.n_blocks * per_seq_block + io)
        return float(per_step * self.n_steps)

    def with_(self, **kw) -> "SpotShape":
        return replace(self, **kw)


def _cfg(name, dtype, L, D, H, dh, F, g, ntxt, P, K, T, seeds, fam):
    return SpotShape(name=name, dtype=dtype, n_blocks=L, hidden=D, n_heads=H, head_dim=dh, mlp_hidden=F,
                     grid_h=g, grid_w=g, n_txt=ntxt, n_prompts=P, seeds_per_prompt=K, n_steps=T,
                     seeds=tuple(seeds), weight_family=fam)


CONFIGS: Dict[int, SpotShape] = {
    1: _cfg("cfg1_tiny_fp32", torch.float32, 2, 256, 4, 64, 1024, 8, 32, 1, 4, 4, range(4), 1),
    2: _cfg("cfg2_block_bf16", torch.bfloat16, 1, 3072, 24, 128, 12288, 32, 256, 1, 8, 1, range(8), 0),
    3: _cfg("cfg3_512_bf16", torch.bfloat16, 60, 3072, 24, 128, 12288, 32, 256, 1, 16, 10, range(16), 0),
    4: _cfg("cfg4_1280_bf16", torch.bfloat16, 60, 3072, 24, 128, 12288, 80, 256, 1, 4, 8, range(4), 0),
    5: _cfg("cfg5_sweep_bf16", torch.bfloat16, 60, 3072, 24, 128, 12288, 32, 256, 8, 32, 6, range(256), 0),
}


def _tid(shape: SpotShape, local: int) -> int:
    return shape.weight_family * (1 << 20) + local


def block_tensor_shapes(s: SpotShape) -> Dict[str, tuple]:
    D, F = s.hidden, s.mlp_hidden
    return {"mod_w": (6 * D, D), "mod_b": (6 * D,), "qkv_w": (3 * D, D), "qkv_b": (3 * D,),
            "out_w": (D, D), "out_b": (D,), "fc1_w": (F, D), "fc1_b": (F,), "fc2_w": (D, F), "fc2_b": (D,)}


def global_tensor_shapes(s: SpotShape) -> Dict[str, tuple]:
    D, C = s.hidden, s.latent_ch
    return {"time_w1": (D, 256), "time_b1": (D,), "time_w2": (D, D), "time_b2": (D,),
            "img_in_w": (D, C), "img_in_b": (D,), "txt_in_w": (D, s.txt_dim), "txt_in_b": (D,),
            "final_mod_w": (2 * D, D), "final_mod_b": (2 * D,), "proj_w": (C, D), "proj_b": (C,)}


def make_block_weights(s: SpotShape, block: int, device="cpu") -> Dict[str, torch.Tensor]:
    """Weights of one joint block: keys '<stream>.<tensor>' plus unit gains."""
    out: Dict[str, torch.Tensor] = {}
    shapes = block_tensor_shapes(s)
    for si, stream in enumerate(STREAMS):
        for j, name in enumerate(BLOCK_TENSORS):
            shp = shapes[name]
            n = 1
            for d in shp:
                n *= d
            tid = _tid(s, BLOCK_ID0 + (block * 2 + si) * 16 + j)
            out[f"{stream}.{name}"] = hash_normal(tid, n, 0.02, s.dtype, device).reshape(shp)
        out[f"{stream}.q_gain"] = torch.ones(s.head_dim, dtype=s.dtype, device=device)
        out[f"{stream}.k_gain"] = torch.ones(s.head_dim, dtype=s.dtype, device=device)
    return out


def make_global_weights(s: SpotShape, device="cpu") -> Dict[str, torch.Tensor]:
    out: Dict[str, torch.Tensor] = {}
    for name, shp in global_tensor_shapes(s).items():
        n = 1
        for d in shp:
            n *= d
        out[name] = hash_normal(_tid(s, GLOBAL_IDS[name]), n, 0.02, s.dtype, device).reshape(shp)
    out["txt_gain"] = torch.ones(s.txt_dim, dtype=s.dtype, device=device)
    return out


def make_weights(s: SpotShape, device="cpu", blocks: Optional[Iterable[int]] = None) -> Dict[str, object]:
    """{'global': {...}, 'blocks': [ {...}, ... ]} for blocks 0..n_blocks-1 (or the given subset)."""
    blocks = range(s.n_blocks) if blocks is None else blocks
    return {"global": make_global_weights(s, device), "blocks": [make_block_weights(s, b, device) for b in blocks]}


def make_text_emb(s: SpotShape, device="cpu", prompts: Optional[Iterable[int]] = None) -> torch.Tensor:
    """[P, n_txt, txt_dim] ~ N(0,1) in the config dtype; prompt g has its own tensor id."""
    prompts = list(range(s.n_prompts) if prompts is None else prompts)
    rows = [hash_normal(_tid(s, TEXT_EMB_ID0 + g), s.n_txt * s.txt_dim, 1.0, s.dtype, device)
            .reshape(s.n_txt, s.txt_dim) for g in prompts]
    return torch.stack(rows, 0)


def make_probe(s: SpotShape, device="cpu") -> torch.Tensor:
    """[n_img * C] ~ N(0,1), fp32: the fixed linear reward probe (stand-in for the reward model)."""
    return hash_normal(_tid(s, GLOBAL_IDS["probe"]), s.n_img * s.latent_ch, 1.0, torch.float32, device)


def make_block_inputs(s: SpotShape, n_seqs: int, device="cpu"):
    """Inputs of the single-block config: h_img [B,n_img,D], h_txt [B,n_txt,D] (config dtype), temb [D] fp32."""
    D = s.hidden
    h_img = hash_normal(_tid(s, GLOBAL_IDS["blk_h_img"]), n_seqs * s.n_img * D, 1.0, s.dtype, device)
    h_txt = hash_normal(_tid(s, GLOBAL_IDS["blk_h_txt"]), n_seqs * s.n_txt * D, 1.0, s.dtype, device)
    temb = hash_normal(_tid(s, GLOBAL_IDS["blk_temb"]), D, 1.0, torch.float32, device)
    return h_img.reshape(n_seqs, s.n_img, D), h_txt.reshape(n_seqs, s.n_txt, D), temb
