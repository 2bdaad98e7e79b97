"""Oracle: Euler flow-matching sampler, probe reward, seed selection (TEST INFRASTRUCTURE, fp64).

  * PAPER.md:59  "refines a latent representation over a fixed number of denoising steps"
  * PAPER.md:61  "Each sample is scored by a reward model, yielding a per-sample scalar reward r_k"
  * PAPER.md:175 per-prompt reward standard deviation sigma_g (bandit feedback)
  * PAPER.md:229 "top-k/bottom-k strategy over per-prompt exploration rewards, retaining the
    highest- and lowest-scoring seeds"; "top and bottom K/2 by reward"

Readings S8-S12 of DESIGN.md: deterministic Euler x_{i+1} = x_i + (t_{i+1} - t_i) v_i on a
caller-supplied grid t_0 > ... > t_T, model evaluated at t_0..t_{T-1}; reward = linear probe
<p, x_T>/sqrt(N_img C); population std; ties broken by lower index.
"""
from __future__ import annotations

import math
from typing import Callable, Dict, List, Sequence, Tuple

import numpy as np

from . import mmdit, philox

Array = np.ndarray


def euler_denoise(x0: Array, timesteps: Sequence[float], velocity: Callable[[Array, float], Array],
                  history: List[Array] | None = None) -> Array:
    """T Euler steps of dx/dt = v(x, t) over the grid `timesteps` (length T+1) (C8)."""
    x = np.array(x0, dtype=np.float64, copy=True)
    for i in range(len(timesteps) - 1):
        v = velocity(x, float(timesteps[i]))
        x = x + (float(timesteps[i + 1]) - float(timesteps[i])) * v
        if history is not None:
            history.append(x.copy())
    return x


def probe_reward(x: Array, probe: Array) -> float:
    """r = <p, x> / sqrt(N_img * C) over the flattened final latent (C9)."""
    flat = x.reshape(-1)
    return float(np.dot(probe.reshape(-1), flat) / math.sqrt(flat.size))


def select_seeds(rewards: Array, k_select: int) -> Dict[str, object]:
    """Per prompt group: mean, population std, argmax, argmin, top-k and bottom-k positions (C9).

    rewards [P, K].  top-k: k largest by (reward descending, index ascending); bottom-k: k smallest
    by (reward ascending, index ascending)."""
    r = np.asarray(rewards, dtype=np.float64)
    P, K = r.shape
    assert 0 <= 2 * k_select <= K
    mean = r.mean(axis=1)
    std = np.sqrt(((r - mean[:, None]) ** 2).mean(axis=1))
    top = np.zeros((P, k_select), dtype=np.int32)
    bottom = np.zeros((P, k_select), dtype=np.int32)
    for g in range(P):
        idx = list(range(K))
        top[g] = sorted(idx, key=lambda i: (-r[g, i], i))[:k_select]
        bottom[g] = sorted(idx, key=lambda i: (r[g, i], i))[:k_select]
    return {"mean": mean, "std": std, "top": top, "bottom": bottom,
            "argmax": np.asarray([sorted(range(K), key=lambda i: (-r[g, i], i))[0] for g in range(P)]),
            "argmin": np.asarray([sorted(range(K), key=lambda i: (r[g, i], i))[0] for g in range(P)])}


def explore(seeds: Sequence[int], text_emb: Array, timesteps: Sequence[float], g: Dict[str, Array],
            blocks: List[Dict[str, Array]], probe: Array, *, n_heads: int, grid_h: int, grid_w: int,
            rope_pairs: Sequence[int], rope_theta: float = 10000.0, ln_eps: float = 1e-6, rms_eps: float = 1e-6,
            latent_ch: int = 64, mode: str = "blas", x0_cast=None,
            history: List[List[Array]] | None = None) -> Tuple[Array, Array]:
    """One prompt x len(seeds) seeds: noise -> T Euler steps of the MMDiT -> probe reward.

    Returns (final latents [K, N_img, C], rewards [K]).  `x0_cast` (e.g. a float32 round trip)
    models the storage precision of the initial latent; everything after it is fp64."""
    n_txt = text_emb.shape[0]
    n_img = grid_h * grid_w
    cos, sin = mmdit.rope_table(grid_h, grid_w, n_txt, rope_pairs, rope_theta)
    h_txt0 = mmdit.text_input(text_emb, g, rms_eps, mode)
    finals, rewards = [], []
    for s in seeds:
        x0 = philox.noise_from_seeds([s], n_img * latent_ch, 0)[0].reshape(n_img, latent_ch)
        if x0_cast is not None:
            x0 = x0_cast(x0)
        hist = [] if history is not None else None
        xT = euler_denoise(x0, timesteps,
                           lambda x, t: mmdit.dit_velocity(x, t, h_txt0, g, blocks, n_heads=n_heads, cos=cos, sin=sin,
                                                           ln_eps=ln_eps, rms_eps=rms_eps, mode=mode), hist)
        if history is not None:
            history.append(hist)
        finals.append(xT)
        rewards.append(probe_reward(xT, probe))
    return np.stack(finals, 0), np.asarray(rewards)
