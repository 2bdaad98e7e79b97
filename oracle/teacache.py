"""Oracle: cached-step exploration, the paper's "effective denoising steps" axis s (TEST INFRASTRUCTURE, fp64).

  * PAPER.md:155 (s4.3.1) "We therefore control effective denoising steps via a caching strategy rather than
    truncation."
  * PAPER.md:157 "we use Teacache [...] that caches and reuses intermediate transformer outputs across adjacent
    denoising steps when their residual difference falls below a threshold.  Each Teacache threshold corresponds to
    an average number of effective denoising steps s"
  * PAPER.md:340 (s6.8) "we sweep the number of denoising steps by setting different Teacache thresholds"

The paper names the technique and gives no formula; the steps below restate the published TeaCache rule in the
notation of this repository (readings T1-T5 of DESIGN.md section 10), one sequence at a time, in the order the
rule is stated:

  for step i = 0 .. T-1 of one sequence (one request = one prompt x one seed):
    h0  = img_in(x_i)                                              (C7)
    m_i = LN(h0) * (1 + scale1) + shift1      block 0, image stream, modulation of t_i   (C5 steps 1-2)
    i == 0 or i == T-1:  compute, acc <- 0                         (first and last step are always computed)
    else: rel = mean|m_i - m_{i-1}| / mean|m_{i-1}| ;  acc <- acc + poly(rel)
          acc <  threshold: SKIP     hL = h0 + R        (R = residual of the last computed step)
          acc >= threshold: compute, acc <- 0
    compute:  hL = blocks(h0, h_txt0, t_i) ;  R <- hL - h0
    m_{i-1} <- m_i (every step, skipped or not)
    v = final(hL, t_i) ;  x_{i+1} = x_i + (t_{i+1} - t_i) v        (C7, C8)

poly is the rescaling polynomial of the rule, poly(r) = sum_j c_j r^j; its fitted coefficients belong to the
released model and are not available, so the default is the identity (c = [0, 1]) (reading T3).
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import numpy as np

from . import mmdit, philox, rollout

Array = np.ndarray


def rel_l1(cur: Array, prev: Array) -> float:
    """mean|cur - prev| / mean|prev| over the whole [N_img, D] tensor (the rule's distance)."""
    return float(np.abs(cur - prev).mean() / np.abs(prev).mean())


def poly_eval(coeffs: Sequence[float], r: float) -> float:
    """sum_j coeffs[j] * r**j (ascending powers)."""
    acc = 0.0
    for j, c in enumerate(coeffs):
        acc += float(c) * r ** j
    return acc


def modulated_input(x: Array, t: float, g: Dict[str, Array], block0: Dict[str, Array], ln_eps: float = 1e-6,
                    mode: str = "blas") -> Tuple[Array, Array]:
    """(h0, m): h0 = img_in(x) (C7) and m = LN(h0)(1 + scale1) + shift1 with block 0's image modulation at t."""
    _, c = mmdit.time_conditioning(t, g, mode)
    h0 = mmdit.linear(x, g["img_in_w"], g["img_in_b"], mode)
    mod = mmdit.modulation(c, block0["img.mod_w"], block0["img.mod_b"], mode)
    shift1, scale1 = mod[0], mod[1]
    return h0, mmdit.layer_norm(h0, ln_eps) * (1.0 + scale1) + shift1


def denoise_cached(x0: Array, timesteps: Sequence[float], h_txt0: Array, g: Dict[str, Array], blocks: List[Dict[str, Array]],
                   threshold: float, coeffs: Sequence[float] = (0.0, 1.0), *, n_heads: int, cos: Array, sin: Array,
                   ln_eps: float = 1e-6, rms_eps: float = 1e-6, mode: str = "blas",
                   trace: Dict[str, list] | None = None) -> Tuple[Array, List[bool]]:
    """T Euler steps of one sequence with the caching rule above.  Returns (x_T, computed[i] for every step).
    `trace`, if given, receives the per-step lists "rel", "acc" (after the update, before the reset), "computed"."""
    T = len(timesteps) - 1
    x = np.array(x0, dtype=np.float64, copy=True)
    acc = 0.0
    m_prev = None
    resid = None
    computed: List[bool] = []
    for i in range(T):
        t = float(timesteps[i])
        h0, m = modulated_input(x, t, g, blocks[0], ln_eps, mode)
        rel = None
        if i == 0 or i == T - 1:
            compute = True
            acc_seen = 0.0
            acc = 0.0
            if m_prev is not None:
                rel = rel_l1(m, m_prev)
        else:
            rel = rel_l1(m, m_prev)
            acc += poly_eval(coeffs, rel)
            acc_seen = acc
            compute = not (acc < threshold)
            if compute:
                acc = 0.0
        m_prev = m
        _, c = mmdit.time_conditioning(t, g, mode)
        if compute:
            h_img, h_txt = h0, h_txt0
            for bw in blocks:
                h_img, h_txt = mmdit.block_forward(h_img, h_txt, c, bw, n_heads=n_heads, cos=cos, sin=sin, ln_eps=ln_eps,
                                                   rms_eps=rms_eps, mode=mode)
            resid = h_img - h0
            hL = h_img
        else:
            hL = h0 + resid
        m_f = mmdit.linear(c[None, :], g["final_mod_w"], g["final_mod_b"], mode)[0]
        D = hL.shape[1]
        y = mmdit.layer_norm(hL, ln_eps) * (1.0 + m_f[:D]) + m_f[D:]
        v = mmdit.linear(y, g["proj_w"], g["proj_b"], mode)
        x = x + (float(timesteps[i + 1]) - t) * v
        computed.append(bool(compute))
        if trace is not None:
            trace.setdefault("rel", []).append(rel)
            trace.setdefault("acc", []).append(acc_seen)
            trace.setdefault("computed", []).append(bool(compute))
    return x, computed


def explore_cached(seeds: Sequence[int], text_emb: Array, timesteps: Sequence[float], g: Dict[str, Array],
                   blocks: List[Dict[str, Array]], probe: Array, threshold: float, coeffs: Sequence[float] = (0.0, 1.0), *,
                   n_heads: int, grid_h: int, grid_w: int, rope_pairs: Sequence[int], rope_theta: float = 10000.0,
                   ln_eps: float = 1e-6, rms_eps: float = 1e-6, latent_ch: int = 64, mode: str = "blas", x0_cast=None,
                   traces: List[Dict[str, list]] | None = None) -> Tuple[Array, Array, Array]:
    """One prompt x len(seeds) seeds with cached steps.  Returns (final latents [K, N_img, C], rewards [K],
    computed [K, T] bool); the effective number of denoising steps of seed k is computed[k].sum()."""
    n_txt = text_emb.shape[0]
    n_img = grid_h * grid_w
    cos, sin = mmdit.rope_table(grid_h, grid_w, n_txt, rope_pairs, rope_theta)
    h_txt0 = mmdit.text_input(text_emb, g, rms_eps, mode)
    finals, rewards, flags = [], [], []
    for s in seeds:
        x0 = philox.noise_from_seeds([s], n_img * latent_ch, 0)[0].reshape(n_img, latent_ch)
        if x0_cast is not None:
            x0 = x0_cast(x0)
        tr = {} if traces is not None else None
        xT, comp = denoise_cached(x0, timesteps, h_txt0, g, blocks, threshold, coeffs, n_heads=n_heads, cos=cos, sin=sin,
                                  ln_eps=ln_eps, rms_eps=rms_eps, mode=mode, trace=tr)
        if traces is not None:
            traces.append(tr)
        finals.append(xT)
        rewards.append(rollout.probe_reward(xT, probe))
        flags.append(comp)
    return np.stack(finals, 0), np.asarray(rewards), np.asarray(flags, dtype=bool)
