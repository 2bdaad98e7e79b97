"""Oracle: stochastic (SDE) sampler step with per-step log-probability (TEST INFRASTRUCTURE, fp64).

  * PAPER.md:227 "The algorithm backbone is FlowGRPO"; PAPER.md:477-482 (Table 2) lists an "SDE window" of denoising
    steps ([0,15] / [0,5]) in which noise is injected during rollout and training.
  * PAPER.md:145 step 5: the seeds selected by exploration are then rolled out at full quality for training - that
    rollout is the consumer of this step; GRPO needs log pi(x_{i+1} | x_i) of every stochastic step.

The paper prints no formula.  The step below is the marginal-preserving reverse-time SDE of a rectified flow
x_t = (1 - t) x_0 + t eps (velocity v = eps - x_0, time running from 1 to 0), derived in DESIGN.md section 11 (readings
D1-D4): with score  grad log p_t(x) = -(x + (1 - t) v) / t  the SDE

      dx = [ v + sigma_t^2 / (2 t) * (x + (1 - t) v) ] dt + sigma_t dW          (dt < 0)

has the same marginals as the ODE dx = v dt for every sigma_t; FlowGRPO's noise schedule is sigma_t = a sqrt(t / (1 - t))
with noise level a.  One Euler-Maruyama step from t_i to t_{i+1} (dt = t_{i+1} - t_i < 0):

      mean    = x (1 + sigma^2/(2 t_i) dt) + v (1 + sigma^2 (1 - t_i)/(2 t_i)) dt
      x_next  = mean + sigma sqrt(-dt) xi ,   xi ~ N(0, I)
      log p   = mean_e[ -(x_next - mean)^2 / (2 sigma^2 (-dt)) ] - log(sigma sqrt(-dt)) - log(2 pi)/2

sigma is singular at t = 1: there FlowGRPO replaces the t in the DENOMINATOR by t_{i+1}, sigma = a sqrt(t_i / (1 - t_{i+1}))
(reading D2).  xi of step i comes
from Philox stream SDE_STREAM_BASE + i of the sequence's seed (reading D3; C2 of SURVEY.md reserves a stream for it).
Steps outside the window, and steps with sigma = 0, are plain Euler steps with log p = 0 (reading D4).
"""
from __future__ import annotations

import math
from typing import Callable, List, Sequence, Tuple

import numpy as np

from . import philox

Array = np.ndarray
SDE_STREAM_BASE = 256


def sde_sigma(t_i: float, t_next: float, noise_level: float) -> float:
    """sigma = a sqrt(t_i / (1 - t')), t' = t_i, or t_next when t_i == 1 (reading D2: only the denominator moves)."""
    td = t_i if t_i < 1.0 else t_next
    return noise_level * math.sqrt(t_i / (1.0 - td))


def sde_step(x: Array, v: Array, t_i: float, t_next: float, noise_level: float, xi: Array) -> Tuple[Array, float]:
    """One stochastic step; returns (x_next, log p(x_next | x)) with the log-density averaged over elements."""
    dt = t_next - t_i
    sig = sde_sigma(t_i, t_next, noise_level)
    if sig == 0.0:
        return x + dt * v, 0.0
    mean = x * (1.0 + sig * sig / (2.0 * t_i) * dt) + v * (1.0 + sig * sig * (1.0 - t_i) / (2.0 * t_i)) * dt
    std = sig * math.sqrt(-dt)
    x_next = mean + std * xi
    logp = float(np.mean(-((x_next - mean) ** 2) / (2.0 * std * std))) - math.log(std) - 0.5 * math.log(2.0 * math.pi)
    return x_next, logp


def step_noise(seed: int, step: int, shape: Sequence[int]) -> Array:
    """xi of Euler step `step` for one sequence: Philox stream SDE_STREAM_BASE + step of its seed (reading D3)."""
    n = int(np.prod(shape))
    return philox.noise_from_seeds([seed], n, SDE_STREAM_BASE + step)[0].reshape(shape)


def denoise_sde(x0: Array, seed: int, timesteps: Sequence[float], velocity: Callable[[Array, float], Array],
                noise_level: float, window: Tuple[int, int], noise_cast=None,
                history: List[Array] | None = None, first_step: int = 0) -> Tuple[Array, Array]:
    """T steps over `timesteps` (length T + 1); steps with window[0] <= j < window[1] are stochastic, j = first_step + i
    the global step index (a resumed rollout passes the number of steps already taken; noise stream = base + j).
    Returns (x_T, logp [T]).  `noise_cast` models the storage precision of xi (the CUDA path makes it in fp32)."""
    T = len(timesteps) - 1
    x = np.array(x0, dtype=np.float64, copy=True)
    logp = np.zeros(T)
    for i in range(T):
        t_i, t_n = float(timesteps[i]), float(timesteps[i + 1])
        v = velocity(x, t_i)
        j = first_step + i
        if window[0] <= j < window[1]:
            xi = step_noise(seed, j, x.shape)
            if noise_cast is not None:
                xi = noise_cast(xi)
            x, logp[i] = sde_step(x, v, t_i, t_n, noise_level, xi)
        else:
            x = x + (t_n - t_i) * v
        if history is not None:
            history.append(x.copy())
    return x, logp
