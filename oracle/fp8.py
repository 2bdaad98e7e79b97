"""Oracle: low-precision (FP8 E4M3) exploration variant of the block Linears (TEST INFRASTRUCTURE, fp64).

  * PAPER.md:67 (s2.2) "Sol-RL proposes first running a cheap exploratory rollout e.g., with reduced denoising steps
    or a quantized model, to identify high-contrast seeds, then performing full-quality rollout only on the selected
    seeds" - the prior art SPOTLIGHT's exploration phase generalises; PAPER.md:340 judges a cheaper exploration by the
    rank correlation of its rewards with the full rollout's (>= 0.8).
The paper does not build this variant; readings Q1-Q4 of DESIGN.md section 13 define it:

  Q1  only the four Linears of a block (QKV, out-proj, fc1, fc2) are quantised; attention, norms, modulation,
      residual stream, input/final layers and the sampler are unchanged.
  Q2  weights: per OUTPUT channel n,  s_n = max_k |W_nk| / 448 (1 if the row is zero),  Wq_nk = e4m3(W_nk / s_n).
  Q3  activations: unit scale, xq = e4m3(x) (saturating at +-448).
  Q4  y_n = s_n * sum_k xq_k Wq_nk + b_n, accumulated exactly (fp32 on the GPU, fp64 here).
  e4m3 = OCP FP8 E4M3 "FN": 1 sign, 4 exponent (bias 7), 3 mantissa bits, no infinities, max 448, subnormals down to
  2^-9; conversion rounds to nearest, ties to even, and saturates to +-448.
"""
from __future__ import annotations

from typing import Dict, List, Tuple

import numpy as np

from . import mmdit

Array = np.ndarray
E4M3_MAX = 448.0


def e4m3(x: Array) -> Array:
    """Nearest E4M3 value (ties to even, saturating), returned as fp64."""
    x = np.asarray(x, dtype=np.float64)
    a = np.minimum(np.abs(x), E4M3_MAX)
    with np.errstate(divide="ignore"):
        e = np.floor(np.log2(np.where(a > 0, a, 1.0)))
    e = np.maximum(e, -6.0)                      # below 2^-6 the grid is the subnormal one, spacing 2^-9
    q = np.exp2(e - 3.0)                         # spacing of the 3-bit mantissa grid in this binade
    r = np.rint(a / q) * q                       # np.rint rounds half to even; a/q is exact (power-of-two divisor)
    return np.sign(x) * np.minimum(r, E4M3_MAX)


def quantize_weight(w: Array) -> Tuple[Array, Array]:
    """(Wq, s): per-output-channel scale s_n = max|W_n| / 448 and Wq = e4m3(W / s) (reading Q2)."""
    amax = np.abs(w).max(axis=1)
    s = np.where(amax > 0, amax / E4M3_MAX, 1.0)
    return e4m3(w / s[:, None]), s


def linear_fp8(x: Array, wq: Array, s: Array, b: Array) -> Array:
    """y = s * (e4m3(x) Wq^T) + b (readings Q3, Q4)."""
    return (e4m3(x) @ wq.T) * s + b


BLOCK_LINEARS = ("qkv", "out", "fc1", "fc2")


def quantize_block(bw: Dict[str, Array]) -> Dict[str, Tuple[Array, Array]]:
    """The quantised weights of one block: name "<stream>.<linear>" -> (Wq, s)."""
    return {f"{st}.{ln}": quantize_weight(bw[f"{st}.{ln}_w"]) for st in ("img", "txt") for ln in BLOCK_LINEARS}


def block_lin(bw: Dict[str, Array], qw: Dict[str, Tuple[Array, Array]]):
    """The `lin` hook of mmdit.block_forward for the FP8 variant."""
    return lambda x, name: linear_fp8(x, qw[name][0], qw[name][1], bw[f"{name}_b"])


def block_forward_fp8(h_img: Array, h_txt: Array, c: Array, bw: Dict[str, Array], qw=None, **kw):
    """mmdit.block_forward with the four Linears replaced by linear_fp8."""
    qw = quantize_block(bw) if qw is None else qw
    return mmdit.block_forward(h_img, h_txt, c, bw, lin=block_lin(bw, qw), **kw)


def dit_velocity_fp8(x: Array, t: float, h_txt0: Array, g: Dict[str, Array], blocks: List[Dict[str, Array]],
                     qblocks: List[Dict[str, Tuple[Array, Array]]], **kw) -> Array:
    """mmdit.dit_velocity with every block in the FP8 variant."""
    return mmdit.dit_velocity(x, t, h_txt0, g, blocks, block_lin=lambda i: block_lin(blocks[i], qblocks[i]), **kw)
