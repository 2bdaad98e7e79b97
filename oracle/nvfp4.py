"""Oracle: NVFP4 (block-scaled 4-bit) variant of the MLP Linears of the exploration rollout (TEST INFRASTRUCTURE).

  * PAPER.md:67 (s2.2) "first running a cheap exploratory rollout e.g., with reduced denoising steps or a quantized
    model, to identify high-contrast seeds, then performing full-quality rollout only on the selected seeds";
    PAPER.md:340 judges a cheaper exploration by the rank correlation of its rewards with the full rollout's (>= 0.8).
The paper does not build this variant; readings N1-N5 of DESIGN.md section 13b define it (it extends the FP8 variant of
oracle/fp8.py: QKV and out-proj stay FP8, the two MLP Linears - 2/3 of the block's Linear FLOPs - go to 4 bits):

  N1  fc1 and fc2 of every block and stream run on NVFP4 operands, weights AND activations (the tensor-core instruction
      takes both operands in the same format); everything else is the FP8 variant.
  N2  NVFP4 = E2M1 values {0, 0.5, 1, 1.5, 2, 3, 4, 6} with sign, in blocks of 16 consecutive elements along K, each block
      with an E4M3 scale factor (oracle/fp8.e4m3: bias 7, max 448, subnormals to 2^-9, round to nearest even).
  N3  activations (unit global scale):  sf_b = e4m3(max_{k in b} |x_k| / 6),  q_k = e2m1(x_k / sf_b)  (q = 0 where
      sf_b = 0); conversion to E2M1 rounds to nearest, ties to the even code, and saturates at +-6.
  N4  weights: per OUTPUT channel n a second-level fp32 scale  s_n = max_k |W_nk| / (6 * 448)  (1 for a zero row), then
      N3 applied to W_n / s_n.
  N5  y_n = s_n * sum_b sfx_b sfw_nb sum_{k in b} qx_k qw_nk + b_n, accumulated exactly here (fp32 on the GPU).
Every value that DECIDES a code (block maximum / 6, quotient x / sf, W / s_n) is formed in fp32 with IEEE division, on
this side and in the CUDA quantisers alike: a 4-bit code is an integer decided by floating point, and both sides must
take that decision in the same precision (the kernel's).
"""
from __future__ import annotations

from typing import Dict, List, Tuple

import numpy as np

from . import fp8, mmdit

Array = np.ndarray
BLOCK = 16
E2M1_MAX = 6.0
f32 = np.float32


def e2m1(x: Array) -> Array:
    """Nearest E2M1 value (1 sign, 2 exponent bits of bias 1, 1 mantissa bit: 0, 0.5, 1, 1.5, 2, 3, 4, 6), ties to the even
    code, saturating at +-6.  Returned as fp64."""
    x = np.asarray(x, dtype=np.float64)
    a = np.minimum(np.abs(x), E2M1_MAX)
    with np.errstate(divide="ignore"):
        e = np.floor(np.log2(np.where(a > 0, a, 1.0)))
    e = np.clip(e, 0.0, 2.0)                     # binades [1,2), [2,4), [4,8); below 1 the grid is the subnormal one (0, 0.5)
    q = np.exp2(e - 1.0)                         # spacing of the 1-bit mantissa grid: 0.5, 1, 2
    r = np.rint(a / q) * q                       # np.rint rounds half to even = the even mantissa code
    return np.sign(x) * np.minimum(r, E2M1_MAX)


def quantize_rows(x: Array) -> Tuple[Array, Array]:
    """(q, sf): x [n, K] (K a multiple of 16) -> E2M1 values q [n, K] and E4M3 block scales sf [n, K/16] (reading N3)."""
    x32 = np.asarray(x, dtype=f32)
    n, K = x32.shape
    assert K % BLOCK == 0
    blocks = x32.reshape(n, K // BLOCK, BLOCK)
    amax = np.abs(blocks).max(axis=2)
    sf = fp8.e4m3((amax / f32(E2M1_MAX)).astype(np.float64)).astype(f32)        # fp32 quotient, then the E4M3 rounding
    with np.errstate(divide="ignore", invalid="ignore"):
        quot = np.where(sf[:, :, None] > 0, blocks / sf[:, :, None], f32(0))    # fp32 IEEE division
    return e2m1(quot.astype(np.float64)).reshape(n, K), sf.astype(np.float64)


def dequantize(q: Array, sf: Array) -> Array:
    return (q.reshape(q.shape[0], -1, BLOCK) * sf[:, :, None]).reshape(q.shape)


def quantize_weight(w: Array) -> Tuple[Array, Array, Array]:
    """(q, sf, s): per-output-channel s_n = max|W_n| / (6 * 448), then quantize_rows(W / s) (reading N4)."""
    w32 = np.asarray(w, dtype=f32)
    amax = np.abs(w32).max(axis=1)
    s = np.where(amax > 0, amax / f32(E2M1_MAX * fp8.E4M3_MAX), f32(1)).astype(f32)
    q, sf = quantize_rows(w32 / s[:, None])
    return q, sf, s.astype(np.float64)


def linear_nvfp4(x: Array, wq: Array, wsf: Array, s: Array, b: Array) -> Array:
    """y = s * (deq(x) deq(W)^T) + b (readings N3, N5)."""
    xq, xsf = quantize_rows(x)
    return (dequantize(xq, xsf) @ dequantize(wq, wsf).T) * s + b


def linear_nvfp4_deq(x: Array, w_deq: Array, s: Array, b: Array) -> Array:
    """linear_nvfp4 with dequantize(wq, wsf) formed once by the caller (tests/golden/make_cfg3_golden.py keeps it per block:
    an E2M1 value times an E4M3 scale has a 5-bit significand, so even a bf16 copy holds it exactly).  Same arithmetic, same
    result bit for bit (pinned in tests/test_oracle_nvfp4.py)."""
    xq, xsf = quantize_rows(x)
    return (dequantize(xq, xsf) @ w_deq.T) * s + b


MLP_LINEARS = ("fc1", "fc2")


def quantize_block(bw: Dict[str, Array]) -> Dict[str, tuple]:
    """Quantised weights of one block: fc1 / fc2 in NVFP4 (q, sf, s), qkv / out in FP8 (Wq, s) (reading N1)."""
    out = {}
    for st in ("img", "txt"):
        for ln in fp8.BLOCK_LINEARS:
            w = bw[f"{st}.{ln}_w"]
            out[f"{st}.{ln}"] = quantize_weight(w) if ln in MLP_LINEARS else fp8.quantize_weight(w)
    return out


def block_lin(bw: Dict[str, Array], qw: Dict[str, tuple]):
    """The `lin` hook of mmdit.block_forward for the NVFP4 variant."""
    def lin(x, name):
        if name.split(".")[1] in MLP_LINEARS:
            return linear_nvfp4(x, *qw[name], bw[f"{name}_b"])
        return fp8.linear_fp8(x, qw[name][0], qw[name][1], bw[f"{name}_b"])
    return lin


def block_forward_nvfp4(h_img: Array, h_txt: Array, c: Array, bw: Dict[str, Array], qw=None, **kw):
    qw = quantize_block(bw) if qw is None else qw
    return mmdit.block_forward(h_img, h_txt, c, bw, lin=block_lin(bw, qw), **kw)


def dit_velocity_nvfp4(x: Array, t: float, h_txt0: Array, g: Dict[str, Array], blocks: List[Dict[str, Array]],
                       qblocks: List[Dict[str, tuple]], **kw) -> Array:
    return mmdit.dit_velocity(x, t, h_txt0, g, blocks, block_lin=lambda i: block_lin(blocks[i], qblocks[i]), **kw)
