"""Oracle: the Qwen-Image-shaped MMDiT forward pass in fp64 (TEST INFRASTRUCTURE).

"each [denoising step] requiring a full forward pass through the DiT backbone"
(PAPER.md:59); model = "Qwen-Image 20B".  The paper gives no block
definition; this file is reading S4-S7 of DESIGN.md written out
step by step, one sequence at a time, no blocking, fusion or reordering.

All Linear layers are y = x W^T + b with W [out, in].  Joint sequence order is text tokens
first, then image tokens.  Inputs are fp64 arrays holding the (already dtype-rounded) values
the CUDA path receives.

Matmul back ends: "blas" = numpy @ (OpenBLAS dgemm); "einsum" = numpy's own C loops with
optimize=False (no BLAS).  Tests cross-check the two and brute-force tiny cases in Python.
"""
from __future__ import annotations

import math
from typing import Dict, List, Sequence, Tuple

import numpy as np

Array = np.ndarray

# Optional host threads for the full-size golden runs (tests/golden/make_cfg3_golden.py).  They only change WHO
# evaluates an independent piece (an attention head, a block of rows of an elementwise map, a sequence), never the
# arithmetic or its order inside a piece; tests/test_oracle_mmdit.py pins the threaded results bit for bit to the
# serial ones.  Default 1 = plain serial code, which is also what bench.py times as the CPU baseline.
_WORKERS = 1


def set_workers(n: int) -> None:
    global _WORKERS
    _WORKERS = max(1, int(n))


def _pmap(fn, items, workers=None):
    items = list(items)
    w = _WORKERS if workers is None else workers
    if w <= 1 or len(items) <= 1:
        return [fn(i) for i in items]
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(w) as ex:
        return list(ex.map(fn, items))


def linear(x: Array, w: Array, b: Array | None, mode: str = "blas") -> Array:
    """y = x W^T + b ; x [n, in], W [out, in]."""
    if mode == "blas":
        y = x @ w.T
    elif mode == "einsum":
        y = np.einsum("ni,oi->no", x, w, optimize=False)
    else:
        raise ValueError(mode)
    return y if b is None else y + b


def silu(x: Array) -> Array:
    return x / (1.0 + np.exp(-x))


def gelu_tanh(x: Array) -> Array:
    """GELU_tanh(x) = x/2 (1 + tanh(sqrt(2/pi) (x + 0.044715 x^3)))  (reading S4)."""
    f = lambda x: 0.5 * x * (1.0 + np.tanh(math.sqrt(2.0 / math.pi) * (x + 0.044715 * x ** 3)))
    if _WORKERS > 1 and x.ndim == 2 and x.shape[0] >= 2 * _WORKERS:
        return np.concatenate(_pmap(f, np.array_split(x, _WORKERS, axis=0)), axis=0)      # elementwise: rows are independent
    return f(x)


def layer_norm(x: Array, eps: float) -> Array:
    """LayerNorm over the last axis, biased variance, no affine (C5 step 2)."""
    mu = x.mean(axis=-1, keepdims=True)
    var = ((x - mu) ** 2).mean(axis=-1, keepdims=True)
    return (x - mu) / np.sqrt(var + eps)


def rms_norm(x: Array, gain: Array, eps: float) -> Array:
    """x / sqrt(mean(x^2) + eps) * gain over the last axis (C5 step 4, C7)."""
    ms = (x ** 2).mean(axis=-1, keepdims=True)
    return x / np.sqrt(ms + eps) * gain


def timestep_embedding(t: float) -> Array:
    """Sinusoidal-256 (C4): a = 1000 t, f_i = exp(-ln(10000) i / 128), [cos(a f) ; sin(a f)]."""
    a = 1000.0 * float(t)
    f = np.exp(-math.log(10000.0) * np.arange(128, dtype=np.float64) / 128.0)
    return np.concatenate([np.cos(a * f), np.sin(a * f)])


def time_conditioning(t: float, g: Dict[str, Array], mode: str = "blas") -> Tuple[Array, Array]:
    """temb = W2 SiLU(W1 e(t) + b1) + b2 ; c = SiLU(temb).  Returns (temb, c), each [D]."""
    e = timestep_embedding(t)[None, :]
    hid = silu(linear(e, g["time_w1"], g["time_b1"], mode))
    temb = linear(hid, g["time_w2"], g["time_b2"], mode)[0]
    return temb, silu(temb)


def rope_positions(grid_h: int, grid_w: int, n_txt: int) -> Array:
    """[S, 3] integer positions (t, h, w) of the joint sequence, text first (C6)."""
    pos = np.zeros((n_txt + grid_h * grid_w, 3), dtype=np.float64)
    base = max(grid_h // 2, grid_w // 2)
    for j in range(n_txt):
        pos[j, :] = base + j
    for r in range(grid_h):
        for c in range(grid_w):
            pos[n_txt + r * grid_w + c] = (0, r - (grid_h + 1) // 2, c - (grid_w + 1) // 2)
    return pos


def rope_table(grid_h: int, grid_w: int, n_txt: int, rope_pairs: Sequence[int], theta: float,
               shift: Tuple[int, int] = (0, 0)) -> Tuple[Array, Array]:
    """cos, sin [S, d_h/2]: pair i belongs to axis a(i) (t pairs, then h, then w) with frequency
    theta**(-i'/n_a), i' the index inside the axis; angle = pos_a * freq (C6).  `shift` moves the
    image grid by (dr, dc) - used by the relative-position pin only."""
    pos = rope_positions(grid_h, grid_w, n_txt)
    pos[n_txt:, 1] += shift[0]
    pos[n_txt:, 2] += shift[1]
    cols = []
    for axis, n_a in enumerate(rope_pairs):
        freq = np.asarray([theta ** (-(i / n_a)) for i in range(n_a)], dtype=np.float64)
        cols.append(pos[:, axis:axis + 1] * freq[None, :])
    ang = np.concatenate(cols, axis=1)
    return np.cos(ang), np.sin(ang)


def apply_rope(x: Array, cos: Array, sin: Array) -> Array:
    """x [S, H, d_h]; rotate interleaved pairs (2i, 2i+1) by the angle of (token s, pair i) (C5 step 5)."""
    xe, xo = x[..., 0::2], x[..., 1::2]
    c, s = cos[:, None, :], sin[:, None, :]
    out = np.empty_like(x)
    out[..., 0::2] = xe * c - xo * s
    out[..., 1::2] = xe * s + xo * c
    return out


def attention(q: Array, k: Array, v: Array) -> Array:
    """softmax(Q K^T / sqrt(d_h)) V per head, all S keys, no mask (C5 step 6). q,k,v [S, H, d_h]."""
    S, H, dh = q.shape
    out = np.empty_like(q)

    def head(h):
        logits = (q[:, h, :] @ k[:, h, :].T) / math.sqrt(dh)
        logits = logits - logits.max(axis=1, keepdims=True)
        p = np.exp(logits)
        p = p / p.sum(axis=1, keepdims=True)
        out[:, h, :] = p @ v[:, h, :]

    _pmap(head, range(H))                                   # heads are independent; serial unless set_workers(n > 1)
    return out


def modulation(c: Array, w: Array, b: Array, mode: str = "blas") -> List[Array]:
    """m = W_mod c + b in R^{6D}, split (shift1, scale1, gate1, shift2, scale2, gate2) (C5 step 1)."""
    m = linear(c[None, :], w, b, mode)[0]
    return list(m.reshape(6, -1))


def block_forward(h_img: Array, h_txt: Array, c: Array, bw: Dict[str, Array], *, n_heads: int,
                  cos: Array, sin: Array, ln_eps: float = 1e-6, rms_eps: float = 1e-6,
                  mode: str = "blas", trace: Dict[str, Array] | None = None, lin=None) -> Tuple[Array, Array]:
    """One joint block for one sequence (C5 steps 1-8).  h_img [N_img, D], h_txt [N_txt, D], c = SiLU(temb) [D].
    `lin(x, name)`, if given, replaces y = x W^T + b for the four block Linears name = "<stream>.qkv|out|fc1|fc2"
    (used by oracle/fp8.py to state the low-precision variant; None = the plain Linear above)."""
    if lin is None:
        lin = lambda x, name: linear(x, bw[f"{name}_w"], bw[f"{name}_b"], mode)
    n_txt = h_txt.shape[0]
    D = h_img.shape[1]
    dh = D // n_heads
    h = {"img": h_img, "txt": h_txt}
    mod, q, k, v = {}, {}, {}, {}
    for s in ("txt", "img"):
        mod[s] = modulation(c, bw[f"{s}.mod_w"], bw[f"{s}.mod_b"], mode)
        shift1, scale1 = mod[s][0], mod[s][1]
        y = layer_norm(h[s], ln_eps) * (1.0 + scale1) + shift1
        qkv = lin(y, f"{s}.qkv")
        n = qkv.shape[0]
        q[s] = rms_norm(qkv[:, 0 * D:1 * D].reshape(n, n_heads, dh), bw[f"{s}.q_gain"], rms_eps)
        k[s] = rms_norm(qkv[:, 1 * D:2 * D].reshape(n, n_heads, dh), bw[f"{s}.k_gain"], rms_eps)
        v[s] = qkv[:, 2 * D:3 * D].reshape(n, n_heads, dh)
        if trace is not None:
            trace[f"{s}.y1"], trace[f"{s}.qkv"] = y, qkv
    Q = apply_rope(np.concatenate([q["txt"], q["img"]], axis=0), cos, sin)
    K = apply_rope(np.concatenate([k["txt"], k["img"]], axis=0), cos, sin)
    V = np.concatenate([v["txt"], v["img"]], axis=0)
    o = attention(Q, K, V).reshape(-1, D)
    if trace is not None:
        trace["Q"], trace["K"], trace["V"], trace["o"] = Q, K, V, o
    o_s = {"txt": o[:n_txt], "img": o[n_txt:]}
    out = {}
    for s in ("txt", "img"):
        _, _, gate1, shift2, scale2, gate2 = mod[s]
        x = h[s] + gate1 * lin(o_s[s], f"{s}.out")
        y2 = layer_norm(x, ln_eps) * (1.0 + scale2) + shift2
        u = gelu_tanh(lin(y2, f"{s}.fc1"))
        out[s] = x + gate2 * lin(u, f"{s}.fc2")
        if trace is not None:
            trace[f"{s}.h_attn"], trace[f"{s}.u"] = x, u
    return out["img"], out["txt"]


def text_input(text_emb: Array, g: Dict[str, Array], rms_eps: float = 1e-6, mode: str = "blas") -> Array:
    """h_txt^0 = RMSNorm(text_emb; gain) W_txt^T + b, once per prompt (C7)."""
    return linear(rms_norm(text_emb, g["txt_gain"], rms_eps), g["txt_in_w"], g["txt_in_b"], mode)


def dit_velocity(x: Array, t: float, h_txt0: Array, g: Dict[str, Array], blocks: List[Dict[str, Array]], *,
                 n_heads: int, cos: Array, sin: Array, ln_eps: float = 1e-6, rms_eps: float = 1e-6,
                 mode: str = "blas", trace: List[Array] | None = None, block_lin=None) -> Array:
    """v = DiT(x, t, text) for one sequence.  x [N_img, C] -> v [N_img, C] (C7).
    `block_lin(block_index)` -> the `lin` hook of block_forward for that block (None = plain Linears)."""
    _, c = time_conditioning(t, g, mode)
    h_img = linear(x, g["img_in_w"], g["img_in_b"], mode)
    h_txt = h_txt0
    for bi, bw in enumerate(blocks):
        h_img, h_txt = block_forward(h_img, h_txt, c, bw, n_heads=n_heads, cos=cos, sin=sin,
                                     ln_eps=ln_eps, rms_eps=rms_eps, mode=mode,
                                     lin=None if block_lin is None else block_lin(bi))
        if trace is not None:
            trace.append(h_img)
    m_f = linear(c[None, :], g["final_mod_w"], g["final_mod_b"], mode)[0]
    D = h_img.shape[1]
    scale_f, shift_f = m_f[:D], m_f[D:]
    y = layer_norm(h_img, ln_eps) * (1.0 + scale_f) + shift_f
    return linear(y, g["proj_w"], g["proj_b"], mode)


def dit_velocity_multi(xs: Sequence[Array], t: float, h_txt0s: Sequence[Array], g: Dict[str, Array], blocks, *,
                       n_heads: int, cos: Array, sin: Array, ln_eps: float = 1e-6, rms_eps: float = 1e-6,
                       mode: str = "blas", block_lin=None, workers: int = 1) -> List[Array]:
    """dit_velocity for several INDEPENDENT sequences at the same t ("K samples from each of P prompts",
    PAPER.md:61), with the loop over blocks outermost and the loop over sequences inside it, so that a driver which
    can only hold one block's fp64 weights at a time (tests/golden/make_cfg3_golden.py) widens each block once per
    pass instead of once per sequence.  Sequence j sees exactly the operations of dit_velocity(xs[j], t,
    h_txt0s[j], ...) in the same order - no arithmetic is shared between sequences - and the test
    test_dit_velocity_multi_is_dit_velocity pins the two bit for bit.  `workers` > 1 hands the sequences of a block to
    host threads (same pin)."""
    _, c = time_conditioning(t, g, mode)
    h_img = [linear(x, g["img_in_w"], g["img_in_b"], mode) for x in xs]
    h_txt = list(h_txt0s)
    for bi, bw in enumerate(blocks):
        lin = None if block_lin is None else block_lin(bi)
        res = _pmap(lambda j: block_forward(h_img[j], h_txt[j], c, bw, n_heads=n_heads, cos=cos, sin=sin,
                                            ln_eps=ln_eps, rms_eps=rms_eps, mode=mode, lin=lin), range(len(xs)), workers)
        for j, (hi, ht) in enumerate(res):
            h_img[j], h_txt[j] = hi, ht
    m_f = linear(c[None, :], g["final_mod_w"], g["final_mod_b"], mode)[0]
    D = h_img[0].shape[1]
    scale_f, shift_f = m_f[:D], m_f[D:]
    return [linear(layer_norm(h, ln_eps) * (1.0 + scale_f) + shift_f, g["proj_w"], g["proj_b"], mode) for h in h_img]
