"""Pins for oracle/fp8.py (CPU only).  The E4M3 rounding is pinned against PyTorch's float8_e4m3fn cast (an independent
implementation) on every representable value, on midpoints (ties to even) and on random data; saturation and the
subnormal grid by hand; the quantised Linear by its error bound and by exactness on representable inputs; the hook in
mmdit.block_forward by equality with the plain block when the hook is the plain Linear."""
import numpy as np
import torch

from oracle import fp8, mmdit
from synth import CONFIGS, make_block_inputs, make_weights
from tests.helpers import np64, rel_l2, weights_np64


def _all_e4m3_values():
    bits = torch.arange(256, dtype=torch.uint8)
    v = bits.view(torch.float8_e4m3fn).to(torch.float64).numpy()
    return v[np.isfinite(v)]


def test_e4m3_against_torch_cast():
    grid = np.unique(_all_e4m3_values())
    assert grid.max() == 448.0 and np.abs(grid[grid != 0]).min() == 2.0 ** -9 and len(grid) == 253
    assert (fp8.e4m3(grid) == grid).all()                               # representable values are fixed points
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.normal(size=200000) * s for s in (1e-3, 0.05, 1.0, 30.0)])
    x = x[np.abs(x) < 440.0].astype(np.float32).astype(np.float64)      # torch's cast does not saturate: stay in range
    ref = torch.from_numpy(x).to(torch.float32).to(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert (fp8.e4m3(x) == ref).all()
    pos = grid[grid >= 0]
    mid = 0.5 * (pos[:-1] + pos[1:])                                    # exact ties
    ref_mid = torch.from_numpy(mid).to(torch.float32).to(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert (fp8.e4m3(mid) == ref_mid).all() and (fp8.e4m3(-mid) == -ref_mid).all()


def test_e4m3_hand_values():
    f = fp8.e4m3
    assert f(np.array([0.0, 1.0, 1.0625, 1.1875, 3.3, 447.0, 448.0, 464.0, 1e9, -1e9])).tolist() == \
        [0.0, 1.0, 1.0, 1.25, 3.25, 448.0, 448.0, 448.0, 448.0, -448.0]    # ties to even: 1.0625 -> 1.0, 1.1875 -> 1.25
    assert f(np.array([2.0 ** -9, 2.0 ** -10, 0.6 * 2.0 ** -9, 1.5 * 2.0 ** -9])).tolist() == \
        [2.0 ** -9, 0.0, 2.0 ** -9, 2.0 ** -8]                             # subnormal grid, spacing 2^-9


def test_weight_quantisation_and_linear():
    rng = np.random.default_rng(2)
    w = rng.normal(size=(48, 256)) * 0.02
    w[5] = 0.0
    wq, s = fp8.quantize_weight(w)
    assert s[5] == 1.0 and (wq[5] == 0).all()
    assert np.allclose(np.abs(wq).max(axis=1)[np.arange(48) != 5], 448.0)     # the row maximum maps to 448
    assert np.abs(wq * s[:, None] - w).max() <= np.abs(w).max(axis=1).max() * 2.0 ** -4 * 1.0001
    x = rng.normal(size=(64, 256))
    b = rng.normal(size=48) * 0.1
    y = fp8.linear_fp8(x, wq, s, b)
    assert 0.01 < rel_l2(y - b, x @ w.T) < 0.08                               # 3 mantissa bits on both operands
    xr = fp8.e4m3(x)                                                          # representable inputs: only W is rounded
    assert np.abs(fp8.linear_fp8(xr, wq, s, b) - ((xr @ wq.T) * s + b)).max() == 0.0


def test_block_hook_is_neutral_and_fp8_block_is_close():
    s = CONFIGS[1]
    g, blocks = weights_np64(make_weights(s))
    h_img, h_txt, temb = (np64(t) for t in make_block_inputs(s, 1))
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    c = mmdit.silu(temb)
    kw = dict(n_heads=s.n_heads, cos=cos, sin=sin)
    bw = blocks[0]
    ref = mmdit.block_forward(h_img[0], h_txt[0], c, bw, **kw)
    plain = lambda x, name: x @ bw[f"{name}_w"].T + bw[f"{name}_b"]
    hooked = mmdit.block_forward(h_img[0], h_txt[0], c, bw, lin=plain, **kw)
    assert all(np.abs(a - b).max() < 1e-13 for a, b in zip(ref, hooked))
    q = fp8.block_forward_fp8(h_img[0], h_txt[0], c, bw, **kw)
    for a, b in zip(q, ref):
        assert 1e-4 < rel_l2(a, b) < 5e-2                                     # quantisation is visible but small
