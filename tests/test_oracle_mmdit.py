"""Pins for oracle/mmdit.py (CPU only).  O3-O6, O11 of DESIGN.md "Oracle pins".

Every check compares the oracle with something other than itself: a torch library routine in fp64
(layer_norm, rms_norm, gelu, silu, scaled_dot_product_attention, complex multiplication for RoPE),
a brute-force Python loop, a closed form or an invariant.
"""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import mmdit
from synth import CONFIGS, make_weights, make_text_emb
from tests.helpers import np64, rel_l2, weights_np64

RNG = np.random.default_rng(20260619)


# ------------------------------------------------------------------ O3: norms, activations
def test_layer_norm_against_torch_and_invariants():
    x = RNG.normal(size=(7, 96)) * 3.0 + 1.5
    y = mmdit.layer_norm(x, 1e-6)
    ref = F.layer_norm(torch.from_numpy(x), (96,), eps=1e-6).numpy()
    assert np.abs(y - ref).max() < 1e-12
    assert np.abs(y.mean(-1)).max() < 1e-12
    var = x.var(-1)
    assert np.allclose(y.var(-1), var / (var + 1e-6), rtol=1e-12)
    assert np.abs(mmdit.layer_norm(5.0 * x, 1e-6) - y).max() < 1e-6      # scale invariance up to eps


def test_rms_norm_against_torch():
    x = RNG.normal(size=(5, 4, 64))
    gain = RNG.normal(size=64)
    y = mmdit.rms_norm(x, gain, 1e-6)
    ref = F.rms_norm(torch.from_numpy(x), (64,), torch.from_numpy(gain), eps=1e-6).numpy()
    assert np.abs(y - ref).max() < 1e-12
    unit = mmdit.rms_norm(x, np.ones(64), 0.0)
    assert np.allclose((unit ** 2).mean(-1), 1.0, rtol=1e-12)


def test_gelu_silu_against_torch():
    x = np.linspace(-6, 6, 2001)
    assert np.abs(mmdit.gelu_tanh(x) - F.gelu(torch.from_numpy(x), approximate="tanh").numpy()).max() < 1e-14
    assert np.abs(mmdit.gelu_tanh(x) - F.gelu(torch.from_numpy(x)).numpy()).max() < 1e-3     # vs erf-GELU
    assert np.abs(mmdit.silu(x) - F.silu(torch.from_numpy(x)).numpy()).max() < 1e-14


def test_timestep_embedding_closed_forms():
    e0 = mmdit.timestep_embedding(0.0)
    assert (e0[:128] == 1.0).all() and (e0[128:] == 0.0).all()
    e = mmdit.timestep_embedding(0.3)
    assert abs((e ** 2).sum() - 128.0) < 1e-9                      # cos^2 + sin^2 per frequency
    assert abs(e[0] - math.cos(300.0)) < 1e-12 and abs(e[128] - math.sin(300.0)) < 1e-12
    f_last = 10000.0 ** (-127.0 / 128.0)
    assert abs(e[127] - math.cos(300.0 * f_last)) < 1e-12 and abs(e[255] - math.sin(300.0 * f_last)) < 1e-12


def test_linear_modes_and_orientation():
    x = RNG.normal(size=(3, 5))
    w = RNG.normal(size=(4, 5))
    b = RNG.normal(size=4)
    brute = np.array([[sum(x[n, i] * w[o, i] for i in range(5)) + b[o] for o in range(4)] for n in range(3)])
    for mode in ("blas", "einsum"):
        assert np.abs(mmdit.linear(x, w, b, mode) - brute).max() < 1e-13


# ------------------------------------------------------------------ O4: RoPE
def test_rope_positions_layout():
    pos = mmdit.rope_positions(4, 6, 3)
    assert (pos[:3] == np.array([[3, 3, 3], [4, 4, 4], [5, 5, 5]])).all()     # base = max(2, 3) = 3
    assert (pos[3] == np.array([0, -2, -3])).all()                              # (r=0,c=0) centred
    assert (pos[3 + 1 * 6 + 2] == np.array([0, -1, -1])).all()
    assert (pos[-1] == np.array([0, 1, 2])).all()
    assert (mmdit.rope_positions(5, 5, 0)[0] == np.array([0, -3, -3])).all()     # ceil(5/2) = 3


def test_rope_table_frequencies():
    cos, sin = mmdit.rope_table(8, 8, 2, (4, 14, 14), 10000.0)
    assert cos.shape == (66, 32)
    # text token 1 sits at position 4 + 1 = 5 on every axis; pair 5 is h-axis pair 1 of 14
    ang = 5.0 * 10000.0 ** (-1.0 / 14.0)
    assert abs(cos[1, 5] - math.cos(ang)) < 1e-12 and abs(sin[1, 5] - math.sin(ang)) < 1e-12
    # image tokens have zero t-axis angle (pure 2-D rotation)
    assert (cos[2:, :4] == 1.0).all() and (sin[2:, :4] == 0.0).all()
    # image token (r=1, c=7): h position -3 on pairs 4..17, w position 3 on pairs 18..31
    tok = 2 + 1 * 8 + 7
    assert abs(sin[tok, 4] - math.sin(-3.0)) < 1e-12 and abs(sin[tok, 18] - math.sin(3.0)) < 1e-12
    assert abs(cos[tok, 31] - math.cos(3.0 * 10000.0 ** (-13.0 / 14.0))) < 1e-12


def test_rope_norm_identity_and_complex_form():
    S, H, dh = 66, 3, 64
    cos, sin = mmdit.rope_table(8, 8, 2, (4, 14, 14), 10000.0)
    x = RNG.normal(size=(S, H, dh))
    y = mmdit.apply_rope(x, cos, sin)
    assert np.allclose((y ** 2).sum(-1), (x ** 2).sum(-1), rtol=1e-12)
    pair_norm = lambda a: a[..., 0::2] ** 2 + a[..., 1::2] ** 2
    assert np.allclose(pair_norm(y), pair_norm(x), rtol=1e-11, atol=1e-12)
    # independent form: (x_even + i x_odd) * exp(i angle)
    z = (x[..., 0::2] + 1j * x[..., 1::2]) * (cos + 1j * sin)[:, None, :]
    assert np.abs(y[..., 0::2] - z.real).max() < 1e-13 and np.abs(y[..., 1::2] - z.imag).max() < 1e-13
    ident = mmdit.apply_rope(x, np.ones_like(cos), np.zeros_like(sin))
    assert (ident == x).all()


def test_rope_relative_position_property():
    gh, gw, dh = 6, 5, 64
    q = RNG.normal(size=(gh * gw, 1, dh))
    k = RNG.normal(size=(gh * gw, 1, dh))
    c0, s0 = mmdit.rope_table(gh, gw, 0, (4, 14, 14), 10000.0)
    c1, s1 = mmdit.rope_table(gh, gw, 0, (4, 14, 14), 10000.0, shift=(3, -2))
    sc0 = mmdit.apply_rope(q, c0, s0)[:, 0] @ mmdit.apply_rope(k, c0, s0)[:, 0].T
    sc1 = mmdit.apply_rope(q, c1, s1)[:, 0] @ mmdit.apply_rope(k, c1, s1)[:, 0].T
    assert np.abs(sc0 - sc1).max() < 1e-10


# ------------------------------------------------------------------ O5: attention
def _attention_bruteforce(q, k, v):
    S, H, dh = q.shape
    out = np.zeros_like(q)
    for h in range(H):
        for i in range(S):
            logit = [sum(q[i, h, d] * k[j, h, d] for d in range(dh)) / math.sqrt(dh) for j in range(S)]
            m = max(logit)
            w = [math.exp(l - m) for l in logit]
            z = sum(w)
            for d in range(dh):
                out[i, h, d] = sum(w[j] * v[j, h, d] for j in range(S)) / z
    return out


@pytest.mark.parametrize("S,H,dh", [(3, 1, 2), (7, 2, 4), (24, 2, 8)])
def test_attention_bruteforce(S, H, dh):
    q, k, v = (RNG.normal(size=(S, H, dh)) * 2.0 for _ in range(3))
    assert np.abs(mmdit.attention(q, k, v) - _attention_bruteforce(q, k, v)).max() < 1e-12


def test_attention_against_torch_sdpa_and_invariants():
    S, H, dh = 96, 4, 64
    q, k, v = (RNG.normal(size=(S, H, dh)) for _ in range(3))
    o = mmdit.attention(q, k, v)
    tq, tk, tv = (torch.from_numpy(a).permute(1, 0, 2)[None] for a in (q, k, v))
    ref = F.scaled_dot_product_attention(tq, tk, tv)[0].permute(1, 0, 2).numpy()
    assert np.abs(o - ref).max() < 1e-12
    perm = RNG.permutation(S)
    assert np.abs(mmdit.attention(q, k[perm], v[perm]) - o).max() < 1e-12     # key order is irrelevant
    vu = np.broadcast_to(RNG.normal(size=(1, H, dh)), (S, H, dh)).copy()
    assert np.abs(mmdit.attention(q, k, vu) - vu).max() < 1e-12               # rows of A sum to 1
    # a constant added to every logit of a row (k -> k + c*q-independent shift is not constant; scale q=0 instead)
    assert np.abs(mmdit.attention(np.zeros_like(q), k, v) - v.mean(0, keepdims=True)).max() < 1e-12
    # peaked softmax (logits ~ N(0, 16^2)): still finite and matches SDPA
    o2 = mmdit.attention(16.0 * q, k, v)
    ref2 = F.scaled_dot_product_attention(16.0 * tq, tk, tv)[0].permute(1, 0, 2).numpy()
    assert np.isfinite(o2).all() and np.abs(o2 - ref2).max() < 1e-11


# ------------------------------------------------------------------ O6: block algebra
def _tiny_block(seed=0):
    s = CONFIGS[1]
    w = make_weights(s, blocks=[0])
    g, blocks = weights_np64(w)
    bw = blocks[0]
    rng = np.random.default_rng(seed)
    bw["img.q_gain"] = rng.normal(size=s.head_dim) + 1.0
    bw["txt.k_gain"] = rng.normal(size=s.head_dim) + 1.0
    h_img = rng.normal(size=(s.n_img, s.hidden))
    h_txt = rng.normal(size=(s.n_txt, s.hidden))
    c = rng.normal(size=s.hidden)
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    return s, bw, h_img, h_txt, c, cos, sin


def test_block_zero_gates_is_identity():
    s, bw, h_img, h_txt, c, cos, sin = _tiny_block()
    D = s.hidden
    for st in ("img", "txt"):
        for chunk in (2, 5):
            bw[f"{st}.mod_w"][chunk * D:(chunk + 1) * D] = 0.0
            bw[f"{st}.mod_b"][chunk * D:(chunk + 1) * D] = 0.0
    o_img, o_txt = mmdit.block_forward(h_img, h_txt, c, bw, n_heads=s.n_heads, cos=cos, sin=sin)
    assert (o_img == h_img).all() and (o_txt == h_txt).all()


def _torch_joint_block(h_img, h_txt, c, bw, s, cos, sin):
    """Independent statement of the joint block with torch library routines (fp64)."""
    T = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    D, H, dh = s.hidden, s.n_heads, s.head_dim
    rot = torch.polar(torch.ones(cos.shape, dtype=torch.float64), torch.atan2(T(sin), T(cos)))   # e^{i angle}
    hs = {"img": T(h_img), "txt": T(h_txt)}
    mods, qs, ks, vs = {}, {}, {}, {}
    for st in ("txt", "img"):
        m = F.linear(T(c), T(bw[f"{st}.mod_w"]), T(bw[f"{st}.mod_b"]))
        mods[st] = m.chunk(6)
        y = F.layer_norm(hs[st], (D,), eps=s.ln_eps) * (1 + mods[st][1]) + mods[st][0]
        qkv = F.linear(y, T(bw[f"{st}.qkv_w"]), T(bw[f"{st}.qkv_b"])).view(-1, 3, H, dh)
        qs[st] = F.rms_norm(qkv[:, 0], (dh,), T(bw[f"{st}.q_gain"]), eps=s.rms_eps)
        ks[st] = F.rms_norm(qkv[:, 1], (dh,), T(bw[f"{st}.k_gain"]), eps=s.rms_eps)
        vs[st] = qkv[:, 2]

    def rope(x):
        z = torch.view_as_complex(x.reshape(x.shape[0], H, dh // 2, 2).contiguous()) * rot[:, None, :]
        return torch.view_as_real(z).reshape(x.shape[0], H, dh)

    Q = rope(torch.cat([qs["txt"], qs["img"]])).permute(1, 0, 2)[None]
    K = rope(torch.cat([ks["txt"], ks["img"]])).permute(1, 0, 2)[None]
    V = torch.cat([vs["txt"], vs["img"]]).permute(1, 0, 2)[None]
    o = F.scaled_dot_product_attention(Q, K, V)[0].permute(1, 0, 2).reshape(-1, D)
    os_ = {"txt": o[:s.n_txt], "img": o[s.n_txt:]}
    out = {}
    for st in ("txt", "img"):
        x = hs[st] + mods[st][2] * F.linear(os_[st], T(bw[f"{st}.out_w"]), T(bw[f"{st}.out_b"]))
        y2 = F.layer_norm(x, (D,), eps=s.ln_eps) * (1 + mods[st][4]) + mods[st][3]
        u = F.gelu(F.linear(y2, T(bw[f"{st}.fc1_w"]), T(bw[f"{st}.fc1_b"])), approximate="tanh")
        out[st] = x + mods[st][5] * F.linear(u, T(bw[f"{st}.fc2_w"]), T(bw[f"{st}.fc2_b"]))
    return out["img"].numpy(), out["txt"].numpy()


def test_block_against_torch_library_statement():
    s, bw, h_img, h_txt, c, cos, sin = _tiny_block(seed=3)
    # make the modulation and the attention matter: larger weights than the 0.02 init
    for k in list(bw):
        if k.endswith("_w") or k.endswith("_b"):
            bw[k] = bw[k] * 3.0
    o_img, o_txt = mmdit.block_forward(h_img, h_txt, c, bw, n_heads=s.n_heads, cos=cos, sin=sin)
    r_img, r_txt = _torch_joint_block(h_img, h_txt, c, bw, s, cos, sin)
    assert rel_l2(o_img, r_img) < 1e-12 and rel_l2(o_txt, r_txt) < 1e-12
    assert rel_l2(o_img, h_img) > 1e-2          # the block did something


def test_block_unmodulated_pre_ln_special_case():
    """scale = shift = 0, gate = 1: the block is a plain pre-LN joint transformer block."""
    s, bw, h_img, h_txt, c, cos, sin = _tiny_block(seed=5)
    D = s.hidden
    for st in ("img", "txt"):
        bw[f"{st}.mod_w"][:] = 0.0
        bw[f"{st}.mod_b"][:] = 0.0
        bw[f"{st}.mod_b"][2 * D:3 * D] = 1.0
        bw[f"{st}.mod_b"][5 * D:6 * D] = 1.0
    o_img, _ = mmdit.block_forward(h_img, h_txt, c, bw, n_heads=s.n_heads, cos=cos, sin=sin)
    o_img2, _ = mmdit.block_forward(h_img, h_txt, 7.0 * c + 1.0, bw, n_heads=s.n_heads, cos=cos, sin=sin)
    assert (o_img == o_img2).all()              # conditioning vector no longer matters
    r_img, _ = _torch_joint_block(h_img, h_txt, c, bw, s, cos, sin)
    assert rel_l2(o_img, r_img) < 1e-12


def test_text_input_and_final_layer_shapes():
    s = CONFIGS[1]
    g, blocks = weights_np64(make_weights(s))
    te = np64(make_text_emb(s))[0]
    h0 = mmdit.text_input(te, g)
    ref = F.linear(F.rms_norm(torch.from_numpy(te), (s.txt_dim,), eps=1e-6), torch.from_numpy(g["txt_in_w"]),
                   torch.from_numpy(g["txt_in_b"])).numpy()
    assert np.abs(h0 - ref).max() < 1e-12
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    x = RNG.normal(size=(s.n_img, s.latent_ch))
    v = mmdit.dit_velocity(x, 0.75, h0, g, blocks, n_heads=s.n_heads, cos=cos, sin=sin)
    assert v.shape == x.shape and np.isfinite(v).all()
    # zero projection => zero velocity
    g0 = dict(g, proj_w=np.zeros_like(g["proj_w"]), proj_b=np.zeros_like(g["proj_b"]))
    assert (mmdit.dit_velocity(x, 0.75, h0, g0, blocks, n_heads=s.n_heads, cos=cos, sin=sin) == 0).all()


# ------------------------------------------------------------------ C4 / C7: conditioning and the final layer
def _read_hand_case():
    rows = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "final_layer_hand.txt")):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            rows[k] = np.asarray([float(t) for t in v])
    return rows


def _hand_case_weights():
    w1 = np.zeros((4, 256))
    w1[0, 0] = 1.0
    return {"time_w1": w1, "time_b1": np.array([0.0, 1.0, 0.0, 0.0]), "time_w2": np.diag([2.0, -1.0, 1.0, 1.0]),
            "time_b2": np.array([0.0, 0.0, 0.0, 1.0]), "img_in_w": np.eye(4), "img_in_b": np.zeros(4),
            "final_mod_w": np.concatenate([np.eye(4), 0.5 * np.eye(4)]),
            "final_mod_b": np.array([0.25, -0.5, 0.0, 1.0, 0.1, 0.2, -0.3, 0.4]),
            "proj_w": np.array([[1.0, 0, 0, 0], [0, 2.0, 0, 0], [0, 0, 1.0, 1.0], [0, 0, 0, -1.0]]),
            "proj_b": np.array([0.0, 0.0, 0.0, 10.0])}


def test_time_conditioning_and_final_layer_hand_worked_case():
    """tests/golden/final_layer_hand.txt: numbers worked out with decimal arithmetic.  Fails if scale_f / shift_f are
    swapped, if temb instead of SiLU(temb) feeds the modulation, if the LN epsilon is not 1e-6 inside the root, if
    W1 / W2 / the biases of the time MLP are composed differently, or if proj is applied transposed."""
    r = _read_hand_case()
    g = _hand_case_weights()
    temb, c = mmdit.time_conditioning(0.0, g)
    assert np.abs(temb - r["temb"]).max() < 1e-15 and np.abs(c - r["c"]).max() < 1e-15
    x = np.stack([r["x0"], r["x1"]])
    none = np.zeros((0, 4))
    v = mmdit.dit_velocity(x, 0.0, none, g, [], n_heads=1, cos=None, sin=None, ln_eps=1e-6)
    assert np.abs(v - np.stack([r["v0"], r["v1"]])).max() < 1e-13
    vm = mmdit.dit_velocity_multi([x[:1], x[1:]], 0.0, [none, none], g, [], n_heads=1, cos=None, sin=None, ln_eps=1e-6)
    assert np.abs(np.concatenate(vm) - np.stack([r["v0"], r["v1"]])).max() < 1e-13
    # the case is sensitive to the epsilon: row x0 has variance 1e-6
    v_bad = mmdit.dit_velocity(x, 0.0, none, g, [], n_heads=1, cos=None, sin=None, ln_eps=1e-5)
    assert np.abs(v_bad[0] - r["v0"]).max() > 0.1


def _torch_velocity(x, t, h_txt0, g, blocks, s, cos, sin, *, swap=False, raw_temb=False, final_eps=None):
    """Independent statement of v = DiT(x, t, text) with torch library routines (fp64); the keyword arguments build
    the plausible MISTAKES the pin must reject."""
    T = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    D = s.hidden
    freqs = torch.pow(torch.tensor(10000.0, dtype=torch.float64), -torch.arange(128, dtype=torch.float64) / 128.0)
    ang = 1000.0 * t * freqs
    e = torch.cat([torch.cos(ang), torch.sin(ang)])
    temb = F.linear(F.silu(F.linear(e, T(g["time_w1"]), T(g["time_b1"]))), T(g["time_w2"]), T(g["time_b2"]))
    c = temb if raw_temb else F.silu(temb)
    h_img, h_txt = F.linear(T(x), T(g["img_in_w"]), T(g["img_in_b"])).numpy(), h_txt0
    for bw in blocks:
        h_img, h_txt = _torch_joint_block(h_img, h_txt, c.numpy(), bw, s, cos, sin)
    a, b = F.linear(c, T(g["final_mod_w"]), T(g["final_mod_b"])).chunk(2)
    scale, shift = (b, a) if swap else (a, b)
    y = F.layer_norm(T(h_img), (D,), eps=s.ln_eps if final_eps is None else final_eps) * (1 + scale) + shift
    return F.linear(y, T(g["proj_w"]), T(g["proj_b"])).numpy()


def test_velocity_against_torch_library_statement_and_its_mutants():
    """Pins dit_velocity end to end (time MLP -> c = SiLU(temb) -> img_in -> blocks -> final modulation split
    (scale_f, shift_f) -> LN with ln_eps -> proj) against torch library routines, with ln_eps != rms_eps and
    weights large enough that every term matters; each plausible mistake moves the result by > 1e-3."""
    s = CONFIGS[1].with_(ln_eps=1e-2)
    g, blocks = weights_np64(make_weights(s))
    for k in g:
        g[k] = g[k] * (8.0 if k.startswith(("final_mod", "time_")) else 3.0)
    te = np64(make_text_emb(s))[0]
    h0 = mmdit.text_input(te, g, s.rms_eps)
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    x = RNG.normal(size=(s.n_img, s.latent_ch)) * 0.05        # small rows: the LN epsilon matters
    for t in (0.75, 0.1):
        v = mmdit.dit_velocity(x, t, h0, g, blocks, n_heads=s.n_heads, cos=cos, sin=sin, ln_eps=s.ln_eps, rms_eps=s.rms_eps)
        ref = _torch_velocity(x, t, h0, g, blocks, s, cos, sin)
        assert rel_l2(v, ref) < 1e-12
        for mistake in (dict(swap=True), dict(raw_temb=True), dict(final_eps=s.rms_eps)):
            assert rel_l2(_torch_velocity(x, t, h0, g, blocks, s, cos, sin, **mistake), ref) > 1e-3, mistake
    # temb / c themselves
    temb, c = mmdit.time_conditioning(0.3, g)
    assert np.abs(c - F.silu(torch.from_numpy(temb)).numpy()).max() < 1e-14 and np.abs(c - temb).max() > 1e-3


def test_dit_velocity_multi_is_dit_velocity():
    """The blocks-outermost loop order used by the full-size golden script gives, per sequence, the bits of dit_velocity."""
    s = CONFIGS[1]
    g, blocks = weights_np64(make_weights(s))
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h0s = [mmdit.text_input(np64(make_text_emb(s, prompts=[p]))[0], g) for p in (0, 1, 0)]
    xs = [RNG.normal(size=(s.n_img, s.latent_ch)) for _ in range(3)]
    vm = mmdit.dit_velocity_multi(xs, 0.6, h0s, g, iter(blocks), n_heads=s.n_heads, cos=cos, sin=sin)
    for j in range(3):
        assert (vm[j] == mmdit.dit_velocity(xs[j], 0.6, h0s[j], g, blocks, n_heads=s.n_heads, cos=cos, sin=sin)).all()
    assert not (vm[0] == vm[2]).all() and rel_l2(vm[0], vm[1]) > 1e-6
    # host threads (over sequences; over heads and row blocks) change nothing, bit for bit
    vt = mmdit.dit_velocity_multi(xs, 0.6, h0s, g, iter(blocks), n_heads=s.n_heads, cos=cos, sin=sin, workers=3)
    mmdit.set_workers(4)
    try:
        vw = mmdit.dit_velocity(xs[1], 0.6, h0s[1], g, blocks, n_heads=s.n_heads, cos=cos, sin=sin)
        u = RNG.normal(size=(1280, 96)) * 3.0
        gw = mmdit.gelu_tanh(u)
    finally:
        mmdit.set_workers(1)
    assert all((vt[j] == vm[j]).all() for j in range(3)) and (vw == vm[1]).all() and (gw == mmdit.gelu_tanh(u)).all()


def test_parameter_count_matches_20b():
    """36 D^2 per block x 60 blocks = 20.4 B parameters: 'Qwen-Image (20B parameters)' PAPER.md:79."""
    s = CONFIGS[3]
    from synth.manifest import block_tensor_shapes
    per_stream = sum(int(np.prod(v)) for v in block_tensor_shapes(s).values())
    total = 2 * per_stream * s.n_blocks
    assert 20.0e9 < total < 20.8e9


# ------------------------------------------------------------------ O11: back ends agree
def test_einsum_and_blas_backends_agree_on_cfg1_velocity():
    s = CONFIGS[1]
    g, blocks = weights_np64(make_weights(s))
    te = np64(make_text_emb(s))[0]
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    x = RNG.normal(size=(s.n_img, s.latent_ch))
    va = mmdit.dit_velocity(x, 0.5, mmdit.text_input(te, g, mode="blas"), g, blocks, n_heads=s.n_heads, cos=cos, sin=sin, mode="blas")
    vb = mmdit.dit_velocity(x, 0.5, mmdit.text_input(te, g, mode="einsum"), g, blocks, n_heads=s.n_heads, cos=cos, sin=sin, mode="einsum")
    assert rel_l2(va, vb) < 1e-12
