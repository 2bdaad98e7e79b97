"""Shared helpers of the -m gpu parity tests: build the library, make inputs with synth/, wrap the oracle."""
import numpy as np
import torch

import paper_2606_19004_b200 as spot
from oracle import mmdit, rollout
from paper_2606_19004_b200 import build as spot_build
from synth import make_probe, make_text_emb, make_weights
from tests.helpers import np64, weights_np64


def ensure_built():
    spot_build.build()
    return spot.load_library()


def device_weights(shape, blocks=None):
    """Weights generated on the device by synth/ and the SAME values copied to the host for the oracle."""
    w = make_weights(shape, device="cuda", blocks=blocks)
    return w


def oracle_weights(w):
    return weights_np64(w)


def f32_timesteps(shape):
    return [float(np.float32(t)) for t in shape.timesteps]


def oracle_explore(shape, w, text_emb, probe, seeds, timesteps, history=None):
    """Oracle rollout for ONE prompt; text_emb [n_txt, D] torch tensor."""
    g, blocks = oracle_weights(w)
    f32 = lambda a: a.astype(np.float32).astype(np.float64)       # the CUDA path stores the initial latent in fp32
    return rollout.explore(list(seeds), np64(text_emb), timesteps, g, blocks, np64(probe), n_heads=shape.n_heads,
                           grid_h=shape.grid_h, grid_w=shape.grid_w, rope_pairs=shape.rope_pairs,
                           rope_theta=shape.rope_theta, ln_eps=shape.ln_eps, rms_eps=shape.rms_eps,
                           latent_ch=shape.latent_ch, x0_cast=f32, history=history)


def oracle_block(shape, bw_np, h_img, h_txt, temb, trace=None):
    """Oracle block forward for a batch: h_img [B,n_img,D], h_txt [B,n_txt,D] numpy fp64; temb [D]."""
    cos, sin = mmdit.rope_table(shape.grid_h, shape.grid_w, shape.n_txt, shape.rope_pairs, shape.rope_theta)
    c = mmdit.silu(temb)
    outs_i, outs_t = [], []
    for b in range(h_img.shape[0]):
        tr = {} if trace is not None else None
        oi, ot = mmdit.block_forward(h_img[b], h_txt[b], c, bw_np, n_heads=shape.n_heads, cos=cos, sin=sin,
                                     ln_eps=shape.ln_eps, rms_eps=shape.rms_eps, trace=tr)
        outs_i.append(oi)
        outs_t.append(ot)
        if trace is not None:
            trace.append(tr)
    return np.stack(outs_i), np.stack(outs_t)
