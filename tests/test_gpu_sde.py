"""-m gpu parity of the stochastic sampler step (spot_sde_update, spot_dit_denoise_sde) against oracle/sde.py
(PAPER.md:227 FlowGRPO backbone, Table 2 "SDE window").

Tolerances: the step is fp32 arithmetic on an fp32 Box-Muller normal (K1's parity bound: 2e-6 absolute), so one step
agrees to 1e-5 relative L2 and the log-probability to 1e-5 absolute; whole rollouts keep the north-star bounds
(1e-4 fp32 config, 5e-2 bf16)."""
import math

import numpy as np
import pytest
import torch

import paper_2606_19004_b200 as spot
from oracle import mmdit, philox, sde
from synth import CONFIGS, hash_normal, make_text_emb
from tests.gpu_common import device_weights, ensure_built, oracle_weights
from tests.helpers import np64, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    ensure_built()


def _seeds(vals):
    return torch.tensor([v if v < 2 ** 63 else v - 2 ** 64 for v in vals], dtype=torch.int64, device="cuda")


@pytest.mark.parametrize("t_i,t_next,a,step", [(0.7, 0.6, 0.8, 2), (1.0, 0.9, 0.7, 0), (0.1, 0.0, 1.0, 9), (0.55, 0.2, 0.3, 5)])
def test_sde_update_matches_oracle(t_i, t_next, a, step):
    seeds = [0, 5, 2 ** 64 - 1]
    E = 64 * 64 + 4 * 37                                        # several 4096-element chunks plus a ragged tail
    x = hash_normal(1001, 3 * E, 1.0, torch.float32, "cuda").reshape(3, E)
    v = hash_normal(1002, 3 * E, 1.0, torch.float32, "cuda").reshape(3, E)
    t_i, t_next = float(np.float32(t_i)), float(np.float32(t_next))
    xo, lp = spot.spot_sde_update(x.clone(), v, _seeds(seeds), step, t_i, t_next, a)
    for b, s in enumerate(seeds):
        xi = sde.step_noise(s, step, (E,))
        ref, ref_lp = sde.sde_step(np64(x[b]), np64(v[b]), t_i, t_next, float(np.float32(a)), xi)
        assert rel_l2(np64(xo[b]), ref) < 1e-5
        assert abs(lp[b].item() - ref_lp) < 1e-5 * max(1.0, abs(ref_lp))
    again, lp2 = spot.spot_sde_update(x.clone(), v, _seeds(seeds), step, t_i, t_next, a)
    assert torch.equal(again, xo) and torch.equal(lp2, lp)     # deterministic
    alone, lp1 = spot.spot_sde_update(x[1:2].clone(), v[1:2], _seeds(seeds[1:2]), step, t_i, t_next, a)
    assert torch.equal(alone[0], xo[1]) and torch.equal(lp1[0], lp[1])          # batch independent


def test_sde_update_zero_noise_is_the_euler_update():
    E = 4096 + 8
    x = hash_normal(1003, 2 * E, 1.0, torch.float32, "cuda").reshape(2, E)
    v = hash_normal(1004, 2 * E, 1.0, torch.float32, "cuda").reshape(2, E)
    xo, lp = spot.spot_sde_update(x.clone(), v, _seeds([1, 2]), 0, 0.75, 0.5, 0.0)
    xe, _ = spot.spot_euler_update(x.clone(), v, -0.25)
    assert torch.equal(xo, xe) and (lp == 0).all()


def test_sde_log_probability_statistics():
    """xi ~ N(0,1): mean(xi^2) -> 1, so log p -> -1/2 - log(sigma sqrt(-dt)) - log(2 pi)/2 on a large latent."""
    E = 1 << 22
    x = torch.zeros((1, E), device="cuda")
    v = torch.zeros((1, E), device="cuda")
    xo, lp = spot.spot_sde_update(x, v, _seeds([123]), 1, 0.5, 0.25, 1.0)
    std = 1.0 * math.sqrt(0.25)
    assert abs(lp.item() - (-0.5 - math.log(std) - 0.5 * math.log(2 * math.pi))) < 2e-3
    assert abs(xo.var().item() - std * std) < 2e-3 and abs(xo.mean().item()) < 2e-3


def test_cfg1_denoise_sde_matches_oracle():
    s = CONFIGS[1]
    w = device_weights(s)
    ctx = spot.Context(s, w, max_seqs=4)
    text = make_text_emb(s, "cuda")
    g, blocks = oracle_weights(w)
    ts = [float(np.float32(t)) for t in np.linspace(1.0, 0.0, 6)]
    seeds = [0, 1, 7]
    a, window = 0.7, (0, 4)
    lat = spot.spot_noise_from_seeds(_seeds(seeds), s.n_img * s.latent_ch).reshape(3, s.n_img, s.latent_ch)
    x0 = np64(lat)
    out, logp = spot.spot_dit_denoise_sde(ctx, _seeds(seeds), lat, text, ts, 1, 3, a, window)
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h_txt0 = mmdit.text_input(np64(text)[0], g)
    vel = lambda x, t: mmdit.dit_velocity(x, t, h_txt0, g, blocks, n_heads=s.n_heads, cos=cos, sin=sin)
    for b, sd in enumerate(seeds):
        ref, ref_lp = sde.denoise_sde(x0[b], sd, ts, vel, float(np.float32(a)), window)
        assert rel_l2(np64(out[b]), ref) < 1e-4
        assert np.abs(np64(logp[b]) - ref_lp).max() < 1e-4 * max(1.0, np.abs(ref_lp).max())
        assert logp[b, 4].item() == 0.0                          # outside the window: deterministic step
    # a rollout split over two calls with first_step = steps already taken is the unsplit rollout, bit for bit
    lat_s = spot.spot_noise_from_seeds(_seeds(seeds), s.n_img * s.latent_ch).reshape(3, s.n_img, s.latent_ch)
    _, lp1 = spot.spot_dit_denoise_sde(ctx, _seeds(seeds), lat_s, text, ts[:3], 1, 3, a, window)
    _, lp2 = spot.spot_dit_denoise_sde(ctx, _seeds(seeds), lat_s, text, ts[2:], 1, 3, a, window, first_step=2)
    assert torch.equal(lat_s, out) and torch.equal(torch.cat([lp1, lp2], 1), logp)
    # an empty window is the plain deterministic denoise, bit for bit
    lat_a = spot.spot_noise_from_seeds(_seeds(seeds), s.n_img * s.latent_ch).reshape(3, s.n_img, s.latent_ch)
    lat_b = lat_a.clone()
    spot.spot_dit_denoise_sde(ctx, _seeds(seeds), lat_a, text, ts, 1, 3, a, (2, 2))
    spot.spot_dit_denoise(ctx, lat_b, text, ts, 1, 3)
    assert torch.equal(lat_a, lat_b)
    # SPOT_OPT_CHUNK_SEQS: the stochastic rollout in chunks of 2 + 1 sequences gives the bits of the one-pass call
    try:
        spot.spot_set_option(ctx, spot.OPT_CHUNK_SEQS, 2)
        lat_c = spot.spot_noise_from_seeds(_seeds(seeds), s.n_img * s.latent_ch).reshape(3, s.n_img, s.latent_ch)
        out_c, logp_c = spot.spot_dit_denoise_sde(ctx, _seeds(seeds), lat_c, text, ts, 1, 3, a, window)
        assert torch.equal(out_c, out) and torch.equal(logp_c, logp)
    finally:
        spot.spot_set_option(ctx, spot.OPT_CHUNK_SEQS, 32)


def test_denoise_sde_bf16_full_width_reduced_depth():
    s = CONFIGS[3].with_(n_blocks=2, seeds_per_prompt=2, n_steps=3)
    w = device_weights(s)
    ctx = spot.Context(s, w, max_seqs=2)
    text = make_text_emb(s, "cuda")
    g, blocks = oracle_weights(w)
    ts = [float(np.float32(t)) for t in s.timesteps]
    seeds = [3, 4]
    lat = spot.spot_noise_from_seeds(_seeds(seeds), s.n_img * s.latent_ch).reshape(2, s.n_img, s.latent_ch)
    x0 = np64(lat)
    out, logp = spot.spot_dit_denoise_sde(ctx, _seeds(seeds), lat, text, ts, 1, 2, 0.7, (0, 2))
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h_txt0 = mmdit.text_input(np64(text)[0], g)
    vel = lambda x, t: mmdit.dit_velocity(x, t, h_txt0, g, blocks, n_heads=s.n_heads, cos=cos, sin=sin)
    ref, ref_lp = sde.denoise_sde(x0[0], seeds[0], ts, vel, float(np.float32(0.7)), (0, 2))
    e = rel_l2(np64(out[0]), ref)
    print(f"sde bf16 depth-2: latents rel-L2 {e:.3e}, logp {np64(logp[0]).tolist()} vs {ref_lp.tolist()}")
    assert e < 5e-2
    assert np.abs(np64(logp[0]) - ref_lp).max() < 1e-4 * max(1.0, np.abs(ref_lp).max())


def test_sde_argument_errors():
    x = torch.zeros((1, 8), device="cuda")
    with pytest.raises(spot.SpotError):
        spot.spot_sde_update(x, x.clone(), _seeds([0]), 0, 0.5, 0.6, 0.5)       # t must decrease
    with pytest.raises(spot.SpotError):
        spot.spot_sde_update(x, x.clone(), _seeds([0]), 0, 0.5, 0.4, -0.5)      # negative noise level
