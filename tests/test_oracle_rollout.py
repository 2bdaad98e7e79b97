"""Pins for oracle/rollout.py (CPU only).  O7-O10 of DESIGN.md "Oracle pins"."""
import numpy as np
import pytest

from oracle import mmdit, philox, rollout
from synth import CONFIGS, make_probe, make_text_emb, make_weights
from tests.helpers import np64, rel_l2, weights_np64

RNG = np.random.default_rng(7)


def test_euler_zero_and_constant_velocity():
    x0 = RNG.normal(size=(16, 8))
    grid = [1.0, 0.8, 0.55, 0.2, 0.0]
    assert (rollout.euler_denoise(x0, grid, lambda x, t: np.zeros_like(x)) == x0).all()      # O7
    v0 = RNG.normal(size=(16, 8))
    xT = rollout.euler_denoise(x0, grid, lambda x, t: v0)
    assert np.abs(xT - (x0 + (grid[-1] - grid[0]) * v0)).max() < 1e-14


def test_euler_rectified_flow_closed_form():
    """O8: x_t = (1-t) x0 + t eps with v = eps - x0 (constant along the path): any grid from t=1 lands on
    x(t_T) = (1 - t_T) x0 + t_T eps exactly."""
    x0 = RNG.normal(size=(32, 4))
    eps = RNG.normal(size=(32, 4))
    for grid in ([1.0, 0.0], [1.0, 0.9, 0.1, 0.0], list(np.linspace(1, 0, 11)), [1.0, 0.7, 0.25]):
        hist = []
        xT = rollout.euler_denoise(eps, grid, lambda x, t: eps - x0, hist)
        tT = grid[-1]
        assert np.abs(xT - ((1 - tT) * x0 + tT * eps)).max() < 1e-14
        for ti, xi in zip(grid[1:], hist):
            assert np.abs(xi - ((1 - ti) * x0 + ti * eps)).max() < 1e-14


def test_euler_evaluates_model_at_t0_to_tTminus1_only():
    seen = []
    rollout.euler_denoise(np.zeros(3), [1.0, 0.75, 0.5, 0.25, 0.0], lambda x, t: (seen.append(t), x)[1])
    assert seen == [1.0, 0.75, 0.5, 0.25]


def test_euler_linear_ode_converges_first_order():
    """dx/dt = -x from t=1 to 0 has x(0) = e x(1); Euler's error halves when the step halves."""
    errs = []
    for T in (50, 100, 200):
        xT = rollout.euler_denoise(np.ones(1), np.linspace(1, 0, T + 1), lambda x, t: -x)
        errs.append(abs(xT[0] - np.e))
    assert 1.9 < errs[0] / errs[1] < 2.1 and 1.9 < errs[1] / errs[2] < 2.1


def test_reward_linear_and_normalised():
    p = RNG.normal(size=4096)
    x, y = RNG.normal(size=(64, 64)), RNG.normal(size=(64, 64))
    r = rollout.probe_reward
    assert abs(r(2.0 * x - 3.0 * y, p) - (2.0 * r(x, p) - 3.0 * r(y, p))) < 1e-12
    assert abs(r(p.reshape(64, 64), p) - (p ** 2).sum() / 64.0) < 1e-10          # sqrt(4096) = 64
    assert r(np.zeros((64, 64)), p) == 0.0


def test_selection_hand_written_with_tie():
    #            0    1    2    3    4    5    6    7
    r = np.array([[0.5, 2.0, -1.0, 2.0, 0.0, -1.0, 3.0, 0.25]])
    out = rollout.select_seeds(r, 3)
    assert out["top"].tolist() == [[6, 1, 3]]           # tie 2.0: lower index first
    assert out["bottom"].tolist() == [[2, 5, 4]]        # tie -1.0: lower index first
    assert out["argmax"].tolist() == [6] and out["argmin"].tolist() == [2]
    assert abs(out["mean"][0] - r.mean()) < 1e-15
    assert abs(out["std"][0] - np.std(r[0])) < 1e-15     # population form (ddof = 0)
    const = rollout.select_seeds(np.full((2, 4), 1.25), 2)
    assert (const["std"] == 0).all() and const["top"].tolist() == [[0, 1], [0, 1]]
    assert const["bottom"].tolist() == [[0, 1], [0, 1]]


def test_selection_against_numpy_sort_random():
    r = RNG.normal(size=(5, 32))
    out = rollout.select_seeds(r, 16)
    for g in range(5):
        order = np.argsort(r[g], kind="stable")
        assert out["bottom"][g].tolist() == order[:16].tolist()
        assert out["top"][g].tolist() == order[::-1][:16].tolist()
    assert set(out["top"][0]).isdisjoint(set(out["bottom"][0]))


def _cfg1():
    s = CONFIGS[1]
    g, blocks = weights_np64(make_weights(s))
    return s, g, blocks, np64(make_text_emb(s))[0], np64(make_probe(s))


def _explore(s, g, blocks, te, probe, seeds, grid, **kw):
    return rollout.explore(seeds, te, grid, g, blocks, probe, n_heads=s.n_heads, grid_h=s.grid_h, grid_w=s.grid_w,
                           rope_pairs=s.rope_pairs, rope_theta=s.rope_theta, latent_ch=s.latent_ch, **kw)


def test_explore_seed_independence_resume_and_backends():
    s, g, blocks, te, probe = _cfg1()
    grid = s.timesteps
    hist = []
    lat, rew = _explore(s, g, blocks, te, probe, [0, 1, 2, 3], grid, history=hist)
    assert lat.shape == (4, s.n_img, s.latent_ch) and np.isfinite(lat).all()
    lat2, rew2 = _explore(s, g, blocks, te, probe, [2], grid)                     # O10: batch independence
    assert (lat2[0] == lat[2]).all() and rew2[0] == rew[2]
    # O10: resume from the latents after step 2
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h0 = mmdit.text_input(te, g)
    vel = lambda x, t: mmdit.dit_velocity(x, t, h0, g, blocks, n_heads=s.n_heads, cos=cos, sin=sin)
    resumed = rollout.euler_denoise(hist[1][1], grid[2:], vel)
    assert (resumed == lat[1]).all()
    # O11: the two matmul back ends agree end to end
    lat3, rew3 = _explore(s, g, blocks, te, probe, [0], grid, mode="einsum")
    assert rel_l2(lat3[0], lat[0]) < 1e-12 and abs(rew3[0] - rew[0]) < 1e-10
    # the rollout moves the latent and rewards differ across seeds
    x0 = philox.noise_from_seeds([0], s.n_img * s.latent_ch)[0].reshape(s.n_img, s.latent_ch)
    assert rel_l2(lat[0], x0) > 1e-2 and np.std(rew) > 1e-2


def test_explore_zero_velocity_returns_noise():
    s, g, blocks, te, probe = _cfg1()
    g0 = dict(g, proj_w=np.zeros_like(g["proj_w"]), proj_b=np.zeros_like(g["proj_b"]))
    lat, rew = _explore(s, g0, blocks, te, probe, [9], s.timesteps)
    x0 = philox.noise_from_seeds([9], s.n_img * s.latent_ch)[0].reshape(s.n_img, s.latent_ch)
    assert (lat[0] == x0).all()
    assert abs(rew[0] - rollout.probe_reward(x0, probe)) < 1e-15
