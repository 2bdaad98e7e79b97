"""Pins for oracle/teacache.py (CPU only): the cached-step exploration rule of PAPER.md:155-157.

What fixes the oracle other than itself:
  * threshold 0 computes every step, so the result must equal the plain rollout oracle exactly;
  * a constant rescaling polynomial makes the skip pattern pure arithmetic, worked by hand from the rule;
  * rel-L1 on hand values; first and last steps always computed; fewer steps as the threshold grows;
  * a skipped step must add the residual of the LAST COMPUTED step: rebuilt in the test from mmdit.dit_velocity's
    per-block trace (an independent route through already pinned functions);
  * identity blocks (all gates zero) have zero residual, so skipping is exact for any threshold.
"""
import numpy as np

from oracle import mmdit, philox, rollout, teacache
from synth import CONFIGS, make_probe, make_text_emb, make_weights
from tests.helpers import np64, weights_np64


def _tiny():
    s = CONFIGS[1]
    g, blocks = weights_np64(make_weights(s))
    text = np64(make_text_emb(s))[0]
    probe = np64(make_probe(s))
    kw = dict(n_heads=s.n_heads, grid_h=s.grid_h, grid_w=s.grid_w, rope_pairs=s.rope_pairs, rope_theta=s.rope_theta,
              latent_ch=s.latent_ch)
    return s, g, blocks, text, probe, kw


def test_rel_l1_and_poly_hand_values():
    assert teacache.rel_l1(np.array([[1.0, 2.0]]), np.array([[1.0, 1.0]])) == 0.5          # (0 + 1)/2 over (1 + 1)/2
    assert teacache.rel_l1(np.array([3.0, -3.0]), np.array([-1.0, 1.0])) == 4.0
    assert teacache.poly_eval([0.0, 1.0], 0.37) == 0.37
    assert abs(teacache.poly_eval([1.0, -2.0, 3.0], 2.0) - (1.0 - 4.0 + 12.0)) < 1e-15


def test_threshold_zero_equals_plain_rollout():
    s, g, blocks, text, probe, kw = _tiny()
    ts = list(np.linspace(1.0, 0.0, 5))
    lat, rew, comp = teacache.explore_cached([0, 3], text, ts, g, blocks, probe, 0.0, **kw)
    ref_lat, ref_rew = rollout.explore([0, 3], text, ts, g, blocks, probe, **kw)
    assert comp.all()
    assert (lat == ref_lat).all() and (rew == ref_rew).all()


def test_constant_polynomial_gives_the_hand_worked_pattern():
    """poly == 1: acc grows by 1 per middle step; compute when acc >= 3 and reset.  T = 10, worked by hand:
    step 0 computed (first); 1: acc 1 skip; 2: acc 2 skip; 3: acc 3 compute, reset; 4, 5 skip; 6 compute; 7, 8 skip;
    9 computed (last)."""
    s, g, blocks, text, probe, kw = _tiny()
    ts = list(np.linspace(1.0, 0.0, 11))
    traces = []
    _, _, comp = teacache.explore_cached([1], text, ts, g, blocks, probe, 3.0, coeffs=(1.0,), traces=traces, **kw)
    assert comp[0].astype(int).tolist() == [1, 0, 0, 1, 0, 0, 1, 0, 0, 1]
    assert traces[0]["acc"][1:9] == [1.0, 2.0, 3.0, 1.0, 2.0, 3.0, 1.0, 2.0]
    # threshold 2.5 behaves the same (first acc >= 2.5 is 3); threshold 1 computes every step
    _, _, c2 = teacache.explore_cached([1], text, ts, g, blocks, probe, 2.5, coeffs=(1.0,), **kw)
    assert (c2 == comp).all()
    _, _, c3 = teacache.explore_cached([1], text, ts, g, blocks, probe, 1.0, coeffs=(1.0,), **kw)
    assert c3.all()


def test_first_and_last_always_computed_and_monotone_in_threshold():
    s, g, blocks, text, probe, kw = _tiny()
    ts = list(np.linspace(1.0, 0.0, 9))
    counts = []
    for thr in (0.0, 0.05, 0.2, 0.8, 1e9):
        _, _, comp = teacache.explore_cached([2], text, ts, g, blocks, probe, thr, **kw)
        assert comp[0, 0] and comp[0, -1]
        counts.append(int(comp.sum()))
    assert counts[0] == 8 and counts[-1] == 2
    assert all(a >= b for a, b in zip(counts, counts[1:]))


def test_skipped_step_reuses_residual_of_last_computed_step():
    """T = 3 with an infinite threshold: step 0 computed, step 1 skipped, step 2 computed (last).  Rebuild the three
    steps from mmdit.dit_velocity (whose trace gives h_img^L of step 0) and the final layer."""
    s, g, blocks, text, probe, kw = _tiny()
    ts = [1.0, 0.6, 0.3, 0.0]
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h_txt0 = mmdit.text_input(text, g)
    x0 = philox.noise_from_seeds([5], s.n_img * s.latent_ch, 0)[0].reshape(s.n_img, s.latent_ch)
    xT, comp = teacache.denoise_cached(x0, ts, h_txt0, g, blocks, float("inf"), n_heads=s.n_heads, cos=cos, sin=sin)
    assert comp == [True, False, True]
    vel = lambda x, t, tr=None: mmdit.dit_velocity(x, t, h_txt0, g, blocks, n_heads=s.n_heads, cos=cos, sin=sin, trace=tr)
    tr = []
    x1 = x0 + (ts[1] - ts[0]) * vel(x0, ts[0], tr)
    R = tr[-1] - (x0 @ g["img_in_w"].T + g["img_in_b"])               # h_img^L - h_img^0 of step 0
    hL = (x1 @ g["img_in_w"].T + g["img_in_b"]) + R
    _, c = mmdit.time_conditioning(ts[1], g)
    m_f = g["final_mod_w"] @ c + g["final_mod_b"]
    D = hL.shape[1]
    mu, var = hL.mean(-1, keepdims=True), hL.var(-1, keepdims=True)
    y = (hL - mu) / np.sqrt(var + 1e-6) * (1.0 + m_f[:D]) + m_f[D:]
    x2 = x1 + (ts[2] - ts[1]) * (y @ g["proj_w"].T + g["proj_b"])
    x3 = x2 + (ts[3] - ts[2]) * vel(x2, ts[2])
    assert np.abs(xT - x3).max() < 1e-12
    # and it differs from the plain rollout (the skip is not a no-op)
    plain = rollout.euler_denoise(x0, ts, lambda x, t: vel(x, t))
    assert np.abs(xT - plain).max() > 1e-6


def test_identity_blocks_make_skipping_exact():
    s, g, blocks, text, probe, kw = _tiny()
    ident = []
    for bw in blocks:
        b2 = dict(bw)
        for st in ("img", "txt"):
            w, b = bw[f"{st}.mod_w"].copy(), bw[f"{st}.mod_b"].copy()
            D = w.shape[0] // 6
            for gi in (2, 5):                                          # gate1, gate2 rows -> 0
                w[gi * D:(gi + 1) * D] = 0.0
                b[gi * D:(gi + 1) * D] = 0.0
            b2[f"{st}.mod_w"], b2[f"{st}.mod_b"] = w, b
        ident.append(b2)
    ts = list(np.linspace(1.0, 0.0, 6))
    lat_c, _, comp = teacache.explore_cached([0], text, ts, g, ident, probe, float("inf"), **kw)
    lat_p, _ = rollout.explore([0], text, ts, g, ident, probe, **kw)
    assert comp[0].astype(int).tolist() == [1, 0, 0, 0, 1]
    assert np.abs(lat_c - lat_p).max() < 1e-13
