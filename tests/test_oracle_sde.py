"""Pins for oracle/sde.py (CPU only): the stochastic sampler step (PAPER.md:227 FlowGRPO backbone, Table 2 "SDE window").

What fixes it other than itself:
  * noise level 0 and steps outside the window reduce to the (pinned) Euler sampler exactly;
  * marginal preservation, the property that DEFINES the drift correction: for Gaussian data the exact velocity
    field is linear, and the SDE started from the exact marginal at t = 0.9 must land on the exact marginal at
    t = 0.2 for any noise level (a dropped or mis-signed correction term, or a wrong (1 - t) factor, misses by far
    more than the Monte-Carlo error);
  * the log-probability against scipy.stats.norm.logpdf;
  * the noise of step i is Philox stream 256 + i of the sequence's seed (pinned generator), steps are uncorrelated.
"""
import math

import numpy as np
from scipy import stats

from oracle import philox, rollout, sde


def test_zero_noise_and_outside_window_are_euler():
    rng = np.random.default_rng(3)
    x0 = rng.normal(size=(8, 4))
    A = rng.normal(size=(4, 4)) * 0.3
    vel = lambda x, t: x @ A * (0.5 + t)
    ts = [1.0, 0.8, 0.55, 0.3, 0.0]
    ref = rollout.euler_denoise(x0, ts, vel)
    x_a, lp_a = sde.denoise_sde(x0, 7, ts, vel, 0.0, (0, 4))
    x_b, lp_b = sde.denoise_sde(x0, 7, ts, vel, 0.7, (2, 2))             # empty window
    assert (x_a == ref).all() and (x_b == ref).all()
    assert (lp_a == 0).all() and (lp_b == 0).all()
    x_c, lp_c = sde.denoise_sde(x0, 7, ts, vel, 0.7, (1, 3))
    assert np.abs(x_c - ref).max() > 1e-3 and lp_c[0] == 0 and lp_c[3] == 0 and lp_c[1] != 0 and lp_c[2] != 0


def _gauss_velocity(s2):
    """Exact velocity field E[eps - x0 | x_t] for x0 ~ N(0, s2), eps ~ N(0, 1): linear in x."""
    return lambda x, t: (t - (1.0 - t) * s2) / ((1.0 - t) ** 2 * s2 + t * t) * x


def test_marginals_are_preserved_for_gaussian_data():
    s2 = 0.25
    var = lambda t: (1.0 - t) ** 2 * s2 + t * t
    rng = np.random.default_rng(11)
    n, steps = 400_000, 700
    ts = np.linspace(0.9, 0.2, steps + 1)
    vel = _gauss_velocity(s2)
    for a in (0.4, 1.0):
        x = rng.normal(size=n) * math.sqrt(var(0.9))
        for i in range(steps):
            x, _ = sde.sde_step(x, vel(x, ts[i]), float(ts[i]), float(ts[i + 1]), a, rng.normal(size=n))
        got = x.var()
        assert abs(got / var(0.2) - 1.0) < 0.02, (a, got, var(0.2))         # exact 0.2; MC error ~0.3 %, O(dt) bias < 1 %
    # sensitivity: without the drift correction the same noise inflates the variance far beyond the tolerance
    x = rng.normal(size=n) * math.sqrt(var(0.9))
    for i in range(steps):
        t, tn = float(ts[i]), float(ts[i + 1])
        sig = sde.sde_sigma(t, tn, 1.0)
        x = x + (tn - t) * vel(x, t) + sig * math.sqrt(t - tn) * rng.normal(size=n)
    assert x.var() / var(0.2) > 1.5


def test_log_probability_matches_scipy():
    rng = np.random.default_rng(5)
    x, v, xi = rng.normal(size=(16, 8)), rng.normal(size=(16, 8)), rng.normal(size=(16, 8))
    t, tn, a = 0.7, 0.6, 0.8
    xn, lp = sde.sde_step(x, v, t, tn, a, xi)
    sig = a * math.sqrt(t / (1 - t))
    mean = x * (1 + sig ** 2 / (2 * t) * (tn - t)) + v * (1 + sig ** 2 * (1 - t) / (2 * t)) * (tn - t)
    ref = stats.norm.logpdf(xn, loc=mean, scale=sig * math.sqrt(t - tn)).mean()
    assert abs(lp - ref) < 1e-12
    assert abs(lp - (-(xi ** 2).mean() / 2 - math.log(sig * math.sqrt(t - tn)) - 0.5 * math.log(2 * math.pi))) < 1e-12


def test_sigma_schedule_and_singular_endpoint():
    assert abs(sde.sde_sigma(0.5, 0.4, 0.7) - 0.7) < 1e-15                    # t/(1-t) = 1
    assert abs(sde.sde_sigma(0.8, 0.7, 1.0) - 2.0) < 1e-12                    # sqrt(0.8/0.2)
    # t = 1: FlowGRPO keeps t in the numerator and moves only the denominator to t_next: sqrt(1/0.1), not sqrt(0.9/0.1)
    assert abs(sde.sde_sigma(1.0, 0.9, 1.0) - math.sqrt(10.0)) < 1e-12
    assert sde.sde_sigma(0.3, 0.2, 0.0) == 0.0


def test_step_noise_is_the_pinned_philox_stream():
    xi3 = sde.step_noise(42, 3, (16, 8))
    assert (xi3.reshape(-1) == philox.noise_from_seeds([42], 128, 256 + 3)[0]).all()
    big = [sde.step_noise(9, i, (1 << 16,)) for i in range(3)]
    for a in range(3):
        assert abs(big[a].mean()) < 0.02 and abs(big[a].var() - 1) < 0.02
        for b in range(a + 1, 3):
            assert abs(np.corrcoef(big[a], big[b])[0, 1]) < 0.02
    assert abs(np.corrcoef(big[0], philox.noise_from_seeds([9], 1 << 16, 0)[0])[0, 1]) < 0.02    # and from the initial latent


def test_resumed_rollout_uses_global_step_indices():
    """A rollout split into two calls (in-flight latents are committed on preemption and resumed) must draw
    the noise of GLOBAL step j from stream base + j and test the window on j: split == unsplit exactly."""
    rng = np.random.default_rng(11)
    x0 = rng.normal(size=(8, 4))
    vel = lambda x, t: -0.3 * x + t
    ts = [1.0, 0.8, 0.6, 0.4, 0.2, 0.0]
    full, lp = sde.denoise_sde(x0, 5, ts, vel, 0.6, (1, 4))
    a, lpa = sde.denoise_sde(x0, 5, ts[:3], vel, 0.6, (1, 4))
    b, lpb = sde.denoise_sde(a, 5, ts[2:], vel, 0.6, (1, 4), first_step=2)
    assert (b == full).all() and (np.concatenate([lpa, lpb]) == lp).all()
    wrong, _ = sde.denoise_sde(a, 5, ts[2:], vel, 0.6, (1, 4))                # forgetting the offset reuses streams 256, 257
    assert np.abs(wrong - full).max() > 1e-3
