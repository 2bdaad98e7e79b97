"""-m gpu parity of the cached-step exploration variant (spot_explore_cached / spot_dit_denoise_cached) against
oracle/teacache.py.

The skip decision is an integer decided by floating point: both sides take it on acc = sum poly(rel) with rel in
(at least) fp32-accurate arithmetic; the comparison is made at thresholds the ORACLE's own trace shows to be a safe
margin away from every accumulated value it was compared with (2e-3 relative on the fp32 config, whose rel agrees to
~1e-5; a constant polynomial, i.e. pure arithmetic, on the bf16 config), and the test asserts that margin.  Then: computed flags bit-exact, rel within 1e-3 (fp32) / 3e-2 (bf16 path), final latents and
rewards within the north-star tolerances (1e-4 fp32, 5e-2 bf16).
"""
import numpy as np
import pytest
import torch

import paper_2606_19004_b200 as spot
from oracle import teacache
from synth import CONFIGS, make_probe, make_text_emb
from tests.gpu_common import device_weights, ensure_built, oracle_weights
from tests.helpers import np64, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    ensure_built()


def _seeds(vals):
    return torch.tensor(list(vals), dtype=torch.int64, device="cuda")


def _oracle(s, w, text, probe, seeds, ts, thr, coeffs=(0.0, 1.0)):
    g, blocks = oracle_weights(w)
    f32 = lambda a: a.astype(np.float32).astype(np.float64)
    traces = []
    lat, rew, comp = teacache.explore_cached(list(seeds), np64(text), ts, g, blocks, np64(probe), thr, coeffs, n_heads=s.n_heads,
                                             grid_h=s.grid_h, grid_w=s.grid_w, rope_pairs=s.rope_pairs, rope_theta=s.rope_theta,
                                             ln_eps=s.ln_eps, rms_eps=s.rms_eps, latent_ch=s.latent_ch, x0_cast=f32, traces=traces)
    return lat, rew, comp, traces


def _margin(traces, thr, T):
    """Smallest relative distance between the threshold and any accumulated value it was compared with."""
    m = np.inf
    for tr in traces:
        for i in range(1, T - 1):
            m = min(m, abs(tr["acc"][i] - thr) / thr)
    return m


def _pick_threshold(s, w, text, probe, seeds, ts, candidates, want_ragged, margin=0.02):
    """First candidate whose oracle run mixes computed and skipped steps with a >= `margin` relative decision margin
    (and, if asked, makes at least one step ragged: some seeds compute while others skip)."""
    T = len(ts) - 1
    for thr in candidates:
        lat, rew, comp, traces = _oracle(s, w, text, probe, seeds, ts, thr)
        mid = comp[:, 1:T - 1]
        ragged = bool(((mid.sum(0) > 0) & (mid.sum(0) < comp.shape[0])).any())
        if mid.any() and not mid.all() and _margin(traces, thr, T) >= margin and (ragged or not want_ragged):
            return thr, lat, rew, comp, traces
    return None


@pytest.fixture(scope="module")
def cfg1():
    s = CONFIGS[1]
    w = device_weights(s)
    ctx = spot.Context(s, w, max_seqs=8)
    return s, w, ctx, make_text_emb(s, "cuda"), make_probe(s, "cuda")


def test_threshold_zero_is_bit_identical_to_plain_explore(cfg1):
    s, w, ctx, text, probe = cfg1
    ts = [float(np.float32(t)) for t in np.linspace(1.0, 0.0, 7)]
    K = s.seeds_per_prompt
    plain = spot.spot_explore(ctx, _seeds(s.seeds), text, ts, probe, 1, K, K // 2)
    lat_p, rew_p = plain["latents"].clone(), plain["rewards"].clone()
    cached = spot.spot_explore_cached(ctx, _seeds(s.seeds), text, ts, probe, 1, K, K // 2, threshold=0.0)
    assert cached["computed"].all()
    assert torch.equal(cached["latents"], lat_p) and torch.equal(cached["rewards"], rew_p)


def test_constant_polynomial_pattern(cfg1):
    """poly == 1, threshold 3, T = 10: the hand-worked pattern of tests/test_oracle_teacache.py."""
    s, w, ctx, text, probe = cfg1
    ts = [float(np.float32(t)) for t in np.linspace(1.0, 0.0, 11)]
    out = spot.spot_explore_cached(ctx, _seeds([1, 2]), text, ts, probe, 1, 2, 1, threshold=3.0, coeffs=[1.0])
    for b in range(2):
        assert out["computed"][b].tolist() == [1, 0, 0, 1, 0, 0, 1, 0, 0, 1]
    lat, rew, comp, _ = _oracle(s, w, text[0], probe, [1, 2], ts, 3.0, coeffs=(1.0,))
    assert rel_l2(np64(out["latents"]), lat) < 1e-4 and rel_l2(np64(out["rewards"]), rew) < 1e-4


def test_cfg1_cached_matches_oracle_with_ragged_decisions(cfg1):
    s, w, ctx, text, probe = cfg1
    ts = [float(np.float32(t)) for t in np.linspace(1.0, 0.0, 9)]
    seeds = [0, 1, 2, 3, 4, 5]
    # thresholds that fall BETWEEN the seeds' first rel values split the batch at step 1 (ragged compaction); the
    # fp32 path reproduces rel to ~1e-5, so a 2e-3 margin is safe here
    _, _, _, tr_inf = _oracle(s, w, text[0], probe, seeds, ts, float("inf"))
    first = sorted(tr["rel"][1] for tr in tr_inf)
    cands = [0.5 * (a + b) for a, b in zip(first, first[1:])]
    cands.sort(key=lambda c: -min(abs(c - f) / c for f in first))
    pick = _pick_threshold(s, w, text[0], probe, seeds, ts, cands, want_ragged=True, margin=2e-3)
    assert pick is not None, "no threshold with a safe decision margin that splits the batch"
    thr, lat, rew, comp, traces = pick
    out = spot.spot_explore_cached(ctx, _seeds(seeds), text, ts, probe, 1, len(seeds), 3, threshold=thr)
    print(f"threshold {thr}: effective steps per seed {comp.sum(1).tolist()} of {len(ts) - 1}; step-1 rel {first}")
    mid = comp[:, 1:-1]
    assert ((mid.sum(0) > 0) & (mid.sum(0) < len(seeds))).any()          # at least one ragged step
    assert (out["computed"].numpy().astype(bool) == comp).all()
    rel_ref = np.array([[0.0 if r is None else r for r in tr["rel"]] for tr in traces])
    assert np.abs(out["rel"].numpy() - rel_ref).max() < 1e-3 * max(1.0, rel_ref.max())
    assert rel_l2(np64(out["latents"]), lat) < 1e-4
    assert rel_l2(np64(out["rewards"]), rew) < 1e-4
    # determinism and batch independence: a seed alone takes the same decisions and gives the same bits
    again = spot.spot_explore_cached(ctx, _seeds(seeds), text, ts, probe, 1, len(seeds), 3, threshold=thr)
    assert torch.equal(again["latents"], out["latents"]) and torch.equal(again["computed"], out["computed"])
    alone = spot.spot_explore_cached(ctx, _seeds([seeds[4]]), text, ts, probe, 1, 1, 0, threshold=thr)
    assert torch.equal(alone["computed"][0], out["computed"][4]) and torch.equal(alone["latents"][0], out["latents"][4])


def test_infinite_threshold_computes_first_and_last_only(cfg1):
    s, w, ctx, text, probe = cfg1
    ts = [float(np.float32(t)) for t in np.linspace(1.0, 0.0, 6)]
    out = spot.spot_explore_cached(ctx, _seeds([7, 8]), text, ts, probe, 1, 2, 1, threshold=float("inf"))
    assert out["computed"].tolist() == [[1, 0, 0, 0, 1]] * 2
    lat, rew, comp, _ = _oracle(s, w, text[0], probe, [7, 8], ts, float("inf"))
    assert rel_l2(np64(out["latents"]), lat) < 1e-4


def test_two_prompts_cached(cfg1):
    """The text rows of a compacted sequence must come from ITS prompt (gather with idx / K)."""
    s, w, ctx, _, probe = cfg1
    s2 = s.with_(n_prompts=2)
    text2 = make_text_emb(s2, "cuda")
    ts = [float(np.float32(t)) for t in np.linspace(1.0, 0.0, 7)]
    seeds = [10, 11, 12, 20, 21, 22]
    out = spot.spot_explore_cached(ctx, _seeds(seeds), text2, ts, probe, 2, 3, 1, threshold=3.0, coeffs=[1.0])
    for g in range(2):
        lat, rew, comp, _ = _oracle(s, w, text2[g], probe, seeds[3 * g:3 * g + 3], ts, 3.0, coeffs=(1.0,))
        assert (out["computed"][3 * g:3 * g + 3].numpy().astype(bool) == comp).all()
        assert rel_l2(np64(out["latents"][3 * g:3 * g + 3]), lat) < 1e-4


def test_cached_bf16_full_width_reduced_depth():
    """Config-3 shapes (hidden 3072, 24 x 128 heads, 1024 + 256 tokens) at depth 2, bf16: the tcgen05 path under the
    compaction, against the oracle within the bf16 tolerance."""
    s = CONFIGS[3].with_(n_blocks=2, seeds_per_prompt=3, n_steps=5)
    w = device_weights(s)
    ctx = spot.Context(s, w, max_seqs=3)
    text, probe = make_text_emb(s, "cuda"), make_probe(s, "cuda")
    ts = [float(np.float32(t)) for t in s.timesteps]
    seeds = [0, 1, 2]
    # constant polynomial: the pattern is arithmetic (no dependence on bf16-level differences in rel)
    out = spot.spot_explore_cached(ctx, _seeds(seeds), text, ts, probe, 1, 3, 1, threshold=2.0, coeffs=[1.0])
    assert out["computed"].tolist() == [[1, 0, 1, 0, 1]] * 3
    lat, rew, comp, traces = _oracle(s, w, text[0], probe, seeds[:1], ts, 2.0, coeffs=(1.0,))
    e = rel_l2(np64(out["latents"][0]), lat[0])
    print(f"cached bf16 depth-2: latents rel-L2 {e:.3e}")
    assert e < 5e-2
    rel_ref = np.array([0.0 if r is None else r for r in traces[0]["rel"]])
    assert np.abs(out["rel"][0].numpy() - rel_ref).max() < 3e-2 * max(1.0, rel_ref.max())


def test_cached_argument_errors(cfg1):
    s, w, ctx, text, probe = cfg1
    ts = [1.0, 0.5, 0.0]
    with pytest.raises(spot.SpotError):
        spot.spot_explore_cached(ctx, _seeds([0, 1]), text, ts, probe, 1, 2, 1, threshold=-1.0)
    with pytest.raises(spot.SpotError):
        spot.spot_explore_cached(ctx, _seeds([0, 1]), text, ts, probe, 1, 2, 1, threshold=0.1, coeffs=[0.0] * 9)
