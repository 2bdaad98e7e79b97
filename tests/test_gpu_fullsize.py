"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The fp64 oracle cannot run a 60-block rollout inside a test (186 TFLOP per seed), so:
  * config 3 (and one seed of config 5) are compared with oracle results computed once on the CPU by the
    committed script tests/golden/make_cfg3_golden.py (oracle/ + synth/ only) and stored under tests/golden/;
    the weights regenerated on the device are first proven identical to the ones the oracle used (checksums);
  * properties that hold at any size cover the rest: a seed's result does not depend on the batch it runs in
    (bit-identical), rewards agree with an independent reduction of the returned latents, selection agrees
    with the oracle's selection rule applied to the returned rewards;
  * config-4 / config-5 shapes are additionally compared with the live oracle at reduced depth.
"""
import json
import os

import numpy as np
import pytest
import torch

import paper_2606_19004_b200 as spot
from oracle import rollout
from synth import CONFIGS, make_probe, make_text_emb, make_weights, tensor_checksum
from tests.gpu_common import device_weights, ensure_built, f32_timesteps, oracle_explore
from tests.helpers import np64, rel_l2

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    ensure_built()


def _seeds(vals):
    return torch.tensor(list(vals), dtype=torch.int64, device="cuda")


def _load_golden(name):
    path = os.path.join(GOLDEN, name + ".json")
    if not os.path.exists(path):
        pytest.skip(f"{name}.json not present (written by tests/golden/make_cfg3_golden.py)")
    meta = json.load(open(path))
    lat = np.load(os.path.join(GOLDEN, name + "_latent.npy")).astype(np.float64)
    return meta, lat


@pytest.fixture(scope="module")
def full_model():
    """The 60-block, 40.8 GB weight set of configs 3-5, generated on the device."""
    s = CONFIGS[3]
    w = make_weights(s, device="cuda")
    torch.cuda.synchronize()
    return s, w


def _check_weights(meta, w, text, probe):
    assert {k: tensor_checksum(v) for k, v in sorted(w["global"].items())} == meta["global_checksums"]
    for b, want in enumerate(meta["block_checksums"]):
        got = {k: tensor_checksum(v) for k, v in sorted(w["blocks"][b].items())}
        assert got == want, f"block {b}: device-generated weights differ from the oracle's"
    assert tensor_checksum(text) == meta["text_checksum"] and tensor_checksum(probe) == meta["probe_checksum"]


def test_cfg3_full_size_against_golden(full_model):
    s, w = full_model
    meta, lat_ref = _load_golden("cfg3_seed0")
    assert meta["n_blocks"] == s.n_blocks and meta["n_steps"] == s.n_steps
    text, probe = make_text_emb(s, "cuda"), make_probe(s, "cuda")
    _check_weights(meta, w, text, probe)
    ctx = spot.Context(s, w, max_seqs=s.n_seqs)
    ts = f32_timesteps(s)
    assert ts == meta["timesteps"]
    K = s.seeds_per_prompt
    out = spot.spot_explore(ctx, _seeds(s.seeds), text, ts, probe, 1, K, K // 2)      # bench.py's launch configuration
    torch.cuda.synchronize()
    i = list(s.seeds).index(meta["seed"])
    e_lat = rel_l2(np64(out["latents"][i]), lat_ref)
    e_rew = abs(out["rewards"][i].item() - meta["reward"]) / max(abs(meta["reward"]), 1e-30)
    print(f"cfg3 full size, seed {meta['seed']}: latents rel-L2 {e_lat:.3e}, reward rel err {e_rew:.3e} "
          f"(reward {out['rewards'][i].item():.6f} vs oracle {meta['reward']:.6f})")
    assert e_lat < 5e-2
    assert abs(out["rewards"][i].item() - meta["reward"]) < 5e-2 * max(np.abs(np64(out["rewards"])).max(), 1e-30)
    # properties at full size --------------------------------------------------------------------------------
    lat = np64(out["latents"])
    rew = np64(out["rewards"])
    ref_rew = np.array([rollout.probe_reward(lat[b], np64(probe)) for b in range(K)])       # independent reduction
    assert np.abs(rew - ref_rew).max() < 1e-5 * max(1.0, np.abs(ref_rew).max())
    sel = rollout.select_seeds(out["rewards"].cpu().numpy()[None, :].astype(np.float64), K // 2)
    assert out["top"].cpu().tolist() == sel["top"].tolist() and out["bottom"].cpu().tolist() == sel["bottom"].tolist()
    assert abs(out["stats"][0, 1].item() - sel["std"][0]) < 1e-5 * max(1.0, sel["std"][0])
    assert np.isfinite(lat).all() and np.std(rew) > 0
    # seed independence: the sampled seed alone gives the same bits as inside the 16-seed batch
    alone = spot.spot_explore(ctx, _seeds([meta["seed"]]), text, ts, probe, 1, 1, 0)
    assert torch.equal(alone["latents"][0], out["latents"][i]) and torch.equal(alone["rewards"][0], out["rewards"][i])
    # so every other seed of the batch is covered by the same code path that the golden seed verified


def test_cfg3_full_size_fp8_against_golden(full_model):
    """The FP8 (E4M3) exploration variant at config 3's full size against oracle/fp8.py's result for one seed
    (tests/golden/cfg3_seed0_fp8*, written by make_cfg3_golden.py --precision fp8).  Over 600 block evaluations a few
    percent of the activation codes land on the neighbouring E4M3 value (the value being rounded differs at the bf16
    level between the two sides), so the bound is the north-star's 5e-2 on the latents and on the reward relative to the
    reward scale of the batch - the quantity the variant exists for is the ranking, checked against bf16 below."""
    s, w = full_model
    meta, lat_ref = _load_golden("cfg3_seed0_fp8")
    assert meta["precision"] == "fp8" and meta["n_blocks"] == s.n_blocks and meta["n_steps"] == s.n_steps
    text, probe = make_text_emb(s, "cuda"), make_probe(s, "cuda")
    _check_weights(meta, w, text, probe)
    ctx = spot.Context(s, w, max_seqs=s.n_seqs)
    ts = f32_timesteps(s)
    K = s.seeds_per_prompt
    bf = spot.spot_explore(ctx, _seeds(s.seeds), text, ts, probe, 1, K, K // 2)
    rew_bf = np64(bf["rewards"]).copy()
    ctx.enable_fp8(True)
    try:
        out = spot.spot_explore(ctx, _seeds(s.seeds), text, ts, probe, 1, K, K // 2)
        torch.cuda.synchronize()
    finally:
        ctx.enable_fp8(False)
    i = list(s.seeds).index(meta["seed"])
    e_lat = rel_l2(np64(out["latents"][i]), lat_ref)
    rew = np64(out["rewards"])
    scale = max(np.abs(rew).max(), 1e-30)
    e_rew = abs(rew[i] - meta["reward"]) / scale
    rank = lambda a: np.argsort(np.argsort(a))
    rho = np.corrcoef(rank(rew), rank(rew_bf))[0, 1]
    print(f"cfg3 full size FP8, seed {meta['seed']}: latents rel-L2 vs fp8 oracle {e_lat:.3e}, reward {rew[i]:.6f} vs oracle "
          f"{meta['reward']:.6f} ({e_rew:.3e} of the batch's reward scale); Spearman with the bf16 rollout {rho:.3f}")
    assert e_lat < 5e-2
    assert e_rew < 5e-2
    assert rho >= 0.8                                              # PAPER.md:340 rank-fidelity criterion


def test_cfg5_prompt_independence_and_golden(full_model):
    """Config 5 (8 prompts x 32 seeds): a prompt group inside the 256-sequence batch is bit-identical to the same
    group run alone; one seed of prompt 7 is compared with the stored oracle result when present."""
    s3, w = full_model
    s = CONFIGS[5]
    text, probe = make_text_emb(s, "cuda"), make_probe(s, "cuda")
    ctx = spot.Context(s, w, max_seqs=s.n_seqs)
    ts = f32_timesteps(s)
    P, K = s.n_prompts, s.seeds_per_prompt
    out = spot.spot_explore(ctx, _seeds(s.seeds), text, ts, probe, P, K, K // 2)
    torch.cuda.synchronize()
    rew = out["rewards"].cpu().numpy().astype(np.float64).reshape(P, K)
    sel = rollout.select_seeds(rew, K // 2)
    assert out["top"].cpu().tolist() == sel["top"].tolist() and out["bottom"].cpu().tolist() == sel["bottom"].tolist()
    assert np.abs(out["stats"].cpu().numpy()[:, 1] - sel["std"]).max() < 1e-5
    g = 7
    alone = spot.spot_explore(ctx, _seeds(s.seeds[g * K:(g + 1) * K]), text[g:g + 1].contiguous(), ts, probe, 1, K, K // 2)
    assert torch.equal(alone["rewards"], out["rewards"][g * K:(g + 1) * K])
    assert torch.equal(alone["latents"], out["latents"][g * K:(g + 1) * K])
    assert torch.equal(alone["top"], out["top"][g:g + 1]) and torch.equal(alone["stats"], out["stats"][g:g + 1])
    path = os.path.join(GOLDEN, "cfg5_p7.json")
    if os.path.exists(path):
        meta = json.load(open(path))
        lat_ref = np.load(os.path.join(GOLDEN, "cfg5_p7_latent.npy")).astype(np.float64)
        i = list(s.seeds).index(meta["seed"])
        e_lat = rel_l2(np64(out["latents"][i]), lat_ref)
        print(f"cfg5 full size, seed {meta['seed']}: latents rel-L2 {e_lat:.3e}, reward {out['rewards'][i].item():.6f} vs {meta['reward']:.6f}")
        assert e_lat < 5e-2
        assert abs(out["rewards"][i].item() - meta["reward"]) < 5e-2 * np.abs(rew).max()


def test_cfg4_shape_reduced_depth_against_live_oracle():
    """Config-4 shapes (80x80 grid -> 6400 image tokens, S = 6656, 52 key tiles) at L = 1, K = 1, T = 2."""
    s = CONFIGS[4].with_(n_blocks=1, seeds_per_prompt=1, n_steps=2, seeds=(1,))
    w = device_weights(s)
    ctx = spot.Context(s, w, max_seqs=2)
    text, probe = make_text_emb(s, "cuda"), make_probe(s, "cuda")
    ts = f32_timesteps(s)
    out = spot.spot_explore(ctx, _seeds(s.seeds), text, ts, probe, 1, 1, 0)
    lat, rew = oracle_explore(s, w, text[0], probe, s.seeds, ts)
    e_lat, e_rew = rel_l2(np64(out["latents"]), lat), rel_l2(np64(out["rewards"]), rew)
    print(f"cfg4 shape (L=1,T=2): latents rel-L2 {e_lat:.3e} rewards {e_rew:.3e}")
    assert e_lat < 5e-2 and e_rew < 5e-2
    both = spot.spot_explore(ctx, _seeds([9, 1]), text, ts, probe, 1, 2, 1)
    assert torch.equal(both["latents"][1], out["latents"][0])
