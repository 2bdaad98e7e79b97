"""fp64 CPU oracle of the SPOTLIGHT seed-exploration rollout (TEST INFRASTRUCTURE).

This package is the slow, plain, step-by-step statement of what the hot path
computes.  It is test infrastructure: only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import it.  It
imports nothing from `paper_2606_19004_b200/` and shares no code, tables or
constants with the CUDA path.

Paper passages it follows (PAPER.md = /root/reference/PAPER.md):
  * PAPER.md:59  (§2.1) "starts from random Gaussian noise and refines a latent
    representation over a fixed number of denoising steps ... each requiring a
    full forward pass through the DiT backbone"               -> rollout.denoise
  * PAPER.md:61  (§2.1) "K samples from each of P prompts ... K distinct noise
    seeds ... per-sample scalar reward r_k"                    -> philox, rollout
  * PAPER.md:67  (§2.2) "selecting the top and bottom K/2 by reward"
  * PAPER.md:229 (§5) "top-k/bottom-k strategy over per-prompt exploration
    rewards, retaining the highest- and lowest-scoring seeds"  -> rollout.select_seeds
  * PAPER.md:175 (§4.3.2) per-prompt reward standard deviation sigma_g
  * PAPER.md:251 (§6.1) Qwen-Image 20B, deterministic random seed per sample.

The paper is silent on every inner definition (RNG, block, RoPE, sampler);
those are the readings S1-S16 listed in DESIGN.md, which bind this oracle and
the CUDA path equally.

Pins (tests/test_oracle_*.py, run with -m "not gpu"): see DESIGN.md "Oracle pins".
Parity unpinned: faithfulness of the block definition to the released Qwen-Image
checkpoint (weights and reference implementation are not available; the metric
does not need it).
"""
