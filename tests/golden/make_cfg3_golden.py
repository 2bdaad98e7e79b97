"""Writes tests/golden/cfg3_seed0.json + cfg3_seed0_latent.npy: the fp64 ORACLE's result for one sampled
seed of config 3 at FULL size (60 blocks, hidden 3072, 1024 + 256 tokens, 10 Euler steps), the launch
configuration bench.py times.  Calls only oracle/ and the input generators in synth/ (CPU); never the CUDA
path.  Cost: ~40 min to generate the 20.4 G weights on 8 cores + ~15 min of fp64 BLAS (186 TFLOP).

    python tests/golden/make_cfg3_golden.py [--blocks L] [--steps T] [--seed S] [--out NAME]
    python tests/golden/make_cfg3_golden.py --config 5 --prompt 7 --seed 229 --out cfg5_p7     (config 5, prompt 7)
    python tests/golden/make_cfg3_golden.py --precision fp8 --out cfg3_seed0_fp8               (FP8 variant, oracle/fp8.py)
    python tests/golden/make_cfg3_golden.py --precision nvfp4 --out cfg3_seed0_nvfp4 --workers 8 (NVFP4 variant, oracle/nvfp4.py)
    python tests/golden/make_cfg3_golden.py --config 4 --seed 0 --out cfg4_seed0 --weight-cache /tmp/spot_weights
    python tests/golden/make_cfg3_golden.py --config 5 --prompt 7 --seeds 224:240 --out cfg5_p7_a --weight-cache /tmp/spot_weights

The GPU test (tests/test_gpu_fullsize.py) regenerates the same weights on the device, checks their
per-block checksums against the ones stored here, runs the 16-seed batch and compares seed S.
"""
import argparse
import json
import os
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import fp8, mmdit, nvfp4, philox, rollout  # noqa: E402
from synth import CONFIGS, make_probe, make_text_emb, tensor_checksum  # noqa: E402
from synth.manifest import make_block_weights, make_global_weights  # noqa: E402


def np64(t):
    return t.to(torch.float64).numpy()


class BlockSource:
    """Blocks of the shared weight manifest as bf16 torch dicts, one at a time.  With --weight-cache DIR each block is
    generated once (synth/ only), stored there with its checksums and memory-mapped afterwards, so that several runs
    of this script (configs 3-5 share the weights) pay the ~40 min of generation once and never hold 40.8 GB each."""

    def __init__(self, shape, cache_dir, keep_in_ram):
        self.s, self.dir, self.keep = shape, cache_dir, keep_in_ram
        self.ram, self.sums = {}, {}
        if cache_dir:
            os.makedirs(cache_dir, exist_ok=True)

    def get(self, b):
        if b in self.ram:
            return self.ram[b]
        bw = None
        if self.dir:
            f, fs = os.path.join(self.dir, f"block{b:02d}.pt"), os.path.join(self.dir, f"block{b:02d}.sums.json")
            if os.path.exists(f) and os.path.exists(fs):
                bw = torch.load(f, mmap=True, weights_only=True)
                self.sums[b] = json.load(open(fs))
        if bw is None:
            bw = make_block_weights(self.s, b)
            self.sums[b] = {k: tensor_checksum(v) for k, v in sorted(bw.items())}
            if self.dir:
                torch.save(bw, f + ".tmp")
                os.replace(f + ".tmp", f)
                json.dump(self.sums[b], open(fs, "w"))
        if self.keep:
            self.ram[b] = bw
        return bw


def nvfp4_prepare_block(bw, cache_dir, b):
    """Reading N1 for one block: fc1 / fc2 quantised with oracle/nvfp4.py and kept DEQUANTISED in bf16 (exact: an E2M1 value
    times an E4M3 scale has a 5-bit significand) with their fp64 channel scales; qkv / out quantised with oracle/fp8.py and
    kept as 1-byte E4M3 tensors.  The bf16 copies of the eight Linears are dropped.  With a cache directory the result is
    stored there (written by --prep-workers processes ahead of the rollout)."""
    f = os.path.join(cache_dir, f"nv_block{b:02d}.pt") if cache_dir else None
    if f and os.path.exists(f):
        small, q = torch.load(f, weights_only=True)
        return small, q
    bw = dict(bw)
    q = {}
    for st in ("img", "txt"):
        for ln in fp8.BLOCK_LINEARS:
            wfull = np64(bw.pop(f"{st}.{ln}_w"))
            if ln in nvfp4.MLP_LINEARS:
                wq, wsf, sc = nvfp4.quantize_weight(wfull)
                q[f"{st}.{ln}"] = (torch.from_numpy(nvfp4.dequantize(wq, wsf)).to(torch.bfloat16), torch.from_numpy(sc))
            else:
                wq, sc = fp8.quantize_weight(wfull)
                q[f"{st}.{ln}"] = (torch.from_numpy(wq).to(torch.float8_e4m3fn), torch.from_numpy(sc))
    small = {k: v.clone() for k, v in bw.items()}
    if f:
        torch.save((small, q), f + ".tmp")
        os.replace(f + ".tmp", f)
    return small, q


def _prep_worker(args):
    config, n_blocks, cache_dir, b = args
    torch.set_num_threads(2)
    s = CONFIGS[config]
    if n_blocks is not None:
        s = s.with_(n_blocks=n_blocks)
    src = BlockSource(s, cache_dir, keep_in_ram=False)
    bw = src.get(b)                                        # generates + stores the bf16 block and its checksums
    nvfp4_prepare_block(bw, cache_dir, b)
    return b


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--blocks", type=int, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--seed", type=int, default=0, help="one seed: the result is stored as [N_img, C] with keys seed / reward")
    ap.add_argument("--seeds", default=None, help="A:B = seeds A..B-1 of the prompt, all in one pass (blocks outermost, "
                    "oracle.mmdit.dit_velocity_multi): stored as [n, N_img, C] with keys seeds / rewards")
    ap.add_argument("--out", default="cfg3_seed0")
    ap.add_argument("--config", type=int, default=3, choices=[3, 4, 5])
    ap.add_argument("--prompt", type=int, default=0)
    ap.add_argument("--precision", default="bf16", choices=["bf16", "fp8", "nvfp4"],
                    help="fp8 / nvfp4: the low-precision exploration variants as oracle/fp8.py / oracle/nvfp4.py state them "
                         "(DESIGN.md sections 13, 13b)")
    ap.add_argument("--workers", type=int, default=1, help="host threads: over the sequences with --seeds (BLAS is then "
                    "limited to one thread per call), else over attention heads / row blocks (oracle.mmdit.set_workers)")
    ap.add_argument("--prep-workers", type=int, default=0, help="nvfp4 with --weight-cache: processes that generate and "
                    "quantise the blocks ahead of the rollout")
    ap.add_argument("--weight-cache", default=None, help="directory (outside the repository) for the generated bf16 blocks")
    a = ap.parse_args()
    s = CONFIGS[a.config]
    if a.blocks is not None:
        s = s.with_(n_blocks=a.blocks)
    if a.steps is not None:
        s = s.with_(n_steps=a.steps)
    multi = a.seeds is not None
    seeds = list(range(*[int(v) for v in a.seeds.split(":")])) if multi else [a.seed]
    here = os.path.dirname(os.path.abspath(__file__))
    t0 = time.time()
    gw = make_global_weights(s)
    lowp = a.precision in ("fp8", "nvfp4")
    src = BlockSource(s, a.weight_cache, keep_in_ram=a.weight_cache is None or lowp)
    qblocks = {}
    if a.precision == "nvfp4" and a.weight_cache and a.prep_workers > 1:
        import multiprocessing as mp
        with mp.get_context("spawn").Pool(a.prep_workers) as pool:
            for b in pool.imap_unordered(_prep_worker, [(a.config, a.blocks, a.weight_cache, b) for b in range(s.n_blocks)]):
                print(f"block {b} prepared ({time.time() - t0:.0f} s)", flush=True)
    if a.weight_cache is None or lowp:
        for b in range(s.n_blocks):
            bw = src.get(b)
            if a.precision == "nvfp4":
                bw, qblocks[b] = nvfp4_prepare_block(bw, a.weight_cache, b)
                src.ram[b] = bw
            if a.precision == "fp8":
                # quantise once with the oracle's quantiser and keep the codes as 1-byte tensors (exact: the values are
                # E4M3-representable); the bf16 copies of the four Linears are dropped (20 GB instead of 40.8 GB)
                bw = dict(bw)
                q = {}
                for st in ("img", "txt"):
                    for ln in fp8.BLOCK_LINEARS:
                        wq, sc = fp8.quantize_weight(np64(bw.pop(f"{st}.{ln}_w")))
                        q[f"{st}.{ln}"] = (torch.from_numpy(wq).to(torch.float8_e4m3fn), sc)
                qblocks[b] = q
                src.ram[b] = bw
            print(f"block {b} generated ({time.time() - t0:.0f} s)", flush=True)
    gsum = {k: tensor_checksum(v) for k, v in sorted(gw.items())}
    text = make_text_emb(s, prompts=[a.prompt])
    probe = make_probe(s)
    ts = [float(np.float32(t)) for t in s.timesteps]
    g = {k: np64(v) for k, v in gw.items()}
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h0 = mmdit.text_input(np64(text)[0], g, s.rms_eps)
    x0 = philox.noise_from_seeds(seeds, s.n_img * s.latent_ch).reshape(len(seeds), s.n_img, s.latent_ch)
    x0 = x0.astype(np.float32).astype(np.float64)          # the CUDA path stores the initial latent in fp32
    t1 = time.time()

    class LazyBlocks:                                      # widen one block at a time to fp64 (2.7 GB transient)
        def __iter__(self):
            for b in range(s.n_blocks):
                yield {k: np64(v) for k, v in src.get(b).items()}
                if b % 10 == 9:
                    print(f"    block {b} ({time.time() - t1:.0f} s)", flush=True)

    hist = []

    def fp8_lin(bi):                                       # the `lin` hook of oracle/fp8.py, codes widened per call
        def lin(x, name):
            wq8, sc = qblocks[bi][name]
            return fp8.linear_fp8(x, wq8.to(torch.float64).numpy(), sc, np64(src.get(bi)[f"{name}_b"]))
        return lin

    def nvfp4_lin(bi):                                     # the `lin` hook of oracle/nvfp4.py (block_lin), weights widened per call
        def lin(x, name):
            ent = qblocks[bi][name]
            bias = np64(src.get(bi)[f"{name}_b"])
            if name.split(".")[1] in nvfp4.MLP_LINEARS:
                return nvfp4.linear_nvfp4_deq(x, ent[0].to(torch.float64).numpy(), ent[1].numpy(), bias)
            return fp8.linear_fp8(x, ent[0].to(torch.float64).numpy(), ent[1].numpy(), bias)
        return lin

    kw = dict(n_heads=s.n_heads, cos=cos, sin=sin, ln_eps=s.ln_eps, rms_eps=s.rms_eps,
              block_lin=fp8_lin if a.precision == "fp8" else nvfp4_lin if a.precision == "nvfp4" else None)

    if a.workers > 1 and not multi:
        mmdit.set_workers(a.workers)

    def vel(x, t):
        if multi and a.workers > 1:
            from threadpoolctl import threadpool_limits
            with threadpool_limits(limits=1, user_api="blas"):
                v = np.stack(mmdit.dit_velocity_multi(list(x), t, [h0] * len(seeds), g, LazyBlocks(), workers=a.workers, **kw))
        elif multi:
            v = np.stack(mmdit.dit_velocity_multi(list(x), t, [h0] * len(seeds), g, LazyBlocks(), **kw))
        else:
            v = mmdit.dit_velocity(x, t, h0, g, LazyBlocks(), **kw)
        print(f"  velocity at t={t:.3f} done ({time.time() - t1:.0f} s)", flush=True)
        return v

    xT = rollout.euler_denoise(x0 if multi else x0[0], ts, vel, hist)
    rewards = [rollout.probe_reward(x, np64(probe)) for x in (xT if multi else [xT])]
    np.save(os.path.join(here, a.out + "_latent.npy"), xT.astype(np.float32))
    l2 = lambda h: [float(np.linalg.norm(r)) for r in h] if multi else float(np.linalg.norm(h))
    meta = {"written_by": "tests/golden/make_cfg3_golden.py (oracle/ + synth/ only)", "config": s.name, "n_blocks": s.n_blocks,
            "n_steps": s.n_steps, "precision": a.precision, "prompt": a.prompt, "timesteps": ts,
            "latent_l2": l2(xT), "x0_l2": l2(x0 if multi else x0[0]), "per_step_l2": [l2(h) for h in hist],
            "global_checksums": gsum, "block_checksums": [src.sums[b] for b in range(s.n_blocks)],
            "text_checksum": tensor_checksum(text),
            "probe_checksum": tensor_checksum(probe), "oracle_seconds": time.time() - t1, "weightgen_seconds": t1 - t0,
            "host_cores": os.cpu_count()}
    if multi:
        meta.update(seeds=seeds, rewards=rewards)
    else:
        meta.update(seed=a.seed, reward=rewards[0],
                    per_step_head=[[float(v) for v in h.reshape(-1)[:16]] for h in hist])
    with open(os.path.join(here, a.out + ".json"), "w") as f:
        json.dump(meta, f, indent=1)
    print("done", rewards, time.time() - t0)


if __name__ == "__main__":
    main()
