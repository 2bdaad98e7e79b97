#!/usr/bin/env python
"""bench.py - seed-exploration rollout throughput on B200 (contract: see DESIGN.md "Measurement").

A "step" is ONE whole pass of the hot path over one batch: seeds -> Philox/Box-Muller latents -> T Euler steps
of the 60-block MMDiT -> probe rewards -> top/bottom-k selection (spot_explore).  Default workload = config 3
of BASELINE.json (512x512, 60 blocks, 1 prompt x 16 seeds, 10 Euler steps, bf16), the configuration the
metric's ">= 50 % of dense BF16 peak" target is quoted on.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3|cfg4|cfg5] [--scaling weak|strong]
                    [--impl reference] [--dry-run]

N > 1 runs one rank per GPU over NCCL.  Either the caller starts the ranks (python -m torch.distributed.run
--nproc-per-node N ... bench.py --gpus N: WORLD_SIZE must then equal --gpus) or, when WORLD_SIZE is not set,
bench.py re-executes itself under torch.distributed.run with N ranks on 127.0.0.1.  It refuses to run when fewer
than N CUDA devices are visible, and prints n_gpus = the number of ranks that actually joined the process group.
  --scaling weak   (default) replicated weights, every rank explores its own P x K batch with disjoint seeds;
  --scaling strong ONE P x K batch, sequence b on rank floor(b N / B) (sharding.explore_sharded).
Both have no data-path collective; the fp32 rewards are all-gathered once per step.
  --dry-run        host logic only (gloo, a stub step, no GPU, no library): the launcher / sharding / timing /
                   JSON plumbing of the N > 1 path, used by the -m "not gpu" tests.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from synth import CONFIGS, make_probe, make_text_emb, make_weights  # noqa: E402

METRIC = "image-tokens*steps/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch of gemm_tcgen05_v3_kernel, averaged over its four uses in a
# block, from one `ncu --set full` capture per workload (profiles/r2_ncu_full_gemm.txt, commands in profiles/r2_ncu.md):
#   cfg3 (16 seqs): QKV+RoPE 0.939, out-proj 0.623, fc1 1.273, fc2 2.488 GB;  cfg4 (4 x 6656 tokens): 1.229, 0.823, 1.608, 3.570 GB;
#   cfg5 (a chunk of 32 seqs): 2.036, 1.250, 2.837, 6.162 GB
GEMM_DRAM_TRAFFIC_PER_LAUNCH = {"cfg3": 1.331e9, "cfg4": 1.807e9, "cfg5": 3.071e9}
WORKLOADS = {"cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.rows, self.proc = gpu_index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.idx), "-lms", "200"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons, power = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); power.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7), ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons), "samples": len(sm)}


SAMPLE_SEEDS = 3          # oracle sample: this many seeds x 1 Euler step x SAMPLE_BLOCKS of the L blocks (about 10 s on 16 cores)
SAMPLE_BLOCKS = 2


def oracle_sample(shape, w_host, text_host, n_blocks_sample: int, n_seeds: int = SAMPLE_SEEDS):
    """The oracle as it stands on a bounded sample: `n_seeds` seeds, 1 Euler step, `n_blocks_sample` of the L blocks
    at full width (work is exactly linear in seeds, steps and blocks).  Returns seconds."""
    from oracle import mmdit, philox
    from tests.helpers import np64
    g = {k: np64(v) for k, v in w_host["global"].items()}
    blocks = [{k: np64(v) for k, v in b.items()} for b in w_host["blocks"][:n_blocks_sample]]
    te = np64(text_host)[0]
    t0 = time.perf_counter()
    cos, sin = mmdit.rope_table(shape.grid_h, shape.grid_w, shape.n_txt, shape.rope_pairs, shape.rope_theta)
    h0 = mmdit.text_input(te, g)
    for seed in range(n_seeds):
        x0 = philox.noise_from_seeds([seed], shape.n_img * shape.latent_ch)[0].reshape(shape.n_img, shape.latent_ch)
        v = mmdit.dit_velocity(x0, 1.0, h0, g, blocks, n_heads=shape.n_heads, cos=cos, sin=sin)
        _ = x0 + (-0.1) * v
    return time.perf_counter() - t0


def cpu_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        n = [i["num_threads"] for i in threadpool_info() if i.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count() or 1


def workload_config(shape) -> dict:
    """The keys of `config` that name the workload; both arms print them."""
    return {"workload": shape.name, "n_prompts": shape.n_prompts, "seeds_per_prompt": shape.seeds_per_prompt,
            "euler_steps": shape.n_steps, "blocks": shape.n_blocks, "hidden": shape.hidden,
            "image_tokens": shape.n_img, "text_tokens": shape.n_txt}


def run_reference(args, shape):
    """--impl reference: the fp64 oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    nb = SAMPLE_BLOCKS
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    w = make_weights(shape, device=dev, blocks=range(nb))
    w_host = {"global": {k: v.cpu() for k, v in w["global"].items()}, "blocks": [{k: v.cpu() for k, v in b.items()} for b in w["blocks"]]}
    text = make_text_emb(shape, dev, prompts=[0]).cpu()
    del w
    times = []
    for i in range(args.warmup + args.steps):
        dt = oracle_sample(shape, w_host, text, nb)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    value = SAMPLE_SEEDS * shape.n_img * (nb / shape.n_blocks) / (ms / 1e3)
    cores = cpu_threads()
    sample = (f"{SAMPLE_SEEDS} seeds x 1 Euler step x {nb} of {shape.n_blocks} blocks at full width per step "
              "(work is linear in seeds, steps, blocks)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {**workload_config(shape), "sample": sample},
            "cpu_baseline": {"value": value, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_kernels(args, shape):
    """--kernels: each kernel of the path alone at the workload's shapes, L2 flushed between iterations, one
    CUDA-event pair per launch; prints one JSON line with achieved GB/s (HBM-bound kernels, algorithmic bytes of
    DESIGN.md section 5) or TFLOP/s (tensor-bound kernels) against the measured burst peaks."""
    import paper_2606_19004_b200 as spot
    from paper_2606_19004_b200 import build as spot_build
    from synth import hash_normal
    spot_build.build()
    spot.load_library()
    peaks = load_peaks()
    torch.cuda.set_device(0)
    B, S, D, F, H, dh = shape.n_seqs, shape.seq, shape.hidden, shape.mlp_hidden, shape.n_heads, shape.head_dim
    M = B * S
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    flush_words = flush.view(torch.int32)
    bf = torch.bfloat16

    def rnd(tid, shp, dtype, scale=1.0):
        n = int(np.prod(shp))
        return hash_normal(900 + tid, n, scale, dtype, "cuda").reshape(shp)

    def timed(fn, iters):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(iters):
            flush.zero_()                     # 512 MiB written: nothing of the kernel's operands is left in L2 ...
            if args.flush == "clean":
                flush_words.sum()             # ... then read back, so that L2 holds CLEAN lines: otherwise the write-back of
            # up to 126 MB of dirty flush lines lands inside the timed kernel (10 us of a 60 us kernel, none of it its own)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return statistics.median(ts)

    res = {}

    def hbm(name, fn, nbytes, iters=10):
        ms = timed(fn, iters)
        gbs = nbytes / ms / 1e6
        res[name] = {"bound": "hbm", "ms": ms, "algorithmic_bytes": nbytes, "achieved": gbs, "unit": "GB/s",
                     "peak": peaks["hbm_gbs"], "frac": gbs / peaks["hbm_gbs"]}

    def tensor(name, fn, flops, iters=10):
        ms = timed(fn, iters)
        tf = flops / ms / 1e9
        res[name] = {"bound": "tensor", "ms": ms, "flops": flops, "achieved": tf, "unit": "TFLOP/s",
                     "peak": peaks["bf16_tflops"], "frac": tf / peaks["bf16_tflops"]}

    # K1 Philox + Box-Muller: 2^28 normals (16 seeds x 2^24).  ALU-bound, not HBM-bound: 226 SASS instructions per
    # Philox block of 4 normals (10 rounds of 2 IMAD.WIDE + LOP3/IADD, then logf / sqrtf / sincospif per pair), so the
    # roof is 148 SMs x 128 lanes x sm_max clock / 56.5 instructions per normal (K1)
    seeds = torch.arange(16, dtype=torch.int64, device="cuda")
    nz = torch.empty((16, 1 << 24), dtype=torch.float32, device="cuda")
    ms = timed(lambda: spot.spot_noise_from_seeds(seeds, 1 << 24, 0, nz), 10)
    n_norm = 16.0 * (1 << 24)
    alu_peak = 148 * 128 * 1.965e9 / 56.5 / 1e9                       # G normals/s
    res["K1_noise"] = {"bound": "alu", "ms": ms, "normals": n_norm, "achieved": n_norm / ms / 1e6, "unit": "Gnormal/s",
                       "peak": alu_peak, "frac": n_norm / ms / 1e6 / alu_peak, "written_gbs": 4.0 * n_norm / ms / 1e6,
                       "frac_of_hbm_peak": 4.0 * n_norm / ms / 1e6 / peaks["hbm_gbs"],
                       "peak_kind": "derived, and generous: 148 SMs x 128 lanes x 1.965 GHz / 56.5 SASS instructions per normal counts the "
                                    "MUFU-rate instructions (lg2, sqrt, sin, cos: 16 per clock and SM) at the full issue rate; against the "
                                    "HBM write roof the kernel is at frac_of_hbm_peak.  It runs once per rollout (4 MB at config 3: ~0 % of a step)"}
    del nz
    # K3 LN + modulate: fp32 residual rows in, bf16 out
    h = rnd(1, (M, D), torch.float32)
    sh, sc = rnd(2, (D,), torch.float32, 0.1), rnd(3, (D,), torch.float32, 0.1)
    hbm("K3_ln_modulate", lambda: spot.spot_ln_modulate(h, sh, sc, 1e-6, bf), M * D * (4.0 + 2.0))
    # K4 QK-RMSNorm + RoPE in place on q and k
    qkv = rnd(4, (B, S, 3, H, dh), bf)
    gains = [torch.ones(dh, dtype=bf, device="cuda") for _ in range(4)]
    ang = rnd(5, (S, dh // 2), torch.float32, 3.0)             # a rotation table (cos, sin of arbitrary angles): norm-preserving
    cs, sn = torch.cos(ang).contiguous(), torch.sin(ang).contiguous()
    hbm("K4_qk_norm_rope", lambda: spot.spot_qk_norm_rope(qkv, shape.n_txt, gains, cs, sn, 1e-6), 2.0 * 2 * B * S * H * dh * 2)
    # K5 attention
    tensor("K5_attention", lambda: spot.spot_attention(qkv, spot.IMPL_TCGEN05), 4.0 * S * S * dh * H * B)
    qkv_attn = qkv
    tensor("K5_attention_prev_two_pass", lambda: spot.spot_attention(qkv, spot.IMPL_TCGEN05_2CTA), 4.0 * S * S * dh * H * B)
    del qkv
    # K6 Euler update (+ reward): 2^26 elements so that the working set exceeds L2
    Bx, E = 1024, shape.n_img * shape.latent_ch if shape.n_img * shape.latent_ch <= 65536 else 65536
    x, v, pr = rnd(7, (Bx, E), torch.float32), rnd(8, (Bx, E), torch.float32), rnd(9, (E,), torch.float32)
    hbm("K6_euler_update", lambda: spot.spot_euler_update(x, v, -0.1), 12.0 * Bx * E)
    hbm("K6_euler_update_reward", lambda: spot.spot_euler_update(x, v, -0.1, pr), 12.0 * Bx * E + 4.0 * E)
    del x, v
    # K2 the four GEMMs of a block (image + text rows together, one weight set)
    for name, (N, K, epi) in {"K2_gemm_qkv": (3 * D, D, spot.EPI_BIAS), "K2_gemm_out": (D, D, spot.EPI_GATE_RESIDUAL),
                              "K2_gemm_fc1": (F, D, spot.EPI_BIAS_GELU), "K2_gemm_fc2": (D, F, spot.EPI_GATE_RESIDUAL)}.items():
        a, w, b = rnd(10, (M, K), bf), rnd(11, (N, K), bf, 0.02), rnd(12, (N,), bf, 0.02)
        gate, resid = rnd(13, (N,), torch.float32, 0.1), torch.zeros((M, N), dtype=torch.float32, device="cuda")
        out = torch.empty((M, N), dtype=bf, device="cuda")
        tensor(name, lambda: spot.spot_linear(a, w, b, epi, spot.IMPL_AUTO, gate=gate, residual=resid, out=out), 2.0 * M * N * K)
        del a, w, out, resid
    # K2 + K4 fused: the QKV projection whose epilogue applies QK-RMSNorm + RoPE (what the rollout launches)
    a, w, b = rnd(10, (B, S, D), bf), rnd(11, (3 * D, D), bf, 0.02), rnd(12, (3 * D,), bf, 0.02)
    tensor("K2_gemm_qkv_rope_fused", lambda: spot.spot_qkv_rope_linear(a, w, b, gains[0], gains[1], cs, sn, 0, 1e-6),
           2.0 * M * 3 * D * D)
    del a, w
    # K2 on E4M3 operands (the low-precision exploration variant); peak = measured bf16 burst x 2
    for name, (N, K, epi) in {"K2_fp8_gemm_out": (D, D, spot.EPI_GATE_RESIDUAL), "K2_fp8_gemm_fc1": (F, D, spot.EPI_BIAS_GELU),
                              "K2_fp8_gemm_fc2": (D, F, spot.EPI_GATE_RESIDUAL)}.items():
        a8 = spot.spot_quantize_e4m3(rnd(10, (M, K), bf))
        wq, ws = spot.spot_quantize_weight_rows(rnd(11, (N, K), bf, 0.02))
        b = rnd(12, (N,), bf, 0.02)
        gate, resid = rnd(13, (N,), torch.float32, 0.1), torch.zeros((M, N), dtype=torch.float32, device="cuda")
        tensor(name, lambda: spot.spot_linear_fp8(a8, wq, ws, b, epi, gate=gate, residual=resid), 2.0 * M * N * K)
        res[name]["peak"] = 2.0 * peaks["bf16_tflops"]
        res[name]["frac"] = res[name]["achieved"] / res[name]["peak"]
        del a8, wq, resid
    a8 = spot.spot_quantize_e4m3(rnd(10, (B, S, D), bf))
    wq, ws = spot.spot_quantize_weight_rows(rnd(11, (3 * D, D), bf, 0.02))
    b = rnd(12, (3 * D,), bf, 0.02)
    name = "K2_fp8_gemm_qkv_rope_fused"
    tensor(name, lambda: spot.spot_qkv_rope_linear_fp8(a8, wq, ws, b, gains[0], gains[1], cs, sn, 0, 1e-6), 2.0 * M * 3 * D * D)
    res[name]["peak"] = 2.0 * peaks["bf16_tflops"]
    res[name]["frac"] = res[name]["achieved"] / res[name]["peak"]
    del a8, wq
    # NVFP4 exploration variant: block-scaled 4-bit GEMMs of the MLP and the activation quantiser;
    # peak = measured bf16 burst x 4 (nominal fp4 : bf16 ratio)
    for name, (N, K, epi) in {"K2_nvfp4_gemm_fc1": (F, D, spot.EPI_BIAS_GELU), "K2_nvfp4_gemm_fc2": (D, F, spot.EPI_GATE_RESIDUAL)}.items():
        if M % 128 or N % 256 or K % 256:
            continue
        act = rnd(10, (M, K), bf)
        ac, asf = spot.spot_nvfp4_quantize(act)
        wc, wsf, wsc = spot.spot_nvfp4_quantize_weight(rnd(11, (N, K), bf, 0.02))
        b = rnd(12, (N,), bf, 0.02)
        gate, resid = rnd(13, (N,), torch.float32, 0.1), torch.zeros((M, N), dtype=torch.float32, device="cuda")
        tensor(name, lambda: spot.spot_linear_nvfp4(ac, asf, wc, wsf, wsc, b, epi, gate=gate, residual=resid), 2.0 * M * N * K)
        res[name]["peak"] = 4.0 * peaks["bf16_tflops"]
        res[name]["frac"] = res[name]["achieved"] / res[name]["peak"]
        cb, sb = torch.empty_like(ac), torch.empty_like(asf)
        lib = spot.load_library()
        hbm("K12_nvfp4_quantize_K%d" % K, lambda: lib.spot_nvfp4_quantize(act.data_ptr(), M, K, None, cb.data_ptr(), sb.data_ptr(),
                                                                         torch.cuda.current_stream().cuda_stream), M * K * (2.0 + 0.5 + 1.0 / 16))
        del act, ac, asf, wc, wsf, resid, cb, sb
    # K5 sustained, measured last so that its heat does not colour the other rows: the same launch repeated back to back
    # for about 1.5 s (no flush: 377 MB of q, k, v per launch > L2), one event pair around all of them: the rate under
    # the power cap, against the SUSTAINED bf16 peak
    n_rep = 4000
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n_rep):
        spot.spot_attention(qkv_attn, spot.IMPL_TCGEN05)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n_rep
    fl = 4.0 * S * S * dh * H * B
    res["K5_attention_sustained"] = {"bound": "tensor", "ms": ms, "flops": fl, "achieved": fl / ms / 1e9, "unit": "TFLOP/s",
                                     "peak": peaks["bf16_tflops_sustained"], "frac": fl / ms / 1e9 / peaks["bf16_tflops_sustained"],
                                     "peak_kind": f"measured sustained bf16; {n_rep} launches back to back"}
    print(json.dumps({"mode": "kernels", "workload": shape.name, "rows": M, "l2": "512 MiB written" + (", then read back (clean lines)," if args.flush == "clean" else "") + " between iterations",
                      "peaks": peaks, "kernels": res}))


def free_port() -> int:
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        return so.getsockname()[1]


def ensure_ranks(args) -> int:
    """Makes `--gpus N` mean N ranks.  Returns the world size of THIS process (after a re-exec under
    torch.distributed.run when the caller did not start the ranks); exits loudly on any mismatch."""
    env_world = os.environ.get("WORLD_SIZE")
    if args.gpus < 1:
        sys.exit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":                 # the oracle arm: rank 0 alone works, the other ranks (if any) exit 0
        return int(env_world or "1")
    if not args.dry_run and args.impl != "reference":
        have = torch.cuda.device_count()
        if have < args.gpus:
            sys.exit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) are visible: refusing to print a "
                     f"line for fewer GPUs than asked for")
    if env_world is None and args.gpus > 1:
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__), *sys.argv[1:]]
        print("bench.py: starting", args.gpus, "ranks:", " ".join(cmd), file=sys.stderr, flush=True)
        sys.exit(subprocess.call(cmd))
    world = int(env_world or "1")
    if world != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: start the ranks with --nproc-per-node {args.gpus} "
                 f"(or leave WORLD_SIZE unset and bench.py starts them itself)")
    return world


def parallelism_label(scaling: str, world: int, B: int) -> str:
    if scaling == "strong":
        return f"dp{world} strong: one batch of {B} sequences, sequence b on rank floor(b*{world}/{B}), weights replicated"
    return f"dp{world} weak: replicated weights, {B} sequences per rank with disjoint seeds"


def job_seeds(shape, scaling: str, rank: int, world: int):
    """Seeds of this rank.  weak: the job explores world * B sequences, rank r owns [r*B, (r+1)*B); strong: the B seeds of
    the config, all ranks hold all of them (explore_sharded slices)."""
    from paper_2606_19004_b200 import sharding
    B = shape.n_seqs
    if scaling == "strong":
        return [int(v) for v in shape.seeds]
    lo, hi = sharding.shard_range(world * B, rank, world)
    assert hi - lo == B
    return [int(shape.seeds[i % B]) + (i // B) * B for i in range(lo, hi)]


def run_dry(args, shape, world):
    """--dry-run: the N > 1 host logic with a stub step on CPU (gloo)."""
    import torch.distributed as dist
    from paper_2606_19004_b200 import sharding
    rank = int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    joined = torch.ones(1)
    if world > 1:
        dist.all_reduce(joined)
    B, T = shape.n_seqs, shape.n_steps
    seeds = job_seeds(shape, args.scaling, rank, world)
    n_job = B if args.scaling == "strong" else world * B
    lo, hi = sharding.shard_range(B, rank, world) if args.scaling == "strong" else (0, B)
    full = None

    def step():
        nonlocal full
        time.sleep(0.002 * (hi - lo))                                   # the stub: "compute" this rank's sequences
        local = torch.tensor([((s * 2654435761) % 1000) / 1000.0 for s in seeds[lo:hi]], dtype=torch.float32)
        full = sharding.gather_rewards(local, n_job) if world > 1 else local

    for _ in range(args.warmup):
        step()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    ms = sharding.max_over_ranks((time.perf_counter() - t0) * 1e3) / args.steps
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": n_job * shape.n_img * T / (ms / 1e3), "unit": METRIC, "dry_run": True,
                          "n_gpus": int(joined.item()), "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
                          "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "stub", "data": "synthetic",
                          "config": {**workload_config(shape), "parallelism": parallelism_label(args.scaling, world, B)},
                          "rewards_gathered": int(full.numel()), "gpu_launches": 0}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_block(args, shape):
    """--workload cfg2 (BASELINE.json configs[1]; BASELINE.md section 3 "report TFLOP/s"): north-star call (2),
    spot_dit_block_forward, on ONE full-width joint block with B = 8 sequences.  A step = one block evaluation; the
    block's weights (0.68 GB) and intermediates (qkv 189 MB, MLP hidden 252 MB, fp32-free bf16 I/O 126 MB) exceed L2, and
    512 MiB are written and read back between timed iterations anyway (config.l2)."""
    import paper_2606_19004_b200 as spot
    from paper_2606_19004_b200 import build as spot_build
    from synth.manifest import make_block_inputs
    assert int(os.environ.get("WORLD_SIZE", "1")) == 1, "cfg2 is a single-GPU line"
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the product path has no CPU fallback"
    torch.cuda.set_device(0)
    spot_build.build()
    spot.load_library()
    peaks = load_peaks()
    B = shape.n_seqs
    w = make_weights(shape, device="cuda", blocks=[0])
    ctx = spot.Context(shape, w, max_seqs=B)
    h_img, h_txt, temb = make_block_inputs(shape, B, "cuda")
    o_img, o_txt = torch.empty_like(h_img), torch.empty_like(h_txt)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    S, D, F = shape.seq, shape.hidden, shape.mlp_hidden
    flops = B * (2.0 * S * D * (3 * D + D + 2 * F) + 4.0 * S * S * D)
    gemm_flops = B * 2.0 * S * D * (3 * D + D + 2 * F)

    def step():
        spot.spot_dit_block_forward(ctx, 0, h_img, h_txt, temb, o_img, o_txt)

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    spot.spot_get_counters(ctx, reset=True)
    spot.spot_set_option(ctx, spot.OPT_TIMING, 1)
    sampler = ClockSampler(0)
    sampler.start()
    ts = []
    for _ in range(args.steps):
        flush.zero_()
        flush.view(torch.int32).sum()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    counters = spot.spot_get_counters(ctx, reset=True)
    spot.spot_set_option(ctx, spot.OPT_TIMING, 0)
    # sustained: the same call back to back for about a second (what a rollout sees), one event pair
    n_rep = 300
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n_rep):
        step()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms_sus = e0.elapsed_time(e1) / n_rep
    ms = statistics.median(ts)
    # e2e: pinned host buffers -> device, the call, outputs -> pinned host, all inside the timed region
    hp = [t.cpu().pin_memory() for t in (h_img, h_txt, temb)]
    ho = [torch.empty_like(t, device="cpu").pin_memory() for t in (o_img, o_txt)]

    def e2e_step():
        for dst, src in zip((h_img, h_txt, temb), hp):
            dst.copy_(src, non_blocking=True)
        step()
        for dst, src in zip(ho, (o_img, o_txt)):
            dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()

    e2e_step()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    e_ms = (time.perf_counter() - w0) * 1e3 / args.steps
    units = B * shape.n_img
    tf = flops / ms / 1e9
    gemm_tf = gemm_flops * counters["gemm_timed"] / max(1, counters["gemm_launches"]) * args.steps / (counters["gemm_ms"] / 1e3) / 1e12 \
        if counters["gemm_ms"] > 0 else None
    line = {"metric": METRIC, "value": units / (ms / 1e3), "unit": METRIC, "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {**workload_config(shape), "note": "one joint block (spot_dit_block_forward); a step = one block evaluation of 8 sequences",
                       "l2": "512 MiB written and read back between timed iterations; the block's working set exceeds L2 as well"},
            "tflops_per_gpu": tf, "ms_at_100pct_of_burst_peak": flops / peaks["bf16_tflops"] / 1e9,
            "frac_of_bf16_peak": {"burst": tf / peaks["bf16_tflops"], "sustained": tf / peaks["bf16_tflops_sustained"],
                                  "nominal_2250": tf / 2250.0, "peaks": peaks["source"]},
            "sustained": {"ms_per_step": ms_sus, "tflops": flops / ms_sus / 1e9, "launches_back_to_back": n_rep,
                          "frac_of_sustained_peak": flops / ms_sus / 1e9 / peaks["bf16_tflops_sustained"]},
            "clocks": clocks, "gpu_launches": counters["launches"],
            "e2e": {"value": units / (e_ms / 1e3), "unit": METRIC, "ms_per_step": e_ms,
                    "h2d_bytes_per_step": sum(t.numel() * t.element_size() for t in hp),
                    "d2h_bytes_per_step": sum(t.numel() * t.element_size() for t in ho),
                    "note": "pinned host tensors copied by the binding's caller around the device-pointer C-ABI call"},
            "roofline": {"bound": "tensor", "kernel": "gemm_tcgen05_v3_kernel", "achieved": gemm_tf, "peak": peaks["bf16_tflops"],
                         "peak_kind": f"{peaks['source']} burst bf16 (kernel timed in a 2 ms call after an L2 flush)", "unit": "TFLOP/s",
                         "frac": gemm_tf / peaks["bf16_tflops"] if gemm_tf else None, "traffic": None,
                         "launches_timed": counters["gemm_timed"], "avg_launch_ms": counters["gemm_ms"] / max(1, counters["gemm_timed"])},
            "cpu_baseline": None}
    if not args.no_cpu_baseline:
        from oracle import mmdit
        from tests.helpers import np64
        bw = {k: np64(v) for k, v in w["blocks"][0].items()}
        cos, sin = mmdit.rope_table(shape.grid_h, shape.grid_w, shape.n_txt, shape.rope_pairs, shape.rope_theta)
        c = mmdit.silu(np64(temb))
        hi, ht = np64(h_img[:2]), np64(h_txt[:2])
        t0 = time.perf_counter()
        for b in range(2):
            mmdit.block_forward(hi[b], ht[b], c, bw, n_heads=shape.n_heads, cos=cos, sin=sin, ln_eps=shape.ln_eps, rms_eps=shape.rms_eps)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": 2 * shape.n_img / dt, "unit": METRIC, "cores": cpu_threads(), "kind": "oracle", "seconds": dt,
                                "sample": "2 of the 8 sequences through the block (work is linear in sequences)"}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kernels", action="store_true", help="time every kernel alone against its roofline")
    ap.add_argument("--flush", choices=["clean", "dirty"], default="clean",
                    help="--kernels: L2 flush between iterations: 512 MiB written and read back (clean lines, default) or only "
                         "written (the timed kernel then also pays the write-back of the flush's dirty lines)")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="spot", choices=["spot", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own P x K batch (disjoint seeds); strong = ONE P x K batch sharded over "
                         "the ranks through sharding.explore_sharded (SURVEY.md 8(e))")
    ap.add_argument("--dry-run", action="store_true", help="host logic only: gloo, stub step, no GPU (tests)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--gap-probe", action="store_true",
                    help="after the timed region: one more rollout with an event pair around EVERY kernel launch (SPOT_OPT_TIMING = 2); "
                         "the line gains launch_gaps = share of a rollout's wall time in which no kernel of the library runs")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--graph", action="store_true",
                    help="also capture one rollout into a CUDA graph and time its replays beside the eager launches (1 GPU)")
    ap.add_argument("--gemm-impl", type=int, default=0,
                    help="0 auto (CTA pair + TMA-store epilogue, K4 fused), 2 one-CTA tcgen05, 3 CTA pair with per-thread "
                         "epilogue, 4 as 0 with K4 as its own kernel (A/B testing)")
    ap.add_argument("--precision", default="bf16", choices=["bf16", "fp8", "nvfp4"],
                    help="fp8 = the low-precision exploration variant (E4M3 block Linears, DESIGN.md section 13): NOT the "
                         "headline configuration; the line says dtype fp8 and adds the reward rank correlation with bf16")
    ap.add_argument("--cache-threshold", type=float, default=None,
                    help="run the cached-step variant (spot_explore_cached, PAPER.md:155-157) with this threshold; the line "
                         "adds the effective denoising steps; no e2e leg")
    args = ap.parse_args()
    shape = CONFIGS[WORKLOADS[args.workload]]
    world = ensure_ranks(args)
    if args.impl == "reference":
        return run_reference(args, shape)
    if args.dry_run:
        return run_dry(args, shape, world)
    if args.kernels:
        return run_kernels(args, shape)
    if args.precision != "bf16" and args.gemm_impl not in (0,):
        sys.exit("bench.py: --precision fp8 runs only on the default GEMM (--gemm-impl 0); other values would run bf16 Linears")
    if args.workload == "cfg2":
        return run_block(args, shape)

    import paper_2606_19004_b200 as spot
    from paper_2606_19004_b200 import build as spot_build

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the product path has no CPU fallback"
    torch.cuda.set_device(local_rank)
    dist = None
    nccl_log = None
    if world > 1:
        import torch.distributed as dist
        if "NCCL_DEBUG" not in os.environ:                       # keep the communicator's own record (ranks, NVLS, rings) ...
            os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
            nccl_log = os.path.join(ROOT, "gpurun_out", f"nccl_n{world}_rank%p.log")
            os.environ.update(NCCL_DEBUG="INFO", NCCL_DEBUG_SUBSYS="INIT", NCCL_DEBUG_FILE=nccl_log)   # ... out of stdout
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    joined = torch.ones(1, device="cuda")
    if dist is not None:
        dist.all_reduce(joined)                                  # n_gpus of the line = ranks that really joined
    assert int(joined.item()) == world
    if rank == 0:
        spot_build.build()
    if dist is not None:
        dist.barrier()
    spot.load_library()
    peaks = load_peaks()

    P, K, T = shape.n_prompts, shape.seeds_per_prompt, shape.n_steps
    B = P * K
    t0 = time.time()
    weights = make_weights(shape, device="cuda")
    text = make_text_emb(shape, "cuda")
    probe = make_probe(shape, "cuda")
    torch.cuda.synchronize()
    gen_s = time.time() - t0
    ctx = spot.Context(shape, weights, max_seqs=B)
    if args.gemm_impl:
        spot.spot_set_option(ctx, spot.OPT_GEMM_IMPL, args.gemm_impl)
    ts = [float(np.float32(t)) for t in shape.timesteps]
    k_sel = K // 2
    from paper_2606_19004_b200 import sharding
    strong = args.scaling == "strong"
    seeds = torch.tensor(job_seeds(shape, args.scaling, rank, world), dtype=torch.int64, device="cuda")
    n_job = B if strong else world * B                              # sequences the whole job explores per step
    out = None

    cached = args.cache_threshold is not None
    fp8 = args.precision in ("fp8", "nvfp4")
    nvfp4 = args.precision == "nvfp4"
    if cached or fp8 or strong:
        args.no_e2e = True
        assert not (strong and (cached or fp8)), "--scaling strong times the plain bf16 rollout"

    def step():
        nonlocal out
        if strong:
            out = sharding.explore_sharded(ctx, seeds, text, ts, probe, P, K, k_sel)     # shard + all-gather + selection
            return
        if cached:
            out = spot.spot_explore_cached(ctx, seeds, text, ts, probe, P, K, k_sel, args.cache_threshold, None, out)
        else:
            out = spot.spot_explore(ctx, seeds, text, ts, probe, P, K, k_sel, out)
        if dist is not None:
            sharding.gather_rewards(out["rewards"], world * B)      # the path's only exchange: world*B fp32 rewards

    def sync_all():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    full_rewards = None
    if cached or fp8:                            # the full bf16 rollout's rewards, for the rank correlation of PAPER.md:340
        full_rewards = spot.spot_explore(ctx, seeds, text, ts, probe, P, K, k_sel)["rewards"].clone()
    if nvfp4:
        ctx.enable_nvfp4(True)
    elif fp8:
        ctx.enable_fp8(True)
    for _ in range(args.warmup):
        step()
    sync_all()
    spot.spot_get_counters(ctx, reset=True)
    spot.spot_set_option(ctx, spot.OPT_TIMING, 1)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    sync_all()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    counters = spot.spot_get_counters(ctx, reset=True)
    spot.spot_set_option(ctx, spot.OPT_TIMING, 0)
    if dist is not None:
        tt = torch.tensor([ms_total], device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = tt.item()
    ms_step = ms_total / args.steps
    units_per_step = n_job * shape.n_img * T                         # image tokens x Euler steps, all ranks
    value = units_per_step / (ms_step / 1e3)
    eff_frac = float(out["computed"].sum().item()) / (B * T) if cached else 1.0     # share of (sequence, step) pairs computed
    my_seqs = B if not strong else sharding.shard_sizes(B, world)[rank]
    flops_step = shape.flops_per_rollout() * eff_frac * (n_job / B) / world          # per GPU (mean over ranks)
    tflops = flops_step / (ms_step / 1e3) / 1e12

    # roofline of the dominant kernel (tcgen05 GEMM): algorithmic GEMM FLOPs / event-timed GEMM device time
    S, D, F, L = shape.seq, shape.hidden, shape.mlp_hidden, shape.n_blocks
    lin_per_seq_block = 2 * D * (3 * D + D + 2 * F)                   # per token
    gemm_flops_step = eff_frac * T * my_seqs * (L * S * lin_per_seq_block - shape.n_txt * 2 * D * (D + 2 * F))   # last block: no text tail (this rank)
    if nvfp4:      # the event-timed kernel (gemm_tcgen05_v3) runs only QKV and out-proj here; fc1 / fc2 are gemm_nvfp4_kernel launches
        gemm_flops_step = eff_frac * T * my_seqs * (L * S * 2 * D * 4 * D - shape.n_txt * 2 * D * D)
    timed_frac = counters["gemm_timed"] / max(1, counters["gemm_launches"])
    gemm_ms = counters["gemm_ms"]
    gemm_tflops = (gemm_flops_step * args.steps * timed_frac) / (gemm_ms / 1e3) / 1e12 if gemm_ms > 0 else None
    gemm_peak = peaks["bf16_tflops_sustained"] * (2.0 if fp8 else 1.0)
    peak_kind = f"{peaks['source']} sustained bf16 (kernel timed inside a long step)" + (" x 2 (nominal fp8 : bf16 ratio)" if fp8 else "")
    roofline = {"bound": "tensor", "kernel": "gemm_tcgen05_v3_kernel", "achieved": gemm_tflops,
                "peak": gemm_peak, "peak_kind": peak_kind,
                "unit": "TFLOP/s", "frac": (gemm_tflops / gemm_peak) if gemm_tflops else None,
                "traffic": None if fp8 else GEMM_DRAM_TRAFFIC_PER_LAUNCH.get(args.workload), "launches_timed": counters["gemm_timed"],
                "avg_launch_ms": gemm_ms / max(1, counters["gemm_timed"]), "share_of_step": gemm_ms / ms_total / max(timed_frac, 1e-9),
                "flops_per_launch": gemm_flops_step / max(1, counters["gemm_launches"] / args.steps)}

    # e2e: the host-buffer C-ABI call, host<->device copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda t: t.cpu().pin_memory()
        h_seeds, h_text, h_probe = pin(seeds), pin(text), pin(probe)
        h_out = {"latents": torch.empty((B, shape.n_img, shape.latent_ch)).pin_memory(), "rewards": torch.empty(B).pin_memory(),
                 "stats": torch.empty((P, 2)).pin_memory(), "top": torch.empty((P, k_sel), dtype=torch.int32).pin_memory(),
                 "bottom": torch.empty((P, k_sel), dtype=torch.int32).pin_memory()}
        spot.spot_explore_host(ctx, h_seeds, h_text, ts, h_probe, P, K, k_sel, h_out)
        sync_all()
        w0 = time.perf_counter()
        ev0.record()
        for _ in range(args.steps):
            spot.spot_explore_host(ctx, h_seeds, h_text, ts, h_probe, P, K, k_sel, h_out)
        ev1.record()
        sync_all()
        e_ms = ev0.elapsed_time(ev1) / args.steps
        wall_ms = (time.perf_counter() - w0) * 1e3 / args.steps
        e_ms = max(e_ms, wall_ms)                                      # the host call synchronises: wall clock bounds it
        if dist is not None:
            tt = torch.tensor([e_ms], device="cuda")
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e_ms = tt.item()
        h2d = h_seeds.numel() * 8 + h_text.numel() * h_text.element_size() + h_probe.numel() * 4
        d2h = sum(t.numel() * t.element_size() for t in h_out.values())
        e2e = {"value": units_per_step / (e_ms / 1e3), "unit": METRIC, "ms_per_step": e_ms,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}
        assert torch.equal(h_out["rewards"], out["rewards"].cpu()), "host and device entry points disagree"

    gaps = None
    if args.gap_probe and not strong:
        spot.spot_get_counters(ctx, reset=True)
        spot.spot_set_option(ctx, spot.OPT_TIMING, 2)
        sync_all()
        step()
        sync_all()
        cg = spot.spot_get_counters(ctx, reset=True)
        spot.spot_set_option(ctx, spot.OPT_TIMING, 0)
        gaps = {"kernel_ms_sum": cg["gemm_ms"], "launches": cg["gemm_timed"], "rollout_ms": ms_step,
                "idle_share": 1.0 - cg["gemm_ms"] / ms_step,
                "how": "sum of CUDA-event durations around every kernel launch of one extra rollout, against ms_per_step of the timed region"}

    graph = None
    if args.graph and dist is None and not cached and not strong:
        # SURVEY.md 3.2 "capturable as one CUDA graph per config": the same step(), captured once and replayed
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        t0 = time.perf_counter()
        with torch.cuda.graph(g, stream=side):
            step()
        capture_s = time.perf_counter() - t0
        eager_rewards = out["rewards"].clone()
        g.replay()
        sync_all()
        ev0.record()
        for _ in range(args.steps):
            g.replay()
        ev1.record()
        sync_all()
        g_ms = ev0.elapsed_time(ev1) / args.steps
        ev0.record()
        for _ in range(args.steps):
            step()
        ev1.record()
        sync_all()
        eager_ms = ev0.elapsed_time(ev1) / args.steps
        graph = {"ms_per_step": g_ms, "eager_ms_per_step_back_to_back": eager_ms, "eager_over_graph": eager_ms / g_ms,
                 "capture_s": capture_s, "same_rewards_as_eager": bool(torch.equal(out["rewards"], eager_rewards))}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nb = SAMPLE_BLOCKS
        w_host = {"global": {k: v.cpu() for k, v in weights["global"].items()},
                  "blocks": [{k: v.cpu() for k, v in b.items()} for b in weights["blocks"][:nb]]}
        dt = min(oracle_sample(shape, w_host, text[:1].cpu(), nb) for _ in range(2))
        cpu_baseline = {"value": SAMPLE_SEEDS * shape.n_img * (nb / L) / dt, "unit": METRIC, "cores": cpu_threads(), "kind": "oracle",
                        "seconds": dt, "host_cores": os.cpu_count(),
                        "sample": f"{SAMPLE_SEEDS} seeds x 1 Euler step x {nb} of {L} blocks at full width, best of 2 "
                                  "(work is linear in seeds, steps, blocks)"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": int(joined.item()), "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
                "dtype": ("nvfp4 MLP Linears + fp8_e4m3 QKV / out-proj (bf16 attention, fp32 residual): exploration variant, not the headline" if nvfp4
                          else "fp8_e4m3 block Linears (bf16 attention, fp32 residual): exploration variant, not the headline" if fp8 else "bf16"),
                "data": "synthetic",
                "config": {**workload_config(shape),
                           "l2": "inputs (40.8 GB of weights streamed every Euler step) are larger than L2",
                           "chunk_seqs": 32,     # SPOT_OPT_CHUNK_SEQS default: batches above it run chunk by chunk (spot.h)
                           "parallelism": parallelism_label(args.scaling, world, B)},
                "seeds_per_s": n_job / (ms_step / 1e3), "tflops_per_gpu": tflops,
                "frac_of_bf16_peak": {"burst": tflops / peaks["bf16_tflops"], "sustained": tflops / peaks["bf16_tflops_sustained"],
                                      "nominal_2250": tflops / 2250.0, "peaks": peaks["source"]},
                "clocks": clocks, "e2e": e2e, "gpu_launches": counters["launches"], "roofline": roofline,
                "cpu_baseline": cpu_baseline, "weight_gen_s": gen_s}
        if gaps:
            line["launch_gaps"] = gaps
        if graph is not None:
            line["cuda_graph"] = graph
        if nccl_log:
            line["nccl_log"] = os.path.relpath(nccl_log, ROOT)
        rk = lambda v: torch.argsort(torch.argsort(v)).double()
        if fp8:
            line["fp8"] = {"reward_rank_correlation_vs_bf16_per_prompt":
                           [float(torch.corrcoef(torch.stack([rk(out["rewards"][g * K:(g + 1) * K]), rk(full_rewards[g * K:(g + 1) * K])]))[0, 1])
                            for g in range(P)],
                           "reward_rel_l2_vs_bf16": float((out["rewards"] - full_rewards).norm() / full_rewards.norm()),
                           "note": "tflops_per_gpu counts the same algorithmic FLOPs as the bf16 line"}
        if cached:
            eff = out["computed"].sum(1).tolist()
            corr = [float(torch.corrcoef(torch.stack([rk(out["rewards"][g * K:(g + 1) * K]), rk(full_rewards[g * K:(g + 1) * K])]))[0, 1])
                    for g in range(P)]
            line["cache"] = {"threshold": args.cache_threshold, "scheduled_steps": T, "effective_steps_mean": sum(eff) / len(eff),
                             "effective_steps_per_sequence": eff, "reward_rank_correlation_vs_full_rollout_per_prompt": corr,
                             "note": "value counts SCHEDULED steps (PAPER.md:157: cached "
                             "steps reuse the previous transformer residual); tflops_per_gpu counts computed steps only"}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
