#!/usr/bin/env python
"""bench.py - seed-exploration rollout throughput on B200 (contract: see DESIGN.md "Measurement").

A "step" is ONE whole pass of the hot path over one batch: seeds -> Philox/Box-Muller latents -> T Euler steps
of the 60-block MMDiT -> probe rewards -> top/bottom-k selection (spot_explore).  Default workload = config 3
of BASELINE.json (512x512, 60 blocks, 1 prompt x 16 seeds, 10 Euler steps, bf16), the configuration the
metric's ">= 50 % of dense BF16 peak" target is quoted on.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg4|cfg5] [--impl reference]

N > 1 is launched by torch.distributed.run (one rank per GPU); ranks hold replicated weights and disjoint
seed groups (weak scaling, no data-path collective; the K fp32 rewards are all-gathered once per step).
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
# block (QKV+RoPE 1.071 GB, out-proj 0.646 GB, fc1 1.451 GB, fc2 2.680 GB) - profiles/r1_ncu_full_gemm_v3.txt (config 3)
GEMM_DRAM_TRAFFIC_PER_LAUNCH = {"cfg3": 1.462e9}
WORKLOADS = {"cfg3": 3, "cfg4": 4, "cfg5": 5}


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
                       "peak_kind": "derived: 148 SMs x 128 lanes x 1.965 GHz / 56.5 SASS instructions per normal"}
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--gemm-impl", type=int, default=0,
                    help="0 auto (CTA pair + TMA-store epilogue, K4 fused), 2 one-CTA tcgen05, 3 CTA pair with per-thread "
                         "epilogue, 4 as 0 with K4 as its own kernel (A/B testing)")
    ap.add_argument("--precision", default="bf16", choices=["bf16", "fp8"],
                    help="fp8 = the low-precision exploration variant (E4M3 block Linears, DESIGN.md section 13): NOT the "
                         "headline configuration; the line says dtype fp8 and adds the reward rank correlation with bf16")
    ap.add_argument("--cache-threshold", type=float, default=None,
                    help="run the cached-step variant (spot_explore_cached, PAPER.md:155-157) with this threshold; the line "
                         "adds the effective denoising steps; no e2e leg")
    args = ap.parse_args()
    shape = CONFIGS[WORKLOADS[args.workload]]
    if args.impl == "reference":
        return run_reference(args, shape)
    if args.kernels:
        return run_kernels(args, shape)

    import paper_2606_19004_b200 as spot
    from paper_2606_19004_b200 import build as spot_build

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the product path has no CPU fallback"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
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
    # weak scaling: the job explores world * B sequences; rank r owns the contiguous shard [r*B, (r+1)*B)
    from paper_2606_19004_b200 import sharding
    lo, hi = sharding.shard_range(world * B, rank, world)
    assert hi - lo == B
    seeds = torch.tensor([int(shape.seeds[i % B]) + (i // B) * B for i in range(lo, hi)], dtype=torch.int64, device="cuda")
    out = None

    cached = args.cache_threshold is not None
    fp8 = args.precision == "fp8"
    if cached or fp8:
        args.no_e2e = True

    def step():
        nonlocal out
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
    if fp8:
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
    units_per_step = world * B * shape.n_img * T                     # image tokens x Euler steps, all ranks
    value = units_per_step / (ms_step / 1e3)
    eff_frac = float(out["computed"].sum().item()) / (B * T) if cached else 1.0     # share of (sequence, step) pairs computed
    flops_step = shape.flops_per_rollout() * eff_frac
    tflops = flops_step / (ms_step / 1e3) / 1e12                     # per GPU

    # roofline of the dominant kernel (tcgen05 GEMM): algorithmic GEMM FLOPs / event-timed GEMM device time
    S, D, F, L = shape.seq, shape.hidden, shape.mlp_hidden, shape.n_blocks
    lin_per_seq_block = 2 * D * (3 * D + D + 2 * F)                   # per token
    gemm_flops_step = eff_frac * T * B * (L * S * lin_per_seq_block - shape.n_txt * 2 * D * (D + 2 * F))   # last block: no text tail
    timed_frac = counters["gemm_timed"] / max(1, counters["gemm_launches"])
    gemm_ms = counters["gemm_ms"]
    gemm_tflops = (gemm_flops_step * args.steps * timed_frac) / (gemm_ms / 1e3) / 1e12 if gemm_ms > 0 else None
    gemm_peak = peaks["bf16_tflops_sustained"] * (2.0 if fp8 else 1.0)
    peak_kind = f"{peaks['source']} sustained bf16 (kernel timed inside a long step)" + (" x 2 (nominal fp8 : bf16 ratio)" if fp8 else "")
    roofline = {"bound": "tensor", "kernel": "gemm_tcgen05_v3_kernel", "achieved": gemm_tflops,
                "peak": gemm_peak, "peak_kind": peak_kind,
                "unit": "TFLOP/s", "frac": (gemm_tflops / gemm_peak) if gemm_tflops else None,
                "traffic": GEMM_DRAM_TRAFFIC_PER_LAUNCH.get(args.workload), "launches_timed": counters["gemm_timed"],
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

    cpu_baseline = None
    if rank == 0 and not args.no_cpu_baseline:
        nb = SAMPLE_BLOCKS
        w_host = {"global": {k: v.cpu() for k, v in weights["global"].items()},
                  "blocks": [{k: v.cpu() for k, v in b.items()} for b in weights["blocks"][:nb]]}
        dt = min(oracle_sample(shape, w_host, text[:1].cpu(), nb) for _ in range(2))
        cpu_baseline = {"value": SAMPLE_SEEDS * shape.n_img * (nb / L) / dt, "unit": METRIC, "cores": cpu_threads(), "kind": "oracle",
                        "seconds": dt, "host_cores": os.cpu_count(),
                        "sample": f"{SAMPLE_SEEDS} seeds x 1 Euler step x {nb} of {L} blocks at full width, best of 2 "
                                  "(work is linear in seeds, steps, blocks)"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "fp8_e4m3 block Linears (bf16 attention, fp32 residual): exploration variant, not the headline" if fp8 else "bf16",
                "data": "synthetic",
                "config": {**workload_config(shape),
                           "l2": "inputs (40.8 GB of weights streamed every Euler step) are larger than L2",
                           "chunk_seqs": 32,     # SPOT_OPT_CHUNK_SEQS default: batches above it run chunk by chunk (spot.h)
                           "parallelism": f"replicas x{world}, disjoint seed groups"},
                "seeds_per_s": world * B / (ms_step / 1e3), "tflops_per_gpu": tflops,
                "frac_of_bf16_peak": {"burst": tflops / peaks["bf16_tflops"], "sustained": tflops / peaks["bf16_tflops_sustained"],
                                      "nominal_2250": tflops / 2250.0, "peaks": peaks["source"]},
                "clocks": clocks, "e2e": e2e, "gpu_launches": counters["launches"], "roofline": roofline,
                "cpu_baseline": cpu_baseline, "weight_gen_s": gen_s}
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
