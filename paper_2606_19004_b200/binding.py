"""Thin ctypes binding over libspot.so: argument marshalling only.

Every function has the name of the C entry point it calls (include/spot.h, include/spot_kernels.h)
and passes torch tensors as raw device (or host) pointers.  Nothing is computed here; if the shared
library is missing or a call fails, an exception is raised - there is no fallback.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libspot.so")
_lib: Optional[C.CDLL] = None

SPOT_F32, SPOT_BF16 = 0, 1
EPI_BIAS, EPI_BIAS_GELU, EPI_GATE_RESIDUAL = 0, 1, 2
IMPL_AUTO, IMPL_SIMT, IMPL_TCGEN05, IMPL_TCGEN05_2CTA, IMPL_TCGEN05_TMA = 0, 1, 2, 3, 4
OPT_GEMM_IMPL, OPT_ATTN_IMPL, OPT_TIMING, OPT_FP8, OPT_CHUNK_SEQS, OPT_NVFP4 = 0, 1, 2, 3, 4, 5
SPOT_E4M3 = 2     # storage type of the FP8 variant's activations / quantised weights (torch.float8_e4m3fn)
STATUS_NAMES = ["SPOT_OK", "SPOT_ERR_NULL", "SPOT_ERR_SHAPE", "SPOT_ERR_DTYPE", "SPOT_ERR_ALIGN",
                "SPOT_ERR_WORKSPACE", "SPOT_ERR_ARCH", "SPOT_ERR_CUDA", "SPOT_ERR_UNIMPLEMENTED"]


class SpotError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.status_name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        self.cuda_error = cuda_error
        extra = f" (cudaError_t {cuda_error})" if cuda_error else ""
        super().__init__(f"{where}: {self.status_name}{extra}")


class SpotConfig(C.Structure):
    _fields_ = [("n_blocks", C.c_int32), ("hidden", C.c_int32), ("n_heads", C.c_int32), ("head_dim", C.c_int32),
                ("mlp_hidden", C.c_int32), ("grid_h", C.c_int32), ("grid_w", C.c_int32), ("n_txt", C.c_int32),
                ("latent_ch", C.c_int32), ("txt_dim", C.c_int32), ("rope_pairs", C.c_int32 * 3),
                ("rope_theta", C.c_float), ("ln_eps", C.c_float), ("rms_eps", C.c_float), ("dtype", C.c_int)]


_STREAM_FIELDS = ["mod_w", "mod_b", "qkv_w", "qkv_b", "q_gain", "k_gain", "out_w", "out_b", "fc1_w", "fc1_b", "fc2_w", "fc2_b"]


class SpotStreamWeights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _STREAM_FIELDS]


class SpotBlockWeights(C.Structure):
    _fields_ = [("s", SpotStreamWeights * 2)]


class SpotWeights(C.Structure):
    _fields_ = [("time_w1", C.c_void_p), ("time_b1", C.c_void_p), ("time_w2", C.c_void_p), ("time_b2", C.c_void_p),
                ("img_in_w", C.c_void_p), ("img_in_b", C.c_void_p), ("txt_gain", C.c_void_p), ("txt_in_w", C.c_void_p),
                ("txt_in_b", C.c_void_p), ("blocks", C.POINTER(SpotBlockWeights)), ("final_mod_w", C.c_void_p),
                ("final_mod_b", C.c_void_p), ("proj_w", C.c_void_p), ("proj_b", C.c_void_p)]


def library_path() -> str:
    return _LIB_PATH


def load_library() -> C.CDLL:
    """Loads libspot.so (built by paper_2606_19004_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise FileNotFoundError(f"{_LIB_PATH} not found: run `python -m paper_2606_19004_b200.build` "
                                "(or __graft_entry__.build()); there is no fallback path")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, i64, u32, f32, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint32, C.c_float, C.c_size_t
    sig = {
        "spot_create": [C.POINTER(SpotConfig), C.POINTER(SpotWeights), i32, C.POINTER(vp)],
        "spot_destroy": [vp],
        "spot_set_option": [vp, i32, i32],
        "spot_workspace_bytes": [vp, i32, i32, C.POINTER(sz)],
        "spot_last_cuda_error": [vp],
        "spot_get_counters": [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64),
                              C.POINTER(C.c_double), i32],
        "spot_noise_from_seeds": [vp, i32, i64, u32, vp, vp],
        "spot_philox_words": [vp, i32, i64, u32, vp, vp],
        "spot_dit_block_forward": [vp, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp],
        "spot_dit_denoise": [vp, i32, i32, vp, vp, vp, i32, vp, sz, vp],
        "spot_seed_rewards": [vp, i32, i32, vp, vp, i32, vp, vp, vp, vp, vp],
        "spot_select_seeds": [vp, i32, i32, i32, vp, vp, vp, vp],
        "spot_explore": [vp, i32, i32, vp, vp, vp, i32, vp, i32, vp, vp, vp, vp, vp, vp, sz, vp],
        "spot_workspace_bytes_cached": [vp, i32, i32, C.POINTER(sz)],
        "spot_dit_denoise_cached": [vp, i32, i32, vp, vp, vp, i32, C.POINTER(SpotCacheConfig), vp, vp, vp, sz, vp],
        "spot_explore_cached": [vp, i32, i32, vp, vp, vp, i32, vp, i32, C.POINTER(SpotCacheConfig), vp, vp, vp, vp, vp, vp, vp,
                                vp, sz, vp],
        "spot_dit_denoise_sde": [vp, i32, i32, vp, vp, vp, vp, i32, f32, i32, i32, i32, vp, vp, sz, vp],
        "spot_sde_update": [vp, vp, vp, i32, f32, f32, f32, i32, i64, vp, vp, vp],
        "spot_fp8_bytes": [vp, C.POINTER(sz)],
        "spot_fp8_prepare": [vp, vp, sz, vp],
        "spot_nvfp4_bytes": [vp, C.POINTER(sz)],
        "spot_nvfp4_prepare": [vp, vp, sz, vp],
        "spot_quantize_weight_rows": [vp, i64, i64, vp, vp, vp],
        "spot_quantize_e4m3": [i32, vp, i64, vp, vp],
        "spot_linear_fp8": [i32, vp, i64, i64, vp, i64, vp, vp, vp, vp, vp, vp],
        "spot_nvfp4_sizes": [i64, i64, C.POINTER(sz), C.POINTER(sz)],
        "spot_nvfp4_row_scale": [vp, i64, i64, vp, vp],
        "spot_nvfp4_quantize": [vp, i64, i64, vp, vp, vp, vp],
        "spot_linear_nvfp4": [i32, vp, vp, i64, i64, vp, vp, vp, i64, vp, vp, vp, vp, vp, vp],
        "spot_explore_host": [vp, i32, i32, vp, vp, vp, i32, vp, i32, vp, vp, vp, vp, vp, vp, sz, vp],
        "spot_linear": [i32, i32, i32, vp, i64, i64, vp, i64, vp, vp, vp, vp, vp],
        "spot_qkv_rope_linear": [vp, i32, i32, i64, vp, i64, vp, vp, vp, vp, vp, i32, f32, vp, vp],
        "spot_qkv_rope_linear_fp8": [vp, i32, i32, i64, vp, vp, i64, vp, vp, vp, vp, vp, i32, f32, vp, vp],
        "spot_ln_modulate": [i32, vp, i64, i64, vp, vp, f32, vp, vp],
        "spot_qk_norm_rope": [i32, vp, i32, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, f32, vp],
        "spot_attention": [i32, i32, vp, vp, i32, i32, i32, i32, vp],
        "spot_euler_update": [vp, vp, f32, i32, i64, vp, vp, vp, vp],
        "spot_euler_update_static": [vp, vp, f32, i32, i64, vp, vp, vp],
        "spot_rope_table": [vp, vp, vp],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = C.c_int
    lib.spot_status_string.argtypes = [C.c_int]
    lib.spot_status_string.restype = C.c_char_p
    lib.spot_version.argtypes = []
    lib.spot_version.restype = C.c_char_p
    _lib = lib
    return lib


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    assert t.is_contiguous(), "libspot takes dense row-major buffers"
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0


def _dt(dtype: torch.dtype) -> int:
    if dtype == torch.float32:
        return SPOT_F32
    if dtype == torch.bfloat16:
        return SPOT_BF16
    if dtype == torch.float8_e4m3fn:
        return SPOT_E4M3
    raise TypeError(f"unsupported dtype {dtype}")


def _check(status: int, where: str, ctx: Optional["Context"] = None) -> None:
    if status != 0:
        ce = load_library().spot_last_cuda_error(ctx.handle) if (ctx is not None and status == 7) else 0
        raise SpotError(status, where, ce)


class SpotCacheConfig(C.Structure):
    _fields_ = [("threshold", C.c_float), ("n_coeffs", C.c_int32), ("coeffs", C.c_float * 8)]


def _cache_cfg(threshold: float, coeffs: Optional[Sequence[float]]) -> SpotCacheConfig:
    cc = SpotCacheConfig(threshold=float(threshold), n_coeffs=0)
    if coeffs is not None:
        cc.n_coeffs = len(coeffs)
        for j, v in enumerate(list(coeffs)[:8]):      # the library rejects n_coeffs > 8
            cc.coeffs[j] = float(v)
    return cc


class Context:
    """spot_ctx: validated config + borrowed weights (keeps the torch tensors alive)."""

    def __init__(self, shape, weights: Dict[str, object], max_seqs: int):
        lib = load_library()
        self.shape = shape
        self._keep = weights
        cfg = SpotConfig(n_blocks=shape.n_blocks, hidden=shape.hidden, n_heads=shape.n_heads, head_dim=shape.head_dim,
                         mlp_hidden=shape.mlp_hidden, grid_h=shape.grid_h, grid_w=shape.grid_w, n_txt=shape.n_txt,
                         latent_ch=shape.latent_ch, txt_dim=shape.txt_dim, rope_pairs=(C.c_int32 * 3)(*shape.rope_pairs),
                         rope_theta=shape.rope_theta, ln_eps=shape.ln_eps, rms_eps=shape.rms_eps, dtype=_dt(shape.dtype))
        g = weights["global"]
        blocks: List[Dict[str, torch.Tensor]] = weights["blocks"]
        arr = (SpotBlockWeights * max(1, len(blocks)))()
        for b, bw in enumerate(blocks):
            for si, stream in enumerate(("img", "txt")):
                for f in _STREAM_FIELDS:
                    setattr(arr[b].s[si], f, _ptr(bw[f"{stream}.{f}"]))
        w = SpotWeights(blocks=C.cast(arr, C.POINTER(SpotBlockWeights)))
        for name in ("time_w1", "time_b1", "time_w2", "time_b2", "img_in_w", "img_in_b", "txt_gain", "txt_in_w",
                     "txt_in_b", "final_mod_w", "final_mod_b", "proj_w", "proj_b"):
            setattr(w, name, _ptr(g[name]))
        self._cfg, self._w, self._arr = cfg, w, arr
        self.cfg_struct = cfg
        h = C.c_void_p()
        _check(lib.spot_create(C.byref(cfg), C.byref(w), max_seqs, C.byref(h)), "spot_create")
        self.handle = h
        self.max_seqs = max_seqs
        self._ws: Optional[torch.Tensor] = None

    def close(self) -> None:
        if getattr(self, "handle", None):
            load_library().spot_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def enable_fp8(self, on: bool = True) -> None:
        """Low-precision exploration variant: quantise the block Linears once (E4M3 weights +
        per-output-channel scales in a buffer this object keeps alive) and switch the context's block Linears."""
        lib = load_library()
        if on and getattr(self, "_fp8_buf", None) is None:
            n = C.c_size_t()
            _check(lib.spot_fp8_bytes(self.handle, C.byref(n)), "spot_fp8_bytes", self)
            self._fp8_buf = torch.empty(int(n.value), dtype=torch.uint8, device="cuda")
            _check(lib.spot_fp8_prepare(self.handle, _ptr(self._fp8_buf), self._fp8_buf.numel(), _stream()), "spot_fp8_prepare", self)
        _check(lib.spot_set_option(self.handle, OPT_FP8, 1 if on else 0), "spot_set_option", self)

    def enable_nvfp4(self, on: bool = True) -> None:
        """4-bit exploration variant: FP8 variant + fc1 / fc2 on NVFP4 operands.  on=True switches both
        on; on=False switches both off (back to bf16)."""
        lib = load_library()
        if on:
            self.enable_fp8(True)
            if getattr(self, "_nvfp4_buf", None) is None:
                n = C.c_size_t()
                _check(lib.spot_nvfp4_bytes(self.handle, C.byref(n)), "spot_nvfp4_bytes", self)
                self._nvfp4_buf = torch.empty(int(n.value), dtype=torch.uint8, device="cuda")
                _check(lib.spot_nvfp4_prepare(self.handle, _ptr(self._nvfp4_buf), self._nvfp4_buf.numel(), _stream()), "spot_nvfp4_prepare", self)
        _check(lib.spot_set_option(self.handle, OPT_NVFP4, 1 if on else 0), "spot_set_option", self)
        if not on:
            _check(lib.spot_set_option(self.handle, OPT_FP8, 0), "spot_set_option", self)

    def workspace(self, n_seqs: int, n_steps: int, cached: bool = False) -> torch.Tensor:
        n = spot_workspace_bytes(self, n_seqs, n_steps, cached)
        if self._ws is None or self._ws.numel() < n:
            self._ws = None
            self._ws = torch.empty(n, dtype=torch.uint8, device="cuda")
        return self._ws


def spot_version() -> str:
    return load_library().spot_version().decode()


def spot_set_option(ctx: Context, opt: int, value: int) -> None:
    _check(load_library().spot_set_option(ctx.handle, opt, value), "spot_set_option", ctx)


def spot_get_counters(ctx: Context, reset: bool = False) -> dict:
    a, b, c, d = C.c_uint64(), C.c_uint64(), C.c_uint64(), C.c_double()
    _check(load_library().spot_get_counters(ctx.handle, C.byref(a), C.byref(b), C.byref(c), C.byref(d), int(reset)),
           "spot_get_counters", ctx)
    return {"launches": int(a.value), "gemm_launches": int(b.value), "gemm_timed": int(c.value), "gemm_ms": float(d.value)}


def spot_workspace_bytes(ctx: Context, n_seqs: int, n_steps: int, cached: bool = False) -> int:
    out = C.c_size_t()
    fn = load_library().spot_workspace_bytes_cached if cached else load_library().spot_workspace_bytes
    _check(fn(ctx.handle, n_seqs, n_steps, C.byref(out)), "spot_workspace_bytes", ctx)
    return int(out.value)


def spot_noise_from_seeds(seeds: torch.Tensor, elems_per_seed: int, stream_id: int = 0,
                          out: Optional[torch.Tensor] = None) -> torch.Tensor:
    assert seeds.dtype in (torch.int64, torch.uint64)
    n = seeds.numel()
    if out is None:
        out = torch.empty((n, elems_per_seed), dtype=torch.float32, device=seeds.device)
    _check(load_library().spot_noise_from_seeds(_ptr(seeds), n, elems_per_seed, stream_id, _ptr(out), _stream()),
           "spot_noise_from_seeds")
    return out


def spot_philox_words(seeds: torch.Tensor, elems_per_seed: int, stream_id: int = 0) -> torch.Tensor:
    n = seeds.numel()
    out = torch.empty((n, elems_per_seed), dtype=torch.int32, device=seeds.device)
    _check(load_library().spot_philox_words(_ptr(seeds), n, elems_per_seed, stream_id, _ptr(out), _stream()),
           "spot_philox_words")
    return out


def spot_dit_block_forward(ctx: Context, block: int, h_img: torch.Tensor, h_txt: torch.Tensor, temb: torch.Tensor,
                           out_img: Optional[torch.Tensor] = None, out_txt: Optional[torch.Tensor] = None):
    n_seqs = h_img.shape[0]
    out_img = torch.empty_like(h_img) if out_img is None else out_img
    out_txt = torch.empty_like(h_txt) if out_txt is None else out_txt
    ws = ctx.workspace(n_seqs, 1)
    _check(load_library().spot_dit_block_forward(ctx.handle, block, n_seqs, _ptr(h_img), _ptr(h_txt), _ptr(temb),
                                                 _ptr(out_img), _ptr(out_txt), _ptr(ws), ws.numel(), _stream()),
           "spot_dit_block_forward", ctx)
    return out_img, out_txt


def _timesteps(ts: Sequence[float]):
    arr = (C.c_float * len(ts))(*[float(t) for t in ts])
    return arr, len(ts) - 1


def spot_dit_denoise(ctx: Context, latents: torch.Tensor, text_emb: torch.Tensor, timesteps: Sequence[float],
                     n_prompts: int, seeds_per_prompt: int) -> torch.Tensor:
    arr, T = _timesteps(timesteps)
    ws = ctx.workspace(n_prompts * seeds_per_prompt, T)
    _check(load_library().spot_dit_denoise(ctx.handle, n_prompts, seeds_per_prompt, _ptr(latents), _ptr(text_emb),
                                           C.cast(arr, C.c_void_p), T, _ptr(ws), ws.numel(), _stream()),
           "spot_dit_denoise", ctx)
    return latents


def spot_seed_rewards(ctx: Context, latents: torch.Tensor, probe: torch.Tensor, n_prompts: int, seeds_per_prompt: int,
                      k_select: int):
    dev = latents.device
    rewards = torch.empty(n_prompts * seeds_per_prompt, dtype=torch.float32, device=dev)
    stats = torch.empty((n_prompts, 2), dtype=torch.float32, device=dev)
    top = torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev)
    bottom = torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev)
    _check(load_library().spot_seed_rewards(ctx.handle, n_prompts, seeds_per_prompt, _ptr(latents), _ptr(probe), k_select,
                                            _ptr(rewards), _ptr(stats), _ptr(top), _ptr(bottom), _stream()),
           "spot_seed_rewards", ctx)
    return rewards, stats, top[:, :k_select], bottom[:, :k_select]


def spot_select_seeds(rewards: torch.Tensor, n_prompts: int, seeds_per_prompt: int, k_select: int):
    """A7 on rewards already on the device: (stats [P, 2], top [P, k], bottom [P, k])."""
    dev = rewards.device
    stats = torch.empty((n_prompts, 2), dtype=torch.float32, device=dev)
    top = torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev)
    bottom = torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev)
    _check(load_library().spot_select_seeds(_ptr(rewards), n_prompts, seeds_per_prompt, k_select, _ptr(stats), _ptr(top),
                                            _ptr(bottom), _stream()), "spot_select_seeds")
    return stats, top[:, :k_select], bottom[:, :k_select]


def spot_explore(ctx: Context, seeds: torch.Tensor, text_emb: torch.Tensor, timesteps: Sequence[float],
                 probe: torch.Tensor, n_prompts: int, seeds_per_prompt: int, k_select: int,
                 out: Optional[dict] = None) -> dict:
    """Device-buffer rollout.  `out` may carry preallocated latents/rewards/stats/top/bottom tensors."""
    dev = seeds.device
    B = n_prompts * seeds_per_prompt
    s = ctx.shape
    if out is None:
        out = {"latents": torch.empty((B, s.n_img, s.latent_ch), dtype=torch.float32, device=dev),
               "rewards": torch.empty(B, dtype=torch.float32, device=dev),
               "stats": torch.empty((n_prompts, 2), dtype=torch.float32, device=dev),
               "top": torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev),
               "bottom": torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev)}
    arr, T = _timesteps(timesteps)
    ws = ctx.workspace(B, T)
    _check(load_library().spot_explore(ctx.handle, n_prompts, seeds_per_prompt, _ptr(seeds), _ptr(text_emb),
                                       C.cast(arr, C.c_void_p), T, _ptr(probe), k_select, _ptr(out["latents"]),
                                       _ptr(out["rewards"]), _ptr(out["stats"]), _ptr(out["top"]), _ptr(out["bottom"]),
                                       _ptr(ws), ws.numel(), _stream()), "spot_explore", ctx)
    return out


def spot_explore_cached(ctx: Context, seeds: torch.Tensor, text_emb: torch.Tensor, timesteps: Sequence[float],
                        probe: torch.Tensor, n_prompts: int, seeds_per_prompt: int, k_select: int, threshold: float,
                        coeffs: Optional[Sequence[float]] = None, out: Optional[dict] = None) -> dict:
    """Cached-step exploration.  Adds out["computed"] [B, T] uint8 (host) and out["rel"] [B, T] fp32
    (host); out["computed"].sum(1) = effective denoising steps per sequence.  Synchronises once per Euler step."""
    dev = seeds.device
    B = n_prompts * seeds_per_prompt
    s = ctx.shape
    if out is None:
        out = {"latents": torch.empty((B, s.n_img, s.latent_ch), dtype=torch.float32, device=dev),
               "rewards": torch.empty(B, dtype=torch.float32, device=dev),
               "stats": torch.empty((n_prompts, 2), dtype=torch.float32, device=dev),
               "top": torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev),
               "bottom": torch.empty((n_prompts, max(k_select, 1)), dtype=torch.int32, device=dev)}
    arr, T = _timesteps(timesteps)
    out["computed"] = torch.zeros((B, T), dtype=torch.uint8)
    out["rel"] = torch.zeros((B, T), dtype=torch.float32)
    ws = ctx.workspace(B, T, cached=True)
    cc = _cache_cfg(threshold, coeffs)
    _check(load_library().spot_explore_cached(ctx.handle, n_prompts, seeds_per_prompt, _ptr(seeds), _ptr(text_emb),
                                              C.cast(arr, C.c_void_p), T, _ptr(probe), k_select, C.byref(cc),
                                              _ptr(out["latents"]), _ptr(out["rewards"]), _ptr(out["stats"]), _ptr(out["top"]),
                                              _ptr(out["bottom"]), _ptr(out["computed"]), _ptr(out["rel"]), _ptr(ws), ws.numel(),
                                              _stream()), "spot_explore_cached", ctx)
    return out


def spot_dit_denoise_cached(ctx: Context, latents: torch.Tensor, text_emb: torch.Tensor, timesteps: Sequence[float],
                            n_prompts: int, seeds_per_prompt: int, threshold: float,
                            coeffs: Optional[Sequence[float]] = None):
    """In place on latents; returns (latents, computed [B, T] uint8 host, rel [B, T] fp32 host)."""
    B = n_prompts * seeds_per_prompt
    arr, T = _timesteps(timesteps)
    computed = torch.zeros((B, T), dtype=torch.uint8)
    rel = torch.zeros((B, T), dtype=torch.float32)
    ws = ctx.workspace(B, T, cached=True)
    cc = _cache_cfg(threshold, coeffs)
    _check(load_library().spot_dit_denoise_cached(ctx.handle, n_prompts, seeds_per_prompt, _ptr(latents), _ptr(text_emb),
                                                  C.cast(arr, C.c_void_p), T, C.byref(cc), _ptr(computed), _ptr(rel), _ptr(ws),
                                                  ws.numel(), _stream()), "spot_dit_denoise_cached", ctx)
    return latents, computed, rel


def spot_dit_denoise_sde(ctx: Context, seeds: torch.Tensor, latents: torch.Tensor, text_emb: torch.Tensor,
                         timesteps: Sequence[float], n_prompts: int, seeds_per_prompt: int, noise_level: float,
                         window: Sequence[int], first_step: int = 0):
    """In place on latents; returns (latents, logp [B, T] fp32 device).  PAPER.md:227, Table 2 "SDE window".
    `first_step`: global index of this call's first step (a resumed rollout passes the steps already taken)."""
    B = n_prompts * seeds_per_prompt
    arr, T = _timesteps(timesteps)
    logp = torch.empty((B, T), dtype=torch.float32, device=latents.device)
    ws = ctx.workspace(B, T)
    _check(load_library().spot_dit_denoise_sde(ctx.handle, n_prompts, seeds_per_prompt, _ptr(seeds), _ptr(latents), _ptr(text_emb),
                                               C.cast(arr, C.c_void_p), T, float(noise_level), int(window[0]), int(window[1]),
                                               int(first_step), _ptr(logp), _ptr(ws), ws.numel(), _stream()), "spot_dit_denoise_sde", ctx)
    return latents, logp


def spot_sde_update(x: torch.Tensor, v: torch.Tensor, seeds: torch.Tensor, step: int, t_i: float, t_next: float,
                    noise_level: float):
    """One stochastic step in place on x [B, ...]; returns (x, logp [B])."""
    B = x.shape[0]
    E = x.numel() // B
    logp = torch.empty(B, dtype=torch.float32, device=x.device)
    partials = torch.empty((B, (E + 4095) // 4096), dtype=torch.float32, device=x.device)
    _check(load_library().spot_sde_update(_ptr(x), _ptr(v), _ptr(seeds), step, t_i, t_next, noise_level, B, E, _ptr(logp),
                                          _ptr(partials), _stream()), "spot_sde_update")
    return x, logp


def spot_explore_host(ctx: Context, h_seeds: torch.Tensor, h_text_emb: torch.Tensor, timesteps: Sequence[float],
                      h_probe: torch.Tensor, n_prompts: int, seeds_per_prompt: int, k_select: int, h_out: dict) -> dict:
    """Host-buffer rollout: all tensors are (pinned) HOST tensors; synchronises the stream."""
    arr, T = _timesteps(timesteps)
    ws = ctx.workspace(n_prompts * seeds_per_prompt, T)
    _check(load_library().spot_explore_host(ctx.handle, n_prompts, seeds_per_prompt, _ptr(h_seeds), _ptr(h_text_emb),
                                            C.cast(arr, C.c_void_p), T, _ptr(h_probe), k_select,
                                            _ptr(h_out.get("latents")), _ptr(h_out["rewards"]), _ptr(h_out["stats"]),
                                            _ptr(h_out["top"]), _ptr(h_out["bottom"]), _ptr(ws), ws.numel(), _stream()),
           "spot_explore_host", ctx)
    return h_out


# ---- kernel-level entry points (include/spot_kernels.h) -------------------------------------------
def spot_linear(a: torch.Tensor, w: torch.Tensor, bias: torch.Tensor, epi: int = EPI_BIAS, impl: int = IMPL_AUTO,
                gate: Optional[torch.Tensor] = None, residual: Optional[torch.Tensor] = None,
                out: Optional[torch.Tensor] = None) -> torch.Tensor:
    M, K = a.shape
    N = w.shape[0]
    if epi != EPI_GATE_RESIDUAL and out is None:
        out = torch.empty((M, N), dtype=a.dtype, device=a.device)
    _check(load_library().spot_linear(_dt(w.dtype), impl, epi, _ptr(a), M, K, _ptr(w), N, _ptr(bias), _ptr(gate),
                                      _ptr(residual), _ptr(out), _stream()), "spot_linear")
    return residual if epi == EPI_GATE_RESIDUAL else out


def spot_qkv_rope_linear(a: torch.Tensor, w: torch.Tensor, bias: torch.Tensor, q_gain: torch.Tensor, k_gain: torch.Tensor,
                         cos: torch.Tensor, sin: torch.Tensor, pos_off: int, eps: float) -> torch.Tensor:
    """a [n_seqs, rows_per_seq, K] bf16 -> [n_seqs, rows_per_seq, 3 * hidden] bf16 (QKV projection with K4 fused)."""
    n_seqs, rps, K = a.shape
    hidden = w.shape[0] // 3
    out = torch.empty((n_seqs, rps, 3 * hidden), dtype=a.dtype, device=a.device)
    _check(load_library().spot_qkv_rope_linear(_ptr(a), n_seqs, rps, K, _ptr(w), hidden, _ptr(bias), _ptr(q_gain), _ptr(k_gain),
                                               _ptr(cos), _ptr(sin), pos_off, eps, _ptr(out), _stream()), "spot_qkv_rope_linear")
    return out


def spot_qkv_rope_linear_fp8(a: torch.Tensor, wq: torch.Tensor, w_scale: torch.Tensor, bias: torch.Tensor, q_gain: torch.Tensor,
                             k_gain: torch.Tensor, cos: torch.Tensor, sin: torch.Tensor, pos_off: int, eps: float) -> torch.Tensor:
    """a [n_seqs, rows_per_seq, K] and wq [3 * hidden, K] E4M3 -> [n_seqs, rows_per_seq, 3 * hidden] bf16 (the FP8 rollout's QKV launch)."""
    n_seqs, rps, K = a.shape
    hidden = wq.shape[0] // 3
    out = torch.empty((n_seqs, rps, 3 * hidden), dtype=torch.bfloat16, device=a.device)
    _check(load_library().spot_qkv_rope_linear_fp8(_ptr(a), n_seqs, rps, K, _ptr(wq), _ptr(w_scale), hidden, _ptr(bias), _ptr(q_gain),
                                                   _ptr(k_gain), _ptr(cos), _ptr(sin), pos_off, eps, _ptr(out), _stream()),
           "spot_qkv_rope_linear_fp8")
    return out


def spot_quantize_weight_rows(w: torch.Tensor):
    """bf16 [N, K] -> (E4M3 [N, K], fp32 scale [N]) with s_n = max|W_n| / 448 (DESIGN.md section 13 reading Q2)."""
    N, K = w.shape
    wq = torch.empty((N, K), dtype=torch.float8_e4m3fn, device=w.device)
    scale = torch.empty(N, dtype=torch.float32, device=w.device)
    _check(load_library().spot_quantize_weight_rows(_ptr(w), N, K, _ptr(wq), _ptr(scale), _stream()), "spot_quantize_weight_rows")
    return wq, scale


def spot_quantize_e4m3(x: torch.Tensor) -> torch.Tensor:
    """Unit-scale, saturating, round-to-nearest-even cast to E4M3 (reading Q3)."""
    out = torch.empty(x.shape, dtype=torch.float8_e4m3fn, device=x.device)
    _check(load_library().spot_quantize_e4m3(_dt(x.dtype), _ptr(x), x.numel(), _ptr(out), _stream()), "spot_quantize_e4m3")
    return out


def spot_nvfp4_quantize(x: torch.Tensor, row_scale: Optional[torch.Tensor] = None):
    """bf16 [rows, K] -> (codes uint8 [rows, K / 2], scale-factor atoms uint8 [rows / 128 * K / 64 * 512]) (DESIGN.md section
    13b readings N3 / N4; each row is divided by row_scale[r] first when given).  rows % 128 == 0, K % 64 == 0."""
    rows, K = x.shape
    cb, sb = C.c_size_t(), C.c_size_t()
    _check(load_library().spot_nvfp4_sizes(rows, K, C.byref(cb), C.byref(sb)), "spot_nvfp4_sizes")
    codes = torch.empty((rows, K // 2), dtype=torch.uint8, device=x.device)
    sf = torch.zeros(int(sb.value), dtype=torch.uint8, device=x.device)
    assert codes.numel() == int(cb.value)
    _check(load_library().spot_nvfp4_quantize(_ptr(x), rows, K, _ptr(row_scale), _ptr(codes), _ptr(sf), _stream()), "spot_nvfp4_quantize")
    return codes, sf


def spot_nvfp4_quantize_weight(w: torch.Tensor):
    """bf16 [N, K] -> (codes, scale-factor atoms, fp32 per-row scale s_n = max|W_n| / (6 * 448)) (reading N4)."""
    N, K = w.shape
    scale = torch.empty(N, dtype=torch.float32, device=w.device)
    _check(load_library().spot_nvfp4_row_scale(_ptr(w), N, K, _ptr(scale), _stream()), "spot_nvfp4_row_scale")
    codes, sf = spot_nvfp4_quantize(w, scale)
    return codes, sf, scale


def nvfp4_sf_index(rows: int, K: int) -> torch.Tensor:
    """[rows, K / 16] -> byte offset of the scale factor of (row r, block b) in the atom buffer (layout of csrc/nvfp4.cu)."""
    r = torch.arange(rows).view(-1, 1)
    b = torch.arange(K // 16).view(1, -1)
    return ((r // 128) * (K // 64) + b // 4) * 512 + (r % 32) * 16 + ((r % 128) // 32) * 4 + b % 4


def spot_linear_nvfp4(a_codes: torch.Tensor, a_sf: torch.Tensor, w_codes: torch.Tensor, w_sf: torch.Tensor, w_scale: torch.Tensor,
                      bias: torch.Tensor, epi: int = EPI_BIAS, gate: Optional[torch.Tensor] = None,
                      residual: Optional[torch.Tensor] = None, quantize_out: bool = False):
    """Block-scaled 4-bit Linear on quantised operands; EPI_BIAS / EPI_BIAS_GELU return bf16 [M, N], EPI_GATE_RESIDUAL updates
    `residual` (fp32).  quantize_out (EPI_BIAS_GELU only): the epilogue quantises GELU(y) to NVFP4 and the call returns
    (codes uint8 [M, N / 2], scale-factor atoms) instead - what the rollout's fc1 does."""
    M, K = a_codes.shape[0], a_codes.shape[1] * 2
    N = w_codes.shape[0]
    dev = a_codes.device
    sf_out = None
    if quantize_out:
        cb, sb = C.c_size_t(), C.c_size_t()
        _check(load_library().spot_nvfp4_sizes(M, N, C.byref(cb), C.byref(sb)), "spot_nvfp4_sizes")
        out = torch.empty((M, N // 2), dtype=torch.uint8, device=dev)
        sf_out = torch.zeros(int(sb.value), dtype=torch.uint8, device=dev)
    else:
        out = None if epi == EPI_GATE_RESIDUAL else torch.empty((M, N), dtype=torch.bfloat16, device=dev)
    _check(load_library().spot_linear_nvfp4(epi, _ptr(a_codes), _ptr(a_sf), M, K, _ptr(w_codes), _ptr(w_sf), _ptr(w_scale), N,
                                            _ptr(bias), _ptr(gate), _ptr(residual), _ptr(out), _ptr(sf_out), _stream()), "spot_linear_nvfp4")
    if quantize_out:
        return out, sf_out
    return residual if epi == EPI_GATE_RESIDUAL else out


def spot_linear_fp8(a: torch.Tensor, wq: torch.Tensor, w_scale: torch.Tensor, bias: torch.Tensor, epi: int = EPI_BIAS,
                    gate: Optional[torch.Tensor] = None, residual: Optional[torch.Tensor] = None) -> torch.Tensor:
    """a [M, K] and wq [N, K] E4M3; EPI_BIAS / EPI_BIAS_GELU return E4M3 [M, N], EPI_GATE_RESIDUAL updates `residual` (fp32)."""
    M, K = a.shape
    N = wq.shape[0]
    out = None if epi == EPI_GATE_RESIDUAL else torch.empty((M, N), dtype=torch.float8_e4m3fn, device=a.device)
    _check(load_library().spot_linear_fp8(epi, _ptr(a), M, K, _ptr(wq), N, _ptr(w_scale), _ptr(bias), _ptr(gate), _ptr(residual),
                                          _ptr(out), _stream()), "spot_linear_fp8")
    return residual if epi == EPI_GATE_RESIDUAL else out


def spot_ln_modulate(h: torch.Tensor, shift: torch.Tensor, scale: torch.Tensor, eps: float, dtype: torch.dtype) -> torch.Tensor:
    M, D = h.shape
    out = torch.empty((M, D), dtype=dtype, device=h.device)
    _check(load_library().spot_ln_modulate(_dt(dtype), _ptr(h), M, D, _ptr(shift), _ptr(scale), eps, _ptr(out), _stream()),
           "spot_ln_modulate")
    return out


def spot_qk_norm_rope(qkv: torch.Tensor, n_txt: int, gains: Sequence[torch.Tensor], cos: torch.Tensor, sin: torch.Tensor,
                      eps: float) -> torch.Tensor:
    B, S, three, H, dh = qkv.shape
    assert three == 3
    _check(load_library().spot_qk_norm_rope(_dt(qkv.dtype), _ptr(qkv), B, S, H, dh, n_txt, _ptr(gains[0]), _ptr(gains[1]),
                                            _ptr(gains[2]), _ptr(gains[3]), _ptr(cos), _ptr(sin), eps, _stream()),
           "spot_qk_norm_rope")
    return qkv


def spot_attention(qkv: torch.Tensor, impl: int = IMPL_AUTO) -> torch.Tensor:
    B, S, three, H, dh = qkv.shape
    out = torch.empty((B, S, H * dh), dtype=qkv.dtype, device=qkv.device)
    _check(load_library().spot_attention(_dt(qkv.dtype), impl, _ptr(qkv), _ptr(out), B, S, H, dh, _stream()), "spot_attention")
    return out


def spot_euler_update(x: torch.Tensor, v: torch.Tensor, dt: float, probe: Optional[torch.Tensor] = None):
    B = x.shape[0]
    E = x.numel() // B
    rewards = partials = None
    if probe is not None:
        rewards = torch.empty(B, dtype=torch.float32, device=x.device)
        partials = torch.empty((B, (E + 4095) // 4096), dtype=torch.float32, device=x.device)
    _check(load_library().spot_euler_update(_ptr(x), _ptr(v), dt, B, E, _ptr(probe), _ptr(rewards), _ptr(partials), _stream()),
           "spot_euler_update")
    return x, rewards


STATIC_PARTIALS_MAX = 65536        # include/spot_kernels.h SPOT_STATIC_PARTIALS_MAX


def spot_euler_update_static(x: torch.Tensor, v: torch.Tensor, dt: float, probe: torch.Tensor, rewards: torch.Tensor):
    """spot_euler_update + reward with the library's static scratch: the call allocates nothing; `rewards` [B] fp32 is the
    caller's output buffer."""
    B = x.shape[0]
    E = x.numel() // B
    status = load_library().spot_euler_update_static(_ptr(x), _ptr(v), dt, B, E, _ptr(probe), _ptr(rewards), _stream())
    if status == 5:          # SPOT_ERR_WORKSPACE: rejected before any launch
        raise SpotError(status, f"spot_euler_update_static: n_seqs * ceil(elems / 4096) = {B * ((E + 4095) // 4096)} exceeds the "
                                f"static scratch of {STATIC_PARTIALS_MAX} floats (use spot_euler_update with a caller buffer)")
    _check(status, "spot_euler_update_static")
    return x, rewards


def spot_rope_table(ctx: Context):
    s = ctx.shape
    cos = torch.empty((s.seq, s.head_dim // 2), dtype=torch.float32)
    sin = torch.empty_like(cos)
    _check(load_library().spot_rope_table(ctx.handle, _ptr(cos), _ptr(sin)), "spot_rope_table", ctx)
    return cos, sin


# ---- host bandit planner (include/spot_planner.h) -------------------------------------------------------
class SpotAction(C.Structure):
    _fields_ = [("d", C.c_int32), ("s", C.c_int32)]


def _planner_sigs(lib):
    if getattr(lib, "_planner_ready", False):
        return lib
    vp, i32, dbl = C.c_void_p, C.c_int, C.c_double
    lib.spot_planner_create.argtypes = [C.POINTER(C.c_int32), i32, C.POINTER(C.c_int32), i32, i32, dbl, dbl, i32, C.POINTER(vp)]
    lib.spot_planner_destroy.argtypes = [vp]
    lib.spot_planner_eligible.argtypes = [vp, dbl, dbl, C.POINTER(SpotAction), i32, C.POINTER(i32)]
    lib.spot_planner_select.argtypes = [vp, dbl, dbl, C.POINTER(SpotAction), C.POINTER(dbl)]
    lib.spot_planner_feedback.argtypes = [C.POINTER(C.c_float), i32, C.POINTER(C.c_float), i32, C.POINTER(dbl)]
    lib.spot_planner_update.argtypes = [vp, SpotAction, dbl]
    lib.spot_planner_stats.argtypes = [vp, SpotAction, C.POINTER(dbl), C.POINTER(i32), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    for n in ("create", "destroy", "eligible", "select", "feedback", "update", "stats"):
        getattr(lib, "spot_planner_" + n).restype = C.c_int
    lib._planner_ready = True
    return lib


class Planner:
    """spot_planner: UCB exploration planner (host code in libspot.so; argument marshalling only here)."""

    def __init__(self, d_values, s_values, n_prompts: int, t_step: float, beta: float = 0.5, window: int = 8):
        lib = _planner_sigs(load_library())
        d = (C.c_int32 * len(d_values))(*d_values)
        s = (C.c_int32 * len(s_values))(*s_values)
        h = C.c_void_p()
        _check(lib.spot_planner_create(d, len(d_values), s, len(s_values), n_prompts, t_step, beta, window, C.byref(h)),
               "spot_planner_create")
        self.handle, self._n = h, len(d_values) * len(s_values)

    def __del__(self):
        if getattr(self, "handle", None):
            load_library().spot_planner_destroy(self.handle)
            self.handle = None

    def spot_planner_eligible(self, t_train: float, n_spot: float):
        out = (SpotAction * self._n)()
        n = C.c_int()
        _check(load_library().spot_planner_eligible(self.handle, t_train, n_spot, out, self._n, C.byref(n)), "spot_planner_eligible")
        return [(out[i].d, out[i].s) for i in range(n.value)]

    def spot_planner_select(self, t_train: float, n_spot: float):
        a, u = SpotAction(), C.c_double()
        _check(load_library().spot_planner_select(self.handle, t_train, n_spot, C.byref(a), C.byref(u)), "spot_planner_select")
        return (a.d, a.s), u.value

    def spot_planner_update(self, action, r: float) -> None:
        _check(load_library().spot_planner_update(self.handle, SpotAction(*action), r), "spot_planner_update")

    def spot_planner_stats(self, action):
        m, n, ni, nt = C.c_double(), C.c_int(), C.c_int64(), C.c_int64()
        _check(load_library().spot_planner_stats(self.handle, SpotAction(*action), C.byref(m), C.byref(n), C.byref(ni), C.byref(nt)),
               "spot_planner_stats")
        return {"mean": m.value, "n_i": n.value, "N_i": ni.value, "N": nt.value}


def spot_planner_feedback(sigma_cov, sigma_unc) -> float:
    lib = _planner_sigs(load_library())
    a = (C.c_float * max(1, len(sigma_cov)))(*sigma_cov)
    b = (C.c_float * max(1, len(sigma_unc)))(*sigma_unc)
    r = C.c_double()
    _check(lib.spot_planner_feedback(a, len(sigma_cov), b, len(sigma_unc), C.byref(r)), "spot_planner_feedback")
    return r.value
