"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol the headers
declare, and rejects bad arguments with the documented codes before touching a device."""
import ctypes as C
import os
import re

import pytest
import torch

import paper_2606_19004_b200 as spot
from paper_2606_19004_b200 import binding, build as spot_build
from synth import CONFIGS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    spot_build.build()
    return spot.load_library()


def test_exports_every_declared_symbol(lib):
    declared = set()
    for hdr in ("spot.h", "spot_kernels.h", "spot_planner.h"):
        text = open(os.path.join(ROOT, "include", hdr)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        declared |= set(re.findall(r"\b(spot_[a-z0-9_]+)\s*\(", text))
    assert {"spot_noise_from_seeds", "spot_dit_block_forward", "spot_dit_denoise", "spot_seed_rewards"} <= declared
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/ but not exported"
    assert spot.spot_version().startswith("libspot")
    assert lib.spot_status_string(2).decode().startswith("SPOT_ERR_SHAPE")


def test_option_constants_match_the_header():
    """The binding's OPT_* integers are the values of `spot_option` in include/spot.h."""
    text = open(os.path.join(ROOT, "include", "spot.h")).read()
    enum = dict((k, int(v)) for k, v in re.findall(r"\b(SPOT_OPT_[A-Z0-9_]+)\s*=\s*(\d+)", text))
    assert len(enum) >= 5
    for name, value in enum.items():
        assert getattr(binding, name[len("SPOT_"):]) == value, name


def test_static_scratch_limit_matches_the_header():
    """binding.STATIC_PARTIALS_MAX is SPOT_STATIC_PARTIALS_MAX of include/spot_kernels.h (spot_euler_update_static)."""
    text = open(os.path.join(ROOT, "include", "spot_kernels.h")).read()
    m = re.search(r"#define\s+SPOT_STATIC_PARTIALS_MAX\s+(\d+)", text)
    assert m and int(m.group(1)) == binding.STATIC_PARTIALS_MAX == 65536


def _cfg_struct(s, **over):
    kw = dict(n_blocks=s.n_blocks, hidden=s.hidden, n_heads=s.n_heads, head_dim=s.head_dim, mlp_hidden=s.mlp_hidden,
              grid_h=s.grid_h, grid_w=s.grid_w, n_txt=s.n_txt, latent_ch=s.latent_ch, txt_dim=s.txt_dim,
              rope_pairs=(C.c_int32 * 3)(*s.rope_pairs), rope_theta=s.rope_theta, ln_eps=s.ln_eps, rms_eps=s.rms_eps, dtype=0)
    kw.update(over)
    return binding.SpotConfig(**kw)


def test_create_rejects_bad_arguments(lib):
    s = CONFIGS[1]
    h = C.c_void_p()
    w = binding.SpotWeights()
    assert lib.spot_create(None, C.byref(w), 1, C.byref(h)) == 1                      # NULL
    assert lib.spot_create(C.byref(_cfg_struct(s, n_heads=3)), C.byref(w), 1, C.byref(h)) == 2      # H*d_h != D
    assert lib.spot_create(C.byref(_cfg_struct(s, rope_pairs=(C.c_int32 * 3)(4, 14, 13))), C.byref(w), 1, C.byref(h)) == 2
    assert lib.spot_create(C.byref(_cfg_struct(s, dtype=5)), C.byref(w), 1, C.byref(h)) == 3        # dtype
    assert lib.spot_create(C.byref(_cfg_struct(s)), C.byref(w), 0, C.byref(h)) == 2                 # max_seqs
    assert lib.spot_create(C.byref(_cfg_struct(s)), C.byref(w), 4, C.byref(h)) == 1                 # NULL weights
    assert h.value is None


def test_noise_rejects_bad_arguments(lib):
    buf = torch.zeros(64, dtype=torch.float32)
    seeds = torch.zeros(2, dtype=torch.int64)
    f = lib.spot_noise_from_seeds
    assert f(seeds.data_ptr(), 2, 6, 0, buf.data_ptr(), None) == 2           # not a multiple of 4
    assert f(seeds.data_ptr(), -1, 8, 0, buf.data_ptr(), None) == 2
    assert f(seeds.data_ptr(), 0, 8, 0, None, None) == 0                     # empty input is a no-op
    assert f(None, 2, 8, 0, buf.data_ptr(), None) == 1
    assert f(seeds.data_ptr(), 2, 8, 0, buf.data_ptr() + 4, None) == 4       # misaligned
    if not torch.cuda.is_available():
        assert f(seeds.data_ptr(), 2, 8, 0, buf.data_ptr(), None) == 6       # no device: fail loudly, no CPU fallback


def test_kernel_calls_reject_bad_arguments(lib):
    t = torch.zeros(1024, dtype=torch.float32)
    p = t.data_ptr()
    assert lib.spot_linear(7, 0, 0, p, 4, 16, p, 4, p, None, None, p, None) == 3
    assert lib.spot_linear(0, 0, 0, p, 4, 16, p, 4, p, None, None, None, None) == 1
    assert lib.spot_linear(0, 0, 2, p, 4, 16, p, 4, p, None, None, p, None) == 1       # gate/residual missing
    assert lib.spot_linear(0, 0, 0, p, 0, 16, p, 4, p, None, None, p, None) == 0       # M = 0
    assert lib.spot_ln_modulate(0, p, 4, 100, p, p, 1e-6, p, None) == 2                # D % 128
    assert lib.spot_attention(0, 0, p, p, 1, 8, 1, 48, None) == 2                      # head_dim
    assert lib.spot_euler_update(p, p, 0.1, 1, 6, None, None, None, None) == 2
    f = lib.spot_euler_update_static                                                  # the no-allocation variant (static scratch)
    assert f(p, p, 0.1, 1, 6, p, p, None) == 2                                         # elems % 4
    assert f(p, p, 0.1, 70000, 8, p, p, None) == 2                                     # sequences ride on gridDim.y
    assert f(p, p, 0.1, 1, 8, None, p, None) == 1                                      # probe and rewards are required
    assert f(p, p, 0.1, 40000, 8192, p, p, None) == 5                                  # 80000 partial sums > 65536: rejected before any launch
    assert f(p, p, 0.1, 0, 8, p, p, None) == 0
    if not torch.cuda.is_available():
        assert lib.spot_ln_modulate(0, p, 4, 128, p, p, 1e-6, p, None) == 6


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", str(tmp_path / "libspot.so"))
    with pytest.raises(FileNotFoundError):
        binding.load_library()
