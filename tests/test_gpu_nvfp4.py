"""-m gpu parity of the NVFP4 exploration variant against oracle/nvfp4.py.

Quantisers: codes and scale factors are integers decided by floating point - both sides form every deciding value in fp32
with IEEE division, so they are compared BIT FOR BIT.  Block-scaled GEMM: the same codes on both sides, so the only GPU
error is the accumulation (fp32 with the tensor core's internal alignment) and one bf16 output rounding."""
import numpy as np
import pytest
import torch

import paper_2606_19004_b200 as spot
from oracle import mmdit, nvfp4
from synth import hash_normal
from tests.gpu_common import ensure_built
from tests.helpers import BF16_U, elem_excess, np64, rel_l2

pytestmark = pytest.mark.gpu
E2M1 = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0, -0.0, -0.5, -1.0, -1.5, -2.0, -3.0, -4.0, -6.0])   # code -> value (OCP MX)


@pytest.fixture(scope="module", autouse=True)
def _lib():
    ensure_built()


def _unpack(codes, sf, rows, K):
    """Device buffers -> (E2M1 values [rows, K], E4M3 scales [rows, K / 16]) as fp64."""
    c = codes.cpu().numpy()
    vals = np.empty((rows, K))
    vals[:, 0::2] = E2M1[c & 15]                # element k even: low nibble
    vals[:, 1::2] = E2M1[c >> 4]
    idx = spot.nvfp4_sf_index(rows, K)
    sfv = sf.cpu()[idx.reshape(-1)].view(torch.float8_e4m3fn).to(torch.float64).numpy().reshape(rows, K // 16)
    return vals, sfv


@pytest.mark.parametrize("rows,K,scale", [(128, 64, 1.0), (256, 3072, 1.0), (384, 256, 30.0), (128, 12288, 0.01)])
def test_quantize_rows_bit_exact(rows, K, scale):
    x = hash_normal(1101, rows * K, scale, torch.bfloat16, "cuda").reshape(rows, K)
    x[5, 16:32] = 0                                                          # a zero block
    x[7, :16] = torch.tensor([3.0, -1.5, 0.75, 0.5, 0.25, 0.1, 0.0, -3.0, 2.0, 1.0, 0.6, 0.4, 2.9, 2.2, -0.13, 1.3])   # ties
    codes, sf = spot.spot_nvfp4_quantize(x)
    got_q, got_sf = _unpack(codes, sf, rows, K)
    ref_q, ref_sf = nvfp4.quantize_rows(np64(x))
    assert (got_sf == ref_sf).all()
    assert (got_q == ref_q).all()                                            # every one of the rows * K codes
    assert got_sf[5, 1] == 0 and (got_q[5, 16:32] == 0).all()


def test_quantize_weight_bit_exact():
    N, K = 256, 512
    w = hash_normal(1102, N * K, 0.02, torch.bfloat16, "cuda").reshape(N, K)
    w[9] = 0
    codes, sf, s = spot.spot_nvfp4_quantize_weight(w)
    got_q, got_sf = _unpack(codes, sf, N, K)
    ref_q, ref_sf, ref_s = nvfp4.quantize_weight(np64(w))
    assert (np64(s) == ref_s).all() and s[9].item() == 1.0
    assert (got_sf == ref_sf).all() and (got_q == ref_q).all()


def _linear_case(M, N, K, tid, epi):
    a = hash_normal(tid, M * K, 1.0, torch.bfloat16, "cuda").reshape(M, K)
    w = hash_normal(tid + 1, N * K, 0.05, torch.bfloat16, "cuda").reshape(N, K)
    b = hash_normal(tid + 2, N, 0.1, torch.bfloat16, "cuda")
    gate = hash_normal(tid + 3, N, 0.5, torch.float32, "cuda")
    resid = hash_normal(tid + 4, M * N, 1.0, torch.float32, "cuda").reshape(M, N)
    ac, asf = spot.spot_nvfp4_quantize(a)
    wc, wsf, ws = spot.spot_nvfp4_quantize_weight(w)
    wq, wsf64, s64 = nvfp4.quantize_weight(np64(w))
    ref = nvfp4.linear_nvfp4(np64(a), wq, wsf64, s64, np64(b))
    if epi == spot.EPI_BIAS_GELU:
        ref = mmdit.gelu_tanh(ref)
    if epi == spot.EPI_GATE_RESIDUAL:
        ref = np64(resid) + np64(gate) * ref
        out = spot.spot_linear_nvfp4(ac, asf, wc, wsf, ws, b, epi, gate=gate, residual=resid.clone())
    else:
        out = spot.spot_linear_nvfp4(ac, asf, wc, wsf, ws, b, epi)
    exact = np64(a) @ np64(w).T + np64(b)
    return np64(out), ref, exact


@pytest.mark.parametrize("epi", [0, 1, 2])
@pytest.mark.parametrize("M,N,K", [(128, 256, 256), (256, 512, 1024), (384, 256, 3072), (1280, 768, 512)])
def test_linear_nvfp4(epi, M, N, K):
    """kind::mxf4nvf4 block-scaled GEMM vs the oracle on the SAME codes: single tile, several K blocks (ring wrap), several
    tiles per CTA.  fp32 accumulation of exactly representable products; bf16 outputs add one rounding."""
    got, ref, exact = _linear_case(M, N, K, 1110, epi)
    err = rel_l2(got, ref)
    print(f"nvfp4 linear M={M} N={N} K={K} epi={epi}: rel-L2 vs nvfp4 oracle {err:.3e}")
    if epi == spot.EPI_GATE_RESIDUAL:
        assert err < 2e-5 and elem_excess(got, ref, 2e-5, 2e-5) <= 1.0
    else:
        assert err < 4e-3
        assert elem_excess(got, ref, 1.05 * BF16_U, 4e-3 if epi == spot.EPI_BIAS_GELU else 1e-4) <= 1.0
    if epi == spot.EPI_BIAS:
        assert 0.05 < rel_l2(got, exact) < 0.25            # and the quantisation itself is what oracle/nvfp4.py says it is
    again = _linear_case(M, N, K, 1110, epi)[0]
    assert (again == got).all()                            # deterministic


def test_nvfp4_argument_errors():
    x = torch.zeros((100, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(spot.SpotError):
        spot.spot_nvfp4_quantize(x)                        # rows % 128
    with pytest.raises(spot.SpotError):
        spot.spot_nvfp4_quantize(torch.zeros((128, 48), dtype=torch.bfloat16, device="cuda"))   # K % 64
