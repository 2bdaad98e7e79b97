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
@pytest.mark.parametrize("M,N,K", [(128, 256, 256), (256, 512, 1024), (384, 256, 3072), (1280, 768, 512), (256, 384, 512),
                                   (512, 3072, 768), (384, 768, 512), (128, 384, 2048), (768, 384, 3072)])
def test_linear_nvfp4(epi, M, N, K):
    """kind::mxf4nvf4 block-scaled GEMM vs the oracle on the SAME codes: single tile, several K blocks (ring wrap), several
    tiles per CTA; N = 256 / 512 take the 128 x 256 tiles (one accumulator), N = 768 / 384 / 3072 the 192-column tiles
    (two accumulators; odd tiles start 64 rows into a scale atom): CTA pairs on 256 x 192 where M is a multiple of 256
    (M = 256, 512, 768, 1280), the one-CTA 128 x 192 kernel otherwise (M = 384, 128).  fp32 accumulation of exactly representable products; bf16
    outputs add one rounding."""
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


@pytest.mark.parametrize("M,N,K", [(256, 768, 512), (128, 512, 256), (384, 3072, 1024)])
def test_linear_nvfp4_fused_gelu_quantiser(M, N, K):
    """fc1's epilogue in the rollout: bias -> tanh-GELU -> NVFP4 codes + scales without ever storing u.  The oracle
    quantises its own exact u; the CUDA side quantises tanh.approx-GELU of an fp32-accumulated value, so a code is allowed
    to land on the NEIGHBOURING E2M1 value where u / sf sits within that difference of a rounding boundary: >= 99 % of the
    codes identical, none further than one grid step away, block scales identical or adjacent E4M3 values."""
    a = hash_normal(1130, M * K, 1.0, torch.bfloat16, "cuda").reshape(M, K)
    w = hash_normal(1131, N * K, 0.05, torch.bfloat16, "cuda").reshape(N, K)
    b = hash_normal(1132, N, 0.1, torch.bfloat16, "cuda")
    ac, asf = spot.spot_nvfp4_quantize(a)
    wc, wsf, ws = spot.spot_nvfp4_quantize_weight(w)
    codes, sf = spot.spot_linear_nvfp4(ac, asf, wc, wsf, ws, b, spot.EPI_BIAS_GELU, quantize_out=True)
    got_q, got_sf = _unpack(codes, sf, M, N)
    wq, wsf64, s64 = nvfp4.quantize_weight(np64(w))
    u = mmdit.gelu_tanh(nvfp4.linear_nvfp4(np64(a), wq, wsf64, s64, np64(b)))
    ref_q, ref_sf = nvfp4.quantize_rows(u)
    grid = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0])
    step = lambda v: np.searchsorted(grid, np.abs(v)) * np.sign(v)                # signed position on the E2M1 grid
    same_sf = (got_sf == ref_sf).mean()
    cmp = got_sf == ref_sf                                                        # compare codes where the block scale agrees
    m = np.repeat(cmp, 16, axis=1)
    same = (got_q[m] == ref_q[m]).mean()
    far = np.abs(step(got_q[m]) - step(ref_q[m])).max()
    deq = rel_l2(nvfp4.dequantize(got_q, got_sf), nvfp4.dequantize(ref_q, ref_sf))
    print(f"fused GELU->NVFP4 M={M} N={N} K={K}: scales identical {same_sf:.4f}, codes identical {same:.4f} (max grid distance {far:.0f}), "
          f"dequantised rel-L2 {deq:.3e}")
    assert same_sf > 0.99 and same > 0.99 and far <= 1
    assert np.abs(np.log2(np.where((got_sf > 0) & (ref_sf > 0), got_sf / np.where(ref_sf > 0, ref_sf, 1), 1.0))).max() <= 0.25   # adjacent E4M3 values at most
    assert deq < 3e-2
    # the two-step path (u rounded to bf16, then the quantiser kernel) differs from the fused one by the code flips that one
    # bf16 rounding (2^-9) of the quantiser's input causes - measured 3.3e-2 here, in line with the amplification the oracle
    # test measures; the fused epilogue is the one that matches the oracle
    u_bf = spot.spot_linear_nvfp4(ac, asf, wc, wsf, ws, b, spot.EPI_BIAS_GELU)
    c2, s2 = spot.spot_nvfp4_quantize(u_bf)
    q2, sf2 = _unpack(c2, s2, M, N)
    assert rel_l2(nvfp4.dequantize(q2, sf2), nvfp4.dequantize(got_q, got_sf)) < 6e-2
    again = spot.spot_linear_nvfp4(ac, asf, wc, wsf, ws, b, spot.EPI_BIAS_GELU, quantize_out=True)
    assert torch.equal(again[0], codes) and torch.equal(again[1], sf)


def test_nvfp4_argument_errors():
    x = torch.zeros((100, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(spot.SpotError):
        spot.spot_nvfp4_quantize(x)                        # rows % 128
    with pytest.raises(spot.SpotError):
        spot.spot_nvfp4_quantize(torch.zeros((128, 48), dtype=torch.bfloat16, device="cuda"))   # K % 64


# ------------------------------------------------------------------ the variant inside the block and the rollout
@pytest.fixture(scope="module")
def wide():
    """Config-3 shapes (hidden 3072, 24 x 128 heads, 1024 + 256 tokens) at depth 2."""
    from synth import CONFIGS
    from tests.gpu_common import device_weights
    s = CONFIGS[3].with_(n_blocks=2, seeds_per_prompt=4, n_steps=3)
    w = device_weights(s)
    ctx = spot.Context(s, w, max_seqs=4)
    return s, w, ctx


def test_block_forward_nvfp4_matches_nvfp4_oracle(wide):
    """One full-width block with fc1 / fc2 in NVFP4 and QKV / out-proj in FP8 against oracle/nvfp4.py.
    Parity criterion of the 4-bit variant (N6).  The kernels are exact on identical inputs (tests
    above: codes bit for bit, GEMM 3e-8).  Composed, the two sides quantise values that differ by 1e-3 .. 1e-2 (bf16
    roundings of y2 and u, E4M3 code flips upstream), and a 4-bit quantiser turns such a difference into a DIFFERENT
    rounding of every value near a code boundary: tests/test_oracle_nvfp4.py measures on the oracle alone that an input
    perturbation of 2e-3 / 1e-2 moves one NVFP4 Linear's output by 2.8e-2 / 6.2e-2 (its quantisation noise is 1.3e-1).
    A per-block 2e-2 is therefore not a property any implementation can have; the criterion is that the CUDA path is
    closer to the oracle's variant than the variant is to the exact model (ratio <= 0.75), and the rank fidelity below."""
    from synth import make_block_inputs
    from tests.gpu_common import oracle_weights
    s, w, ctx = wide
    h_img, h_txt, temb = make_block_inputs(s, 2, "cuda")
    _, blocks = oracle_weights(w)
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    c = mmdit.silu(np64(temb))
    b_img, b_txt = spot.spot_dit_block_forward(ctx, 0, h_img, h_txt, temb)          # bf16 path
    b_img, b_txt = b_img.clone(), b_txt.clone()
    ctx.enable_nvfp4(True)
    try:
        o_img, o_txt = spot.spot_dit_block_forward(ctx, 0, h_img, h_txt, temb)
        o_img, o_txt = o_img.clone(), o_txt.clone()
        again, _ = spot.spot_dit_block_forward(ctx, 0, h_img, h_txt, temb)
        assert torch.equal(again, o_img)
    finally:
        ctx.enable_nvfp4(False)
    back, _ = spot.spot_dit_block_forward(ctx, 0, h_img, h_txt, temb)
    assert torch.equal(back, b_img)                                                  # switching off restores the bf16 path
    qw = nvfp4.quantize_block(blocks[0])
    for b in range(2):
        r_img, r_txt = nvfp4.block_forward_nvfp4(np64(h_img[b]), np64(h_txt[b]), c, blocks[0], qw, n_heads=s.n_heads, cos=cos, sin=sin)
        e_i, e_t = rel_l2(np64(o_img[b]), r_img), rel_l2(np64(o_txt[b]), r_txt)
        d_i = rel_l2(np64(o_img[b]), np64(b_img[b]))
        u_i = rel_l2(np64(o_img[b]) - np64(h_img[b]), r_img - np64(h_img[b]))
        print(f"nvfp4 block, sequence {b}: vs nvfp4 oracle img {e_i:.3e} txt {e_t:.3e} (update {u_i:.3e}); nvfp4 vs bf16 path img {d_i:.3e}")
        d_t = rel_l2(np64(o_txt[b]), np64(b_txt[b]))
        assert e_i < 0.75 * d_i and e_t < 0.75 * d_t
        assert 1e-3 < d_i < 0.25                                                     # 4-bit quantisation is visible, and bounded


def test_rollout_nvfp4_matches_oracle_and_ranks_like_bf16(wide):
    from oracle import philox, rollout
    from synth import make_probe, make_text_emb
    from tests.gpu_common import oracle_weights
    s, w, ctx = wide
    text, probe = make_text_emb(s, "cuda"), make_probe(s, "cuda")
    ts = [float(np.float32(t)) for t in s.timesteps]
    seeds = torch.tensor([0, 1, 2, 3], dtype=torch.int64, device="cuda")
    ref_bf16 = spot.spot_explore(ctx, seeds, text, ts, probe, 1, 4, 2)
    lat_b, rew_b = ref_bf16["latents"].clone(), ref_bf16["rewards"].clone()
    ctx.enable_nvfp4(True)
    try:
        out = spot.spot_explore(ctx, seeds, text, ts, probe, 1, 4, 2)
        lat_q, rew_q = out["latents"].clone(), out["rewards"].clone()
        again = spot.spot_explore(ctx, seeds, text, ts, probe, 1, 4, 2)
        assert torch.equal(again["latents"], lat_q)                          # deterministic
        alone = spot.spot_explore(ctx, seeds[2:3].contiguous(), text, ts, probe, 1, 1, 0)
        assert torch.equal(alone["latents"][0], lat_q[2])                    # batch-independent (per-row block scales)
    finally:
        ctx.enable_nvfp4(False)
    g, blocks = oracle_weights(w)
    qblocks = [nvfp4.quantize_block(bw) for bw in blocks]
    cos, sin = mmdit.rope_table(s.grid_h, s.grid_w, s.n_txt, s.rope_pairs, s.rope_theta)
    h_txt0 = mmdit.text_input(np64(text)[0], g)
    x0 = philox.noise_from_seeds([0], s.n_img * s.latent_ch)[0].reshape(s.n_img, s.latent_ch).astype(np.float32).astype(np.float64)
    xT = rollout.euler_denoise(x0, ts, lambda x, t: nvfp4.dit_velocity_nvfp4(x, t, h_txt0, g, blocks, qblocks, n_heads=s.n_heads, cos=cos, sin=sin))
    e = rel_l2(np64(lat_q[0]), xT)
    e_upd = rel_l2(np64(lat_q[0]) - x0, xT - x0)
    d = rel_l2(np64(lat_q), np64(lat_b))
    print(f"nvfp4 rollout (depth 2, 3 steps): vs nvfp4 oracle {e:.3e} (x_T - x_0: {e_upd:.3e}); nvfp4 vs bf16 latents {d:.3e}; "
          f"rewards nvfp4 {rew_q.tolist()} bf16 {rew_b.tolist()}")
    assert e < d and d < 0.15                    # criterion N6: closer to the oracle's variant than the variant is to bf16
    assert torch.argsort(rew_q).tolist() == torch.argsort(rew_b).tolist()           # and the seeds rank as under bf16


def test_nvfp4_needs_fp8_and_preparation(wide):
    s, w, ctx = wide
    fresh = spot.Context(s, w, max_seqs=4)
    with pytest.raises(spot.SpotError):
        spot.spot_set_option(fresh, spot.OPT_NVFP4, 1)       # neither FP8 nor the prepared weights
    ctx.enable_nvfp4(True)
    big = spot.spot_workspace_bytes(ctx, 4, 3)
    ctx.enable_fp8(False)                                    # switching the FP8 variant off takes the 4-bit MLP with it
    assert spot.spot_workspace_bytes(ctx, 4, 3) < big        # the quantised activations live in the workspace
    with pytest.raises(spot.SpotError):
        spot.spot_set_option(ctx, spot.OPT_NVFP4, 1)         # not without SPOT_OPT_FP8
    ctx.enable_nvfp4(False)
