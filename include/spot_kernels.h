/* spot_kernels.h - kernel-level entry points of libspot.so.
 *
 * The four north-star calls live in spot.h.  The calls below expose the individual kernels of the
 * hot path so that the tests can compare each one with the oracle and
 * bench.py can time each one against its roofline.  Same conventions as spot.h: device pointers,
 * row-major, caller-owned buffers, asynchronous on `cuda_stream`, no CPU fallback.
 */
#ifndef SPOT_KERNELS_H_
#define SPOT_KERNELS_H_

#include "spot.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { SPOT_EPI_BIAS = 0, SPOT_EPI_BIAS_GELU = 1, SPOT_EPI_GATE_RESIDUAL = 2 } spot_epilogue;
typedef enum {
  SPOT_IMPL_AUTO = 0,
  SPOT_IMPL_SIMT = 1,
  SPOT_IMPL_TCGEN05 = 2,       /* one CTA per 128 x 256 tile (cta_group::1) */
  SPOT_IMPL_TCGEN05_2CTA = 3,  /* CTA pair per 256 x 256 tile (cta_group::2), per-thread global epilogue; GEMM only */
  SPOT_IMPL_TCGEN05_TMA = 4    /* CTA pair + shared-memory staged TMA store / reduce-add epilogue (what AUTO picks); GEMM only */
} spot_impl;

/* Linear layer y = x W^T + b with a fused epilogue (north_star (b); S4 steps 3, 7, 8).
 *   d_a [M, K], d_w [N, K], d_bias [N] of `dtype`.
 *   SPOT_EPI_BIAS:          d_out [M, N] (dtype)  = y
 *   SPOT_EPI_BIAS_GELU:     d_out [M, N] (dtype)  = GELU_tanh(y)
 *   SPOT_EPI_GATE_RESIDUAL: d_residual [M, N] fp32 += d_gate[N] (fp32) * y    (d_out unused)
 * SPOT_IMPL_TCGEN05 requires dtype bf16, K % 8 == 0, N % 32 == 0 and returns SPOT_ERR_SHAPE otherwise;
 * SPOT_IMPL_SIMT requires K % 16 == 0. */
spot_status spot_linear(spot_dtype dtype, spot_impl impl, spot_epilogue epi, const void *d_a, int64_t M, int64_t K,
                        const void *d_w, int64_t N, const void *d_bias, const float *d_gate, float *d_residual,
                        void *d_out, void *cuda_stream);

/* The QKV projection with K4 fused into its epilogue (north_star (b) + (c); S4 steps 3-5), one stream:
 *   d_out [n_seqs * rows_per_seq, 3 * hidden] bf16 = [ RoPE(RMSNorm(q) * q_gain) | RoPE(RMSNorm(k) * k_gain) | v ],
 *   [q | k | v] = d_a [n_seqs * rows_per_seq, K] d_w[3 * hidden, K]^T + d_bias, heads of 128 columns; row r of a
 *   sequence is rotated by row pos_off + r of d_cos / d_sin [S, 64] fp32 (S >= pos_off + rows_per_seq).
 * bf16 only; hidden % 128 == 0, K % 8 == 0; gains [128] bf16.  Errors as spot_linear. */
spot_status spot_qkv_rope_linear(const void *d_a, int n_seqs, int rows_per_seq, int64_t K, const void *d_w, int64_t hidden,
                                 const void *d_bias, const void *d_q_gain, const void *d_k_gain, const float *d_cos,
                                 const float *d_sin, int pos_off, float eps, void *d_out, void *cuda_stream);

/* y = LayerNorm(h) * (1 + scale) + shift over the last axis, biased variance, no affine (S4
 * step 2).  d_h [M, D] fp32 (residual stream), d_shift/d_scale [D] fp32, d_out [M, D] of `dtype`.
 * D must be 128 * {1,2,4,8,12,16,24,32}.  dtype SPOT_E4M3 writes E4M3 bytes (unit scale, saturating). */
spot_status spot_ln_modulate(spot_dtype dtype, const float *d_h, int64_t M, int64_t D, const float *d_shift,
                             const float *d_scale, float eps, void *d_out, void *cuda_stream);

/* In place on d_qkv [B, S, 3, H, d_h]: q <- RoPE(RMSNorm(q) * gain), k likewise; v untouched (north_star (c);
 * DESIGN.md S4 steps 4-5).  Tokens s < n_txt use the text gains.  d_cos/d_sin [S, d_h/2] fp32. */
spot_status spot_qk_norm_rope(spot_dtype dtype, void *d_qkv, int B, int S, int H, int head_dim, int n_txt,
                              const void *d_q_gain_img, const void *d_k_gain_img, const void *d_q_gain_txt,
                              const void *d_k_gain_txt, const float *d_cos, const float *d_sin, float eps,
                              void *cuda_stream);

/* O = softmax(Q K^T / sqrt(d_h)) V over all S keys per (sequence, head), no mask (north_star (d); DESIGN.md
 * S4 step 6).  d_qkv [B, S, 3, H, d_h] -> d_out [B, S, H * d_h], both `dtype`.  SPOT_IMPL_TCGEN05 requires
 * bf16, d_h = 128 (one-pass kernel, 64-key tiles); for this call SPOT_IMPL_TCGEN05_2CTA selects the previous two-pass
 * tcgen05 kernel (128-key tiles), kept for A/B timing. */
spot_status spot_attention(spot_dtype dtype, spot_impl impl, const void *d_qkv, void *d_out, int B, int S, int H,
                           int head_dim, void *cuda_stream);

/* x <- x + dt * v over [n_seqs, elems] fp32 (north_star (e); S8).  If d_probe != NULL also
 * d_rewards[b] = <probe, x_b> / sqrt(elems) with d_partials [n_seqs, ceil(elems / 4096)] fp32 scratch. */
spot_status spot_euler_update(float *d_x, const float *d_v, float dt, int n_seqs, int64_t elems, const float *d_probe,
                              float *d_rewards, float *d_partials, void *cuda_stream);

/* spot_euler_update with the reward, for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same kernels, same results bit for bit, but the partial-sum scratch is a
 * static __device__ array inside the library (SPOT_STATIC_PARTIALS_MAX floats = 256 KiB, held by every GPU that loads the
 * library until the process exits) instead of a caller buffer.  The call allocates nothing (no cudaMalloc / cudaFree).
 *   d_x [n_seqs, elems] fp32 updated in place, d_v [n_seqs, elems], d_probe [elems], d_rewards [n_seqs] out; all required.
 *   n_seqs * ceil(elems / 4096) > SPOT_STATIC_PARTIALS_MAX -> SPOT_ERR_WORKSPACE, nothing launched (n_seqs <= 65535 and
 *   elems % 4 == 0 as for spot_euler_update, else SPOT_ERR_SHAPE).
 * The first call on a device looks the array's address up (cudaGetSymbolAddress, with that device current) and must be
 * made outside stream capture; later calls are capture-safe.  All calls on a device share the array, which keeps the last
 * call's partial sums: two calls that overlap on the GPU (different streams, no dependency) race on it - serialise them.
 * Nothing needs clearing between calls (every slot is written before it is read). */
#define SPOT_STATIC_PARTIALS_MAX 65536
spot_status spot_euler_update_static(float *d_x, const float *d_v, float dt, int n_seqs, int64_t elems, const float *d_probe,
                                     float *d_rewards, void *cuda_stream);

/* A7 alone: per-prompt statistics and top/bottom-k selection of rewards that are already on the device (spot.h
 * spot_seed_rewards states the ordering rules).  This is the step every rank repeats after the all-gather of the reward
 * shards in the multi-GPU path.  d_rewards [n_prompts * seeds_per_prompt] fp32; d_stats
 * [n_prompts, 2]; d_top / d_bottom [n_prompts, k_select] int32 (may be NULL when k_select == 0).
 * 0 <= 2 * k_select <= seeds_per_prompt <= 1024, else SPOT_ERR_SHAPE. */
spot_status spot_select_seeds(const float *d_rewards, int n_prompts, int seeds_per_prompt, int k_select, float *d_stats,
                              int32_t *d_top, int32_t *d_bottom, void *cuda_stream);

/* One stochastic sampler step on [n_seqs, elems] fp32 (spot.h spot_dit_denoise_sde): x <- mean +
 * sigma sqrt(-dt) xi with xi from Philox stream 256 + step of d_seeds[b]; d_logp[b] = the step's log-probability.
 * noise_level == 0 degenerates to the Euler update (d_logp = 0).  d_partials: [n_seqs, ceil(elems / 4096)] fp32 scratch. */
spot_status spot_sde_update(float *d_x, const float *d_v, const uint64_t *d_seeds, int step, float t_i, float t_next,
                            float noise_level, int n_seqs, int64_t elems, float *d_logp, float *d_partials,
                            void *cuda_stream);

/* FP8 (E4M3) building blocks of the low-precision exploration variant (spot.h).
 * spot_quantize_weight_rows: d_w_bf16 [N, K] bf16 -> d_wq [N, K] E4M3 bytes and d_scale [N] fp32 (s_n = max|W_n| / 448).
 * spot_quantize_e4m3: elementwise e4m3(x) with unit scale (round to nearest even, saturating at +-448), n elements.
 * spot_linear_fp8: as spot_linear with d_a [M, K] and d_wq [N, K] E4M3 bytes, y = d_w_scale[n] * acc + bias (bias bf16);
 *   SPOT_EPI_BIAS / SPOT_EPI_BIAS_GELU write d_out [M, N] as E4M3 bytes, SPOT_EPI_GATE_RESIDUAL updates the fp32
 *   residual.  K % 16 == 0, N % 32 == 0.
 * spot_qkv_rope_linear_fp8: spot_qkv_rope_linear on E4M3 operands: [q | k | v] = d_w_scale[n] * (d_a d_wq^T) + bias with
 *   d_a [n_seqs * rows_per_seq, K] and d_wq [3 * hidden, K] E4M3 bytes, then QK-RMSNorm + RoPE as there; d_out stays
 *   bf16 (attention runs in bf16, reading Q1).  This is the QKV launch of the FP8 rollout.  K % 16 == 0. */
spot_status spot_quantize_weight_rows(const void *d_w_bf16, int64_t N, int64_t K, void *d_wq, float *d_scale, void *cuda_stream);
spot_status spot_quantize_e4m3(spot_dtype dtype, const void *d_in, int64_t n, void *d_out, void *cuda_stream);
spot_status spot_linear_fp8(spot_epilogue epi, const void *d_a, int64_t M, int64_t K, const void *d_wq, int64_t N,
                            const float *d_w_scale, const void *d_bias, const float *d_gate, float *d_residual, void *d_out,
                            void *cuda_stream);
spot_status spot_qkv_rope_linear_fp8(const void *d_a, int n_seqs, int rows_per_seq, int64_t K, const void *d_wq,
                                     const float *d_w_scale, int64_t hidden, const void *d_bias, const void *d_q_gain,
                                     const void *d_k_gain, const float *d_cos, const float *d_sin, int pos_off, float eps,
                                     void *d_out, void *cuda_stream);

/* NVFP4 building blocks of the 4-bit exploration variant (spot.h).  NVFP4 = E2M1
 * values {0, .5, 1, 1.5, 2, 3, 4, 6} with sign in blocks of 16 consecutive elements along K, one E4M3 scale per block.
 * spot_nvfp4_sizes: bytes of the code matrix [rows, K / 2] (element k in the low / high nibble for k even / odd) and of
 *   the scale-factor buffer (512-byte atoms of 128 rows x 4 blocks; see csrc/nvfp4.cu) for a [rows, K] matrix.
 * spot_nvfp4_row_scale: d_scale[r] = max_k |W_rk| / (6 * 448) (1 for a zero row) - the second-level scale of a weight row.
 * spot_nvfp4_quantize: d_src [rows, K] bf16 (each row divided by d_row_scale[r] first when that pointer is not NULL) ->
 *   block scale sf = e4m3(max|x| / 6), codes e2m1(x / sf), all in fp32 with IEEE division.  rows % 128 == 0, K % 64 == 0.
 * spot_linear_nvfp4: y[m, n] = d_w_scale[n] * sum_blocks sfa sfw sum_k a w + bias[n] on the block-scaled tensor-core path
 *   (kind::mxf4nvf4), fp32 accumulation; SPOT_EPI_BIAS / SPOT_EPI_BIAS_GELU write d_out [M, N] bf16,
 *   SPOT_EPI_GATE_RESIDUAL updates the fp32 residual [M, N].  With SPOT_EPI_BIAS_GELU and d_out_sf != NULL the epilogue
 *   quantises instead (what the rollout's fc1 does): d_out receives the E2M1 codes of GELU(y) [M, N / 2] and d_out_sf their
 *   E4M3 block scales (atoms for a [M, N] matrix), reading N3 applied to the fp32 value - the bf16 tensor is never written.
 *   M % 128 == 0, K % 256 == 0, N % 192 == 0 (tiles 128 x 192, two accumulators: epilogue overlapped) or N % 256 == 0
 *   (tiles 128 x 256), else SPOT_ERR_SHAPE. */
spot_status spot_nvfp4_sizes(int64_t rows, int64_t K, size_t *codes_bytes, size_t *sf_bytes);
spot_status spot_nvfp4_row_scale(const void *d_w_bf16, int64_t rows, int64_t K, float *d_scale, void *cuda_stream);
spot_status spot_nvfp4_quantize(const void *d_src_bf16, int64_t rows, int64_t K, const float *d_row_scale, void *d_codes,
                                void *d_sf, void *cuda_stream);
spot_status spot_linear_nvfp4(spot_epilogue epi, const void *d_a_codes, const void *d_a_sf, int64_t M, int64_t K,
                              const void *d_w_codes, const void *d_w_sf, const float *d_w_scale, int64_t N,
                              const void *d_bias, const float *d_gate, float *d_residual, void *d_out, void *d_out_sf,
                              void *cuda_stream);

/* The RoPE table the context built at spot_create (S5): copies cos and sin [S, d_h/2] fp32 to HOST. */
spot_status spot_rope_table(const spot_ctx *ctx, float *h_cos, float *h_sin);

#ifdef __cplusplus
}
#endif
#endif /* SPOT_KERNELS_H_ */
