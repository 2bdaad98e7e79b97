// kernels.h - host-side launchers of every libspot kernel (internal).
#pragma once
#include "common.cuh"

// K1: Philox4x32-10 + Box-Muller (noise.cu)
cudaError_t launch_noise(const uint64_t* d_seeds, int n_seeds, long long elems_per_seed, uint32_t stream_id,
                         float* d_normals, uint32_t* d_words, cudaStream_t st);

// K7: time embedding and skinny Linear (elementwise.cu)
cudaError_t launch_time_embed(const float* d_t, int T, float* d_e /*[T,256]*/, cudaStream_t st);
cudaError_t launch_gemv(spot_dtype wdt, const void* W, const void* b, const float* X, int T, int N, int K,
                        float* out, long long out_stride_t, bool silu_out, cudaStream_t st);
cudaError_t launch_silu(const float* in, float* out, long long n, cudaStream_t st);
// K7 on the tensor cores: c = hi + lo (two bf16 rows per timestep) through the tcgen05 GEMM, then hi + lo + bias
cudaError_t launch_split_hi_lo(const float* c, void* a_bf16, long long n, cudaStream_t st);
cudaError_t launch_fill_f32(float* p, float v, long long n, cudaStream_t st);
// n HOST floats -> device, passed by value as kernel arguments (64 per launch): capture-safe, unlike a copy from pageable memory
cudaError_t launch_put_floats(const float* h_src, int n, float* d_dst, cudaStream_t st);
cudaError_t launch_mod_combine(const float* acc, const void* bias_bf16, int T, int N, float* out, long long stride_t,
                               cudaStream_t st);

// K3: LayerNorm (no affine) * (1 + scale) + shift, fp32 residual rows -> act dtype rows
cudaError_t launch_ln_modulate(spot_dtype odt, const float* h, int M, int D, const float* shift, const float* scale,
                               float eps, void* out, RowMap out_map, cudaStream_t st);
struct LnProblem {          // one stream of launch_ln_modulate2
  const float* h;           // [M, D] fp32 rows
  int M;
  const float* shift;       // [D]
  const float* scale;       // [D]
  void* out;                // activation dtype, rows addressed through out_map
  RowMap out_map;
};
// the same for up to two problems (image and text stream of a block) in ONE launch
cudaError_t launch_ln_modulate2(spot_dtype odt, const LnProblem* probs, int n_probs, int D, float eps, cudaStream_t st);
cudaError_t launch_rmsnorm_rows(spot_dtype dt, const void* in, const void* gain, int M, int D, float eps, void* out,
                                cudaStream_t st);

// K4: per-head RMSNorm(q), RMSNorm(k) + rotary, in place on qkv [B, S, 3, H, d_h]
cudaError_t launch_qk_norm_rope(spot_dtype dt, void* qkv, int B, int S, int H, int dh, int n_txt,
                                const void* qg_img, const void* kg_img, const void* qg_txt, const void* kg_txt,
                                const float* cos_t, const float* sin_t, float eps, cudaStream_t st);

// K6 / K8: Euler update, reward reduction, selection
static const int REWARD_CHUNK = 4096;    // elements per partial sum (fixed => deterministic order)
cudaError_t launch_euler_update(float* x, const float* v, float dt, int B, long long E, const float* probe,
                                float* partials, cudaStream_t st);
cudaError_t launch_reward_partials(const float* x, const float* probe, int B, long long E, float* partials,
                                   cudaStream_t st);
cudaError_t launch_reward_finalize(const float* partials, int B, long long E, float* rewards, cudaStream_t st);
cudaError_t launch_seed_select(const float* rewards, int P, int K, int k_select, float* stats, int32_t* top,
                               int32_t* bottom, cudaStream_t st);

// stochastic sampler step (sde.cu; Table 2 "SDE window"): x <- cx x + cv v + cn xi, xi from Philox
// stream `stream_id` of seeds[b]; logp[b * logp_stride] = log N(x_next; mean, cn^2) averaged over elements; when
// probe != nullptr also the reward partials of the updated x (as launch_euler_update)
cudaError_t launch_sde_update(float* x, const float* v, const uint64_t* seeds, uint32_t stream_id, double cx, double cv,
                              double cn, int B, long long E, const float* probe, float* lp_partials, float* rw_partials,
                              float* logp, long long logp_stride, cudaStream_t st);

// cached-step exploration (teacache.cu)
cudaError_t launch_tc_metric(const float* h0, float* m_prev, const float* shift, const float* scale, long long rows, int D,
                             float eps, bool first, float* row_part, cudaStream_t st);
cudaError_t launch_tc_decide(const float* row_part, int B, int rows_per_seq, bool first, bool force, double threshold,
                             int n_coeffs, const double* d_coeffs, double* acc, int* active_idx, int* pos, int* n_active,
                             int* computed, float* rel, cudaStream_t st);
cudaError_t launch_tc_gather(const float* src, float* dst, const int* idx, int div, int n, long long n_per_seq,
                             cudaStream_t st);
cudaError_t launch_tc_combine(float* h0, float* resid, const float* hc, const int* pos, int B, long long n_per_seq,
                              cudaStream_t st);

// NVFP4 exploration variant (nvfp4.cu, gemm_nvfp4.cu): E2M1 codes [rows, K / 2] + E4M3 block scales in
// 512-byte atoms (128 rows x 4 blocks of 16), fp32 per-row second-level scale for weights
struct Nvfp4Problem {
  const void* a_codes; const void* a_sf;     // activations [M, K / 2], atoms [M / 128][K / 64][512]
  const void* w_codes; const void* w_sf;     // weights     [N, K / 2], atoms [N / 128][K / 64][512]
  const float* w_scale;                      // [N] fp32
  const void* bias;                          // [N] bf16
  int M, N, K;
  void* out;                                 // EPI_BIAS / EPI_BIAS_GELU: [M, N] bf16; with out_sf: E2M1 codes of GELU(y) [M, N / 2]
  void* out_sf;                              // EPI_BIAS_GELU only, optional: scale atoms of the output -> the epilogue quantises (fc2's operand)
  const float* gate;                         // EPI_GATE_RES: [N] fp32
  float* resid;                              // EPI_GATE_RES: [M, N] fp32 residual, updated in place
};
size_t nvfp4_codes_bytes(long long rows, long long K);
size_t nvfp4_sf_bytes(long long rows, long long K);
cudaError_t launch_nvfp4_quantize(const void* src_bf16, RowMap map, int rows, int K, const float* row_scale, void* codes,
                                  void* sf, cudaStream_t st);
cudaError_t launch_nvfp4_row_scale(const void* w_bf16, int rows, int K, float* scale, cudaStream_t st);
bool nvfp4_gemm_supported(const Nvfp4Problem& p);
cudaError_t launch_gemm_nvfp4(Epilogue epi, const Nvfp4Problem* probs, int n_probs, int num_sms, cudaStream_t st);

// FP8 exploration variant (fp8.cu): per-output-channel weight quantisation, unit-scale activation cast
cudaError_t launch_quantize_weight_rows(const void* w_bf16, long long N, int K, void* wq, float* scale, cudaStream_t st);
cudaError_t launch_quantize_e4m3(spot_dtype dt, const void* in, long long n, void* out, cudaStream_t st);

// plumbing
cudaError_t launch_to_f32(spot_dtype dt, const void* in, float* out, long long n, cudaStream_t st);
cudaError_t launch_from_f32(spot_dtype dt, const float* in, void* out, long long n, cudaStream_t st);
cudaError_t launch_broadcast_prompts(const float* src, float* dst, int B, int K, long long n_per_prompt, cudaStream_t st,
                                     int first_seq = 0);

// K9: SIMT GEMM / attention (gemm_simt.cu, attn_simt.cu).  ta/tout: dtype of A and of the output
// matrix (EPI_BIAS / EPI_BIAS_GELU); W and bias have dtype tw.
cudaError_t launch_gemm_simt(spot_dtype ta, spot_dtype tw, spot_dtype tout, Epilogue epi, const GemmProblem& p,
                             cudaStream_t st);
cudaError_t launch_attn_simt(spot_dtype dt, const void* qkv, void* out, int B, int S, int H, int dh, cudaStream_t st);

// K2 / K5: tcgen05 + TMA kernels (gemm_tcgen05.cu, attn_tcgen05.cu), bf16 only.
struct TmaEncoder;   // opaque: resolves cuTensorMapEncodeTiled once
bool tcgen05_gemm_supported(const GemmProblem& p);
cudaError_t launch_gemm_tcgen05(Epilogue epi, const GemmProblem* probs, int n_probs, int num_sms, cudaStream_t st);
cudaError_t launch_gemm_tcgen05_2cta(Epilogue epi, const GemmProblem* probs, int n_probs, int num_sms, cudaStream_t st);
// v3: CTA pairs + TMA-store epilogue (+ EPI_QKV_ROPE, the QKV projection with K4 fused)
cudaError_t launch_gemm_tcgen05_v3(Epilogue epi, const GemmProblem* probs, int n_probs, int num_sms, cudaStream_t st);
bool tcgen05_v3_qkv_rope_supported(const GemmProblem& p);
bool tcgen05_attn_supported(int S, int H, int dh);
cudaError_t launch_attn_tcgen05(const void* qkv, void* out, int B, int S, int H, int dh, int num_sms, cudaStream_t st);
// v3: 64-key tiles, one pass over the scores, double-buffered S per query tile (the default)
cudaError_t launch_attn_tcgen05_v3(const void* qkv, void* out, int B, int S, int H, int dh, int num_sms, cudaStream_t st,
                                   bool out_e4m3 = false);   // out_e4m3: O stored as E4M3 bytes (operand of the FP8 out-projection)
