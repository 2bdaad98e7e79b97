/* spot.h - C ABI of the B200-native SPOTLIGHT seed-exploration rollout (libspot.so).
 *
 * What the library computes (PAPER.md = the paper text, arxiv 2606.19004):
 *   PAPER.md:59  (s2.1) a DiT "starts from random Gaussian noise and refines a latent
 *                representation over a fixed number of denoising steps ..., each requiring a full
 *                forward pass through the DiT backbone";
 *   PAPER.md:61  (s2.1) "K samples from each of P prompts by running denoising with K distinct noise
 *                seeds ... Each sample is scored ..., yielding a per-sample scalar reward r_k";
 *   PAPER.md:229 (s5)   "top-k/bottom-k strategy over per-prompt exploration rewards, retaining the
 *                highest- and lowest-scoring seeds"; "top and bottom K/2 by reward";
 *   PAPER.md:175 (s4.3.2) the per-prompt reward standard deviation sigma_g fed to the bandit planner.
 * The paper fixes only this outer shape; every inner definition (Philox4x32-10 + Box-Muller, the
 * Qwen-Image-shaped joint block, 2-D RoPE, Euler sampler, linear-probe reward) is a reading listed
 * in DESIGN.md (S1-S16) that binds this library and the fp64 oracle alike.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  All matrices are row-major;
 *     every Linear is y = x W^T + b with W stored [out_features, in_features].
 *   - Ownership: the caller owns every buffer.  The library allocates only inside spot_ctx (host
 *     structs, a small device RoPE table, TMA descriptors) and frees it in spot_destroy.  Weights
 *     are BORROWED for the life of the context.
 *   - Errors: every call returns spot_status; nothing throws, aborts or prints.  Argument errors
 *     are detected before any launch.  Launch failures map to SPOT_ERR_CUDA and the cudaError_t
 *     is retrievable with spot_last_cuda_error().
 *   - Asynchrony: device work is enqueued on the caller's stream (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  Only spot_explore_host synchronises.
 *   - CUDA graphs: spot_noise_from_seeds, spot_dit_denoise, spot_seed_rewards and spot_explore (which chains the
 *     three) enqueue only kernel launches and memsets and read no host pointer after they return (the
 *     timestep grid travels as kernel arguments), so after ONE eager call with the same context and options
 *     (which sets function attributes) a call may be captured into a CUDA graph and replayed while the context,
 *     the workspace and the argument buffers stay alive; a replay reproduces the eager call bit for bit.  The
 *     *_cached calls (one synchronisation per step), spot_explore_host and option SPOT_OPT_TIMING != 0 are not
 *     capturable.
 *   - Determinism: same inputs => bit-identical outputs run to run; the result for sequence b does
 *     not depend on the batch size, its position in the batch, or the other sequences.
 *   - There is no CPU fallback: on a machine without an sm_100 device every compute call returns
 *     SPOT_ERR_ARCH.
 */
#ifndef SPOT_H_
#define SPOT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SPOT_OK = 0,
  SPOT_ERR_NULL = 1,          /* a required pointer is NULL */
  SPOT_ERR_SHAPE = 2,         /* inconsistent or unsupported sizes */
  SPOT_ERR_DTYPE = 3,         /* unknown spot_dtype */
  SPOT_ERR_ALIGN = 4,         /* a pointer is not 16-byte aligned */
  SPOT_ERR_WORKSPACE = 5,     /* workspace smaller than spot_workspace_bytes() */
  SPOT_ERR_ARCH = 6,          /* no CUDA device of compute capability 10.x */
  SPOT_ERR_CUDA = 7,          /* a CUDA call failed; see spot_last_cuda_error() */
  SPOT_ERR_UNIMPLEMENTED = 8
} spot_status;

/* SPOT_E4M3 is a STORAGE type of activations / quantised weights in the FP8 exploration variant and
 * of the kernel-level calls that say so; spot_config.dtype must be SPOT_F32 or SPOT_BF16. */
typedef enum { SPOT_F32 = 0, SPOT_BF16 = 1, SPOT_E4M3 = 2 } spot_dtype;

/* Model/workload shape (plain data, copied at spot_create).  n_img = grid_h * grid_w image tokens,
 * joint sequence S = n_txt + n_img with the text tokens FIRST.  hidden == n_heads * head_dim;
 * rope_pairs (t, h, w) must sum to head_dim / 2; head_dim must be 64 or 128; hidden % 128 == 0;
 * latent_ch % 4 == 0; txt_dim == hidden. */
typedef struct {
  int32_t n_blocks, hidden, n_heads, head_dim, mlp_hidden;
  int32_t grid_h, grid_w, n_txt, latent_ch, txt_dim;
  int32_t rope_pairs[3];
  float rope_theta, ln_eps, rms_eps;
  spot_dtype dtype;   /* of weights, biases, gains, text_emb and inter-kernel activations; latents,
                         velocity, rewards, modulation vectors, the residual stream and all
                         accumulators/statistics are always fp32 */
} spot_config;

/* Per-stream block weights, device pointers of `dtype`, 16-byte aligned. */
typedef struct {
  const void *mod_w, *mod_b;    /* [6D, D], [6D]: (shift1, scale1, gate1, shift2, scale2, gate2) */
  const void *qkv_w, *qkv_b;    /* [3D, D], [3D]: rows q | k | v, head h owns rows h*d_h..(h+1)*d_h-1 */
  const void *q_gain, *k_gain;  /* [d_h] each */
  const void *out_w, *out_b;    /* [D, D], [D] */
  const void *fc1_w, *fc1_b;    /* [F, D], [F] */
  const void *fc2_w, *fc2_b;    /* [D, F], [D] */
} spot_stream_weights;

typedef struct { spot_stream_weights s[2]; } spot_block_weights;   /* [0] = image, [1] = text */

typedef struct {
  const void *time_w1, *time_b1, *time_w2, *time_b2;   /* [D,256], [D], [D,D], [D] */
  const void *img_in_w, *img_in_b;                     /* [D,C], [D] */
  const void *txt_gain, *txt_in_w, *txt_in_b;          /* [txt_dim], [D,txt_dim], [D] */
  const spot_block_weights *blocks;                    /* HOST array of n_blocks structs (copied) */
  const void *final_mod_w, *final_mod_b;               /* [2D,D], [2D]: (scale_f, shift_f) */
  const void *proj_w, *proj_b;                         /* [C,D], [C] */
} spot_weights;

typedef struct spot_ctx spot_ctx;

/* Options for spot_set_option. */
typedef enum {
  SPOT_OPT_GEMM_IMPL = 0,   /* 0 = auto (bf16: CTA-pair tcgen05 with TMA-store epilogue, QK-norm+RoPE fused into the QKV projection),
                             * 1 = SIMT FFMA GEMM, 2 = 1-CTA tcgen05, 3 = CTA-pair tcgen05 with per-thread epilogue,
                             * 4 = as 0 but K4 (QK-norm+RoPE) as its own kernel */
  SPOT_OPT_ATTN_IMPL = 1,   /* 0 = auto (tcgen05 for bf16, d_h = 128: one-pass kernel, 64-key tiles), 1 = SIMT attention, 2 = previous two-pass tcgen05 kernel */
  SPOT_OPT_TIMING = 2,      /* 1 = bracket every tcgen05 GEMM launch with CUDA events on the launch stream; 2 = bracket EVERY kernel
                             * launch (gap probe: spot_get_counters then returns the summed device time of all kernels) */
  SPOT_OPT_FP8 = 3,         /* 1 = the four Linears of every block run on E4M3 operands (after spot_fp8_prepare) */
  SPOT_OPT_NVFP4 = 5,       /* 1 = on top of SPOT_OPT_FP8, fc1 / fc2 of every block run on NVFP4 operands (after spot_nvfp4_prepare) */
  SPOT_OPT_CHUNK_SEQS = 4   /* sequences per pass of the block stack in spot_dit_denoise / spot_explore / spot_explore_host: larger
                             * batches run as consecutive chunks of this many sequences (PAPER.md:338 caps an exploration batch at
                             * 32 sequences); 0 = the whole batch in one pass; default 32.  Results do not depend on it, bit for
                             * bit (see "Determinism").  Applies to the stochastic rollout (spot_dit_denoise_sde) as well; the
                             * cached rollout chunks each step's compacted batch of computing sequences. */
} spot_option;

/* Validates cfg and w, builds the RoPE table (S5) and returns a context.  max_seqs bounds
 * n_seqs / n_prompts*seeds_per_prompt of later calls.  Allocates four small device buffers (RoPE cos / sin, reward
 * partial sums) with cudaMalloc and fills the table with blocking cudaMemcpy: the call synchronises with the device
 * like any cudaMalloc / pageable cudaMemcpy does; it is setup, not part of the timed path.  Launches no kernel. */
spot_status spot_create(const spot_config *cfg, const spot_weights *w, int max_seqs, spot_ctx **out);
spot_status spot_destroy(spot_ctx *ctx);
spot_status spot_set_option(spot_ctx *ctx, spot_option opt, int value);
/* Bytes of device workspace needed by spot_dit_block_forward / spot_dit_denoise / spot_explore*
 * for n_seqs sequences and up to n_steps Euler steps (n_prompts <= n_seqs is assumed). */
spot_status spot_workspace_bytes(const spot_ctx *ctx, int n_seqs, int n_steps, size_t *bytes);
/* Counters since the last reset: kernels launched through ctx, tcgen05 GEMM launches, how many of those
 * were event-timed (SPOT_OPT_TIMING) and their summed device time in ms.  The caller must have
 * synchronised the stream(s) first.  Any output pointer may be NULL. */
spot_status spot_get_counters(spot_ctx *ctx, uint64_t *launches, uint64_t *gemm_launches, uint64_t *gemm_timed,
                              double *gemm_ms, int reset);
const char *spot_status_string(spot_status s);
int spot_last_cuda_error(const spot_ctx *ctx);          /* cudaError_t of the last failed CUDA call */
const char *spot_version(void);

/* (1) Seeds -> N(0,1).  PAPER.md:59 "starts from random Gaussian noise", :61 "K distinct noise
 * seeds", :251 "deterministic random seed" per sample.  DESIGN.md S1-S3: Philox4x32-10 with
 * key = (lo32, hi32)(seed) and counter = (lo32(j), hi32(j), stream_id, 0) for the 4-element block
 * j = e/4, then Box-Muller on 24-bit uniforms.  d_out[b*elems_per_seed + e], fp32.
 * elems_per_seed must be a positive multiple of 4; d_out 16-byte aligned; n_seeds <= 65535 (one grid row per
 * sequence); n_seeds == 0 is a no-op. */
spot_status spot_noise_from_seeds(const uint64_t *d_seeds, int n_seeds, int64_t elems_per_seed,
                                  uint32_t stream_id, float *d_out, void *cuda_stream);
/* The raw Philox words of the same elements (u32 per element), for bit-exact checks. */
spot_status spot_philox_words(const uint64_t *d_seeds, int n_seeds, int64_t elems_per_seed,
                              uint32_t stream_id, uint32_t *d_out, void *cuda_stream);

/* (2) One joint text+image block (S4-S6) for n_seqs sequences.
 * d_h_img [n_seqs, n_img, D], d_h_txt [n_seqs, n_txt, D] of cfg.dtype; d_temb [D] fp32 is the
 * PRE-SiLU conditioning vector (the block applies c = SiLU(temb) and its own modulation Linear).
 * Outputs have the input shapes and dtype; in-place (out == in) is allowed. */
spot_status spot_dit_block_forward(spot_ctx *ctx, int block, int n_seqs,
                                   const void *d_h_img, const void *d_h_txt, const float *d_temb,
                                   void *d_out_img, void *d_out_txt,
                                   void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* (3) n_steps flow-matching Euler steps x <- x + (t_{i+1} - t_i) v(x, t_i) (DESIGN.md
 * S8).  d_latents [P*K, n_img, C] fp32, updated in place; sequence b belongs to prompt b / K.
 * d_text_emb [P, n_txt, txt_dim] of cfg.dtype.  h_timesteps is a HOST array of n_steps + 1 floats
 * (read before the call returns).  Resume: calling with h_timesteps + i and n_steps - i continues
 * a run from the latents after step i (the paper's committed state "latent tensors and scheduler
 * metadata"). */
spot_status spot_dit_denoise(spot_ctx *ctx, int n_prompts, int seeds_per_prompt,
                             float *d_latents, const void *d_text_emb,
                             const float *h_timesteps, int n_steps,
                             void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* (4) Rewards and per-prompt statistics/selection (S9-S12).
 * r_b = <probe, latents_b> / sqrt(n_img*C); per prompt: mean, population std; top-k by (reward
 * descending, index ascending) and bottom-k by (reward ascending, index ascending); indices are
 * positions 0..K-1 inside the prompt group.  argmax = d_top[p*k], argmin = d_bottom[p*k].
 * Requires 0 <= 2*k_select <= K <= 1024.  d_top/d_bottom may be NULL when k_select == 0. */
spot_status spot_seed_rewards(spot_ctx *ctx, int n_prompts, int seeds_per_prompt,
                              const float *d_latents, const float *d_probe, int k_select,
                              float *d_rewards /*[P*K]*/, float *d_stats /*[P,2] mean,std*/,
                              int32_t *d_top /*[P,k]*/, int32_t *d_bottom /*[P,k]*/, void *cuda_stream);

/* Whole exploration rollout on device buffers: (1) with stream_id 0 -> (3) with the reward
 * reduction fused into the last Euler update -> selection of (4).  d_latents is an output. */
spot_status spot_explore(spot_ctx *ctx, int n_prompts, int seeds_per_prompt,
                         const uint64_t *d_seeds, const void *d_text_emb,
                         const float *h_timesteps, int n_steps, const float *d_probe, int k_select,
                         float *d_latents, float *d_rewards, float *d_stats,
                         int32_t *d_top, int32_t *d_bottom,
                         void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* The same with HOST buffers: copies seeds, text_emb and probe to the device, runs spot_explore,
 * copies rewards, stats, top/bottom (and the final latents if h_latents != NULL) back, and
 * synchronises the stream.  Host buffers should be pinned for full copy bandwidth.  The staging
 * area lives at the end of the workspace (accounted for by spot_workspace_bytes). */
spot_status spot_explore_host(spot_ctx *ctx, int n_prompts, int seeds_per_prompt,
                              const uint64_t *h_seeds, const void *h_text_emb,
                              const float *h_timesteps, int n_steps, const float *h_probe, int k_select,
                              float *h_latents, float *h_rewards, float *h_stats,
                              int32_t *h_top, int32_t *h_bottom,
                              void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* ---- Cached-step exploration: the paper's "effective denoising steps" axis s -------------------------------
 * PAPER.md:155 "We therefore control effective denoising steps via a caching strategy rather than truncation";
 * PAPER.md:157 "caches and reuses intermediate transformer outputs across adjacent denoising steps when their
 * residual difference falls below a threshold.  Each Teacache threshold corresponds to an average number of
 * effective denoising steps s".  DESIGN.md section 10 (readings T1-T5) states the rule: per sequence and Euler step i,
 *   m_i = LN(img_in(x_i)) (1 + scale1) + shift1 (block 0, image stream);  steps 0 and T-1 always compute (acc <- 0);
 *   otherwise rel = mean|m_i - m_{i-1}| / mean|m_{i-1}|, acc += poly(rel); acc < threshold: SKIP the L blocks and
 *   use h_img^0 + R (R = h_img^L - h_img^0 of the last computed step); else compute and acc <- 0.
 * poly(r) = sum_j coeffs[j] r^j; n_coeffs == 0 selects the identity poly(r) = r.  Sequences decide independently
 * (a request is one prompt x one seed), the computing ones are compacted into a dense batch for the block kernels.
 * These calls copy the list of computing sequences to the host and synchronise the stream ONCE PER EULER STEP.
 * h_computed (HOST, [P*K, n_steps] bytes, may be NULL) receives 1 where the blocks ran; its row sums are the
 * effective steps per sequence.  h_rel (HOST, [P*K, n_steps] fp32, may be NULL) receives rel (0 at step 0).
 * Requires P*K <= 1024, threshold >= 0, n_coeffs <= 8; workspace from spot_workspace_bytes_cached. */
typedef struct {
  float threshold;
  int32_t n_coeffs;
  float coeffs[8];   /* ascending powers */
} spot_cache_config;
spot_status spot_workspace_bytes_cached(const spot_ctx *ctx, int n_seqs, int n_steps, size_t *bytes);
spot_status spot_dit_denoise_cached(spot_ctx *ctx, int n_prompts, int seeds_per_prompt, float *d_latents,
                                    const void *d_text_emb, const float *h_timesteps, int n_steps,
                                    const spot_cache_config *cache, uint8_t *h_computed, float *h_rel,
                                    void *d_workspace, size_t ws_bytes, void *cuda_stream);
/* spot_explore with cached steps (noise -> cached denoise -> rewards -> selection). */
spot_status spot_explore_cached(spot_ctx *ctx, int n_prompts, int seeds_per_prompt, const uint64_t *d_seeds,
                                const void *d_text_emb, const float *h_timesteps, int n_steps, const float *d_probe,
                                int k_select, const spot_cache_config *cache, float *d_latents, float *d_rewards,
                                float *d_stats, int32_t *d_top, int32_t *d_bottom, uint8_t *h_computed, float *h_rel,
                                void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* ---- Stochastic sampler: the full-quality rollout that follows exploration ---------------------------------
 * PAPER.md:145 step 5 (the selected seeds are rolled out with DiT(n+1) for training), :227 "The algorithm backbone is
 * FlowGRPO", Table 2 (:477-482) "SDE window".  DESIGN.md section 11 (readings D1-D4): steps window_lo <= i < window_hi
 * of the grid take the marginal-preserving reverse-SDE step of the rectified flow
 *     mean = x (1 + sigma^2/(2 t_i) dt) + v (1 + sigma^2 (1 - t_i)/(2 t_i)) dt,   x_next = mean + sigma sqrt(-dt) xi,
 *     sigma = noise_level * sqrt(t_i/(1-t')),  t' = t_i, or t_{i+1} when t_i == 1 (FlowGRPO's rule for the singular first
 *     step: only the denominator moves),  dt = t_{i+1} - t_i < 0,
 * with xi ~ N(0, I) from Philox stream 256 + j of the sequence's seed (same generator as (1)), j = first_step + i the
 * GLOBAL index of the step: a rollout split over several calls (resume after a preemption) passes the
 * number of steps already taken as first_step, so that it neither reuses a noise stream nor shifts the window - the
 * window test is window_lo <= j < window_hi as well, and a split rollout is bit-identical to the unsplit one.  All other
 * steps are the Euler steps of (3).  d_logp [P*K, n_steps] fp32 receives log N(x_next; mean, sigma^2 (-dt) I) averaged over the
 * elements of the latent (0 for deterministic steps) - the per-step log-probability GRPO consumes.
 * Requires 1 >= t_0 > t_1 > ... > t_T >= 0, noise_level >= 0, 0 <= window_lo <= window_hi, first_step >= 0 (else
 * SPOT_ERR_SHAPE).  Workspace as (3). */
spot_status spot_dit_denoise_sde(spot_ctx *ctx, int n_prompts, int seeds_per_prompt, const uint64_t *d_seeds,
                                 float *d_latents, const void *d_text_emb, const float *h_timesteps, int n_steps,
                                 float noise_level, int window_lo, int window_hi, int first_step,
                                 float *d_logp, void *d_workspace, size_t ws_bytes, void *cuda_stream);

/* ---- Low-precision exploration variant: FP8 (E4M3) block Linears ----------------------------------------------
 * PAPER.md:67 (s2.2): "first running a cheap exploratory rollout e.g., with reduced denoising steps or a quantized
 * model, to identify high-contrast seeds, then performing full-quality rollout only on the selected seeds";
 * PAPER.md:340 judges a cheaper exploration by the rank correlation of its rewards with the full rollout's.
 * DESIGN.md section 13 (readings Q1-Q4): only the QKV, out-proj, fc1 and fc2 Linears of each block change:
 *   weights      Wq = e4m3(W / s_n), s_n = max_k |W_nk| / 448 per output channel (made once by spot_fp8_prepare),
 *   activations  e4m3(x) with unit scale (written by the producing kernel: LN-modulate, attention, fc1 epilogue),
 *   y_n = s_n * sum_k xq_k Wq_nk + b_n, fp32 accumulation on kind::f8f6f4 tensor-core instructions;
 * attention (bf16 q, k, v), norms, modulation, the fp32 residual stream, the input / final layers and the sampler are
 * unchanged.  spot_fp8_bytes: size of the caller-owned buffer for the quantised weights and scales (about half of the
 * bf16 block weights); spot_fp8_prepare: fills it (asynchronous on the stream; the buffer must outlive the context's
 * FP8 use); spot_set_option(ctx, SPOT_OPT_FP8, 1) then switches every later block / denoise / explore call.
 * bf16 configs with head_dim 128 only (SPOT_ERR_DTYPE / SPOT_ERR_SHAPE otherwise). */
spot_status spot_fp8_bytes(const spot_ctx *ctx, size_t *bytes);
spot_status spot_fp8_prepare(spot_ctx *ctx, void *d_buffer, size_t bytes, void *cuda_stream);

/* ---- 4-bit exploration variant: NVFP4 MLP Linears on top of the FP8 variant ----------------------------------------
 * Same passages.  DESIGN.md section 13b (readings N1-N5): fc1 and fc2 of every block and stream -
 * two thirds of the block's Linear FLOPs - take BOTH operands as NVFP4: E2M1 values {0, .5, 1, 1.5, 2, 3, 4, 6} with
 * sign in blocks of 16 consecutive elements along K, one E4M3 scale factor per block,
 *   activations  sf_b = e4m3(max_b |x| / 6),  q = e2m1(x / sf_b)   (made per call from the bf16 LN / GELU outputs),
 *   weights      the same on W_n / s_n with s_n = max_k |W_nk| / (6 * 448) fp32 per output channel (spot_nvfp4_prepare),
 *   y_n = s_n * sum_b sfx_b sfw_nb sum_{k in b} qx_k qw_nk + b_n on tcgen05.mma kind::mxf4nvf4.block_scale, fp32 accumulation;
 * QKV and out-proj stay on the FP8 path, everything else is unchanged.  spot_nvfp4_bytes / spot_nvfp4_prepare work like
 * their FP8 counterparts; spot_set_option(ctx, SPOT_OPT_NVFP4, 1) needs SPOT_OPT_FP8 switched on and the prepared buffer
 * (SPOT_ERR_SHAPE otherwise) and enlarges the workspace (query spot_workspace_bytes again).  hidden and mlp_hidden must
 * be multiples of 256 and every call's image / text row counts (n_seqs * n_img, n_seqs * n_txt) multiples of 128
 * (SPOT_ERR_SHAPE otherwise).  Switching SPOT_OPT_FP8 off switches this off too. */
spot_status spot_nvfp4_bytes(const spot_ctx *ctx, size_t *bytes);
spot_status spot_nvfp4_prepare(spot_ctx *ctx, void *d_buffer, size_t bytes, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* SPOT_H_ */
