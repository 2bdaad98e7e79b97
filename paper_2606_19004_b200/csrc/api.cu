// api.cu - the C ABI of libspot.so (include/spot.h, include/spot_kernels.h): argument validation,
// workspace carving and the launch sequence of the exploration rollout.  Every step runs in the
// kernels of this directory; there is no CPU or library fallback.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "../../include/spot_kernels.h"
#include "kernels.h"

struct spot_ctx {
  spot_config cfg;
  spot_weights w;
  std::vector<spot_block_weights> blocks;
  int max_seqs;
  int num_sms;
  int last_cuda;
  int gemm_impl, attn_impl;      // 0 auto, 1 force SIMT
  float* d_cos;                  // [S, d_h/2]
  float* d_sin;
  float* d_partials;             // [max_seqs, reward chunks]
  float* d_partials2;            // [max_seqs, reward chunks]: sum xi^2 of the stochastic step
  unsigned long long n_launches; // kernels launched through this context
  int timing;                    // 1: bracket every tcgen05 GEMM launch with CUDA events
  std::vector<cudaEvent_t> ev;   // event pool (pairs)
  size_t ev_used;
  unsigned long long gemm_launches;
  // FP8 exploration variant: quantised copies of the four block Linears, in a caller-owned buffer
  struct Fp8Linear { const uint8_t* w; const float* scale; };
  struct Fp8Block { Fp8Linear lin[2][4]; };   // [stream][qkv, out, fc1, fc2]
  std::vector<Fp8Block> fp8_blocks;
  int fp8;                       // 1: block Linears run on E4M3 operands (SPOT_OPT_FP8; needs spot_fp8_prepare)
  // NVFP4 exploration variant: fc1 / fc2 of every block as E2M1 codes + E4M3 block scales + fp32 row scale
  struct Nv4Linear { const uint8_t* codes; const uint8_t* sf; const float* scale; };
  struct Nv4Block { Nv4Linear lin[2][2]; };   // [stream][fc1, fc2]
  std::vector<Nv4Block> nv4_blocks;
  int nvfp4;                     // 1: the MLP Linears run on the block-scaled 4-bit path (SPOT_OPT_NVFP4; on top of SPOT_OPT_FP8)
  int chunk_seqs;                // sequences per pass of the block stack (SPOT_OPT_CHUNK_SEQS); 0 = whole batch
  int n_img() const { return cfg.grid_h * cfg.grid_w; }
  int seq() const { return cfg.n_txt + n_img(); }
};

namespace {

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
inline size_t esize(spot_dtype d) { return d == SPOT_F32 ? 4 : 2; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

// 0 = unknown, 1 = ok (cc 10.x), -1 = no usable device
int device_state() {
  static int state = 0;
  if (state == 0) {
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
      cudaGetLastError();
      state = -1;
    } else {
      state = prop.major == 10 ? 1 : -1;
    }
  }
  return state;
}

constexpr size_t kMaxTimingEvents = 1 << 16;

struct Workspace {
  // all offsets in bytes from the workspace base
  size_t t_dev, emb, hid, temb, cvec, mod, fmod, txt_norm, txt_h0, h_img, h_txt, ybuf, big, vel, stage, total;
  size_t st_seeds, st_text, st_probe, st_lat, st_rew, st_stats, st_top, st_bot;
  // cached-step variant only (carve(..., cached = true)): uncompacted h_img^0, previous modulated input, cached residual
  size_t nv_codes[2], nv_sf[2], nv_codes2[2], nv_sf2[2];   // NVFP4 variant only: quantised y2 and u of the image / text stream
  size_t md_a, md_acc, md_ones, md_zero;   // tensor-core modulation path (conditioning): split c, accumulators, gate = 1, bias = 0
  size_t tc_h0, tc_mprev, tc_resid, tc_rowpart, tc_acc, tc_coeffs, tc_idx, tc_pos, tc_nact, tc_comp, tc_rel;
};

Workspace carve(const spot_ctx* c, int B, int T, bool cached = false) {
  const spot_config& g = c->cfg;
  const size_t D = g.hidden, S = c->seq(), NI = c->n_img(), NT = g.n_txt, L = g.n_blocks, es = esize(g.dtype);
  const size_t E = NI * g.latent_ch;
  const size_t wide = (size_t)(3 * D > (size_t)g.mlp_hidden ? 3 * D : g.mlp_hidden);
  Workspace w;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += align_up(bytes); return r; };
  const size_t Tp = T > 0 ? T : 1;
  w.t_dev = take((Tp + 1) * 4);
  w.emb = take(Tp * 256 * 4);
  w.hid = take(Tp * D * 4);
  w.temb = take(Tp * D * 4);
  w.cvec = take(Tp * D * 4);
  w.mod = take(Tp * L * 2 * 6 * D * 4);
  w.fmod = take(Tp * 2 * D * 4);
  w.md_a = take(2 * Tp * D * 2);
  w.md_acc = take(2 * 2 * Tp * 6 * D * 4);             // [stream][2 T, 6 D] fp32, reused block after block
  w.md_ones = take(6 * D * 4);
  w.md_zero = take(6 * D * 2);
  w.txt_norm = take((size_t)B * NT * g.txt_dim * es);
  w.txt_h0 = take((size_t)B * NT * D * 4);
  w.h_img = take((size_t)B * NI * D * 4);
  w.h_txt = take((size_t)B * NT * D * 4);
  w.ybuf = take((size_t)B * S * D * es);
  w.big = take((size_t)B * S * wide * es);
  w.vel = take((size_t)B * E * 4);
  w.stage = o;
  w.st_seeds = take((size_t)B * 8);
  w.st_text = take((size_t)B * NT * g.txt_dim * es);
  w.st_probe = take(E * 4);
  w.st_lat = take((size_t)B * E * 4);
  w.st_rew = take((size_t)B * 4);
  w.st_stats = take((size_t)B * 2 * 4);
  w.st_top = take((size_t)B * 4);
  w.st_bot = take((size_t)B * 4);
  w.nv_codes[0] = w.nv_codes[1] = w.nv_sf[0] = w.nv_sf[1] = w.nv_codes2[0] = w.nv_codes2[1] = w.nv_sf2[0] = w.nv_sf2[1] = 0;
  if (c->nvfp4) {
    const size_t rows[2] = {(size_t)B * NI, (size_t)B * NT};
    for (int s = 0; s < 2; ++s) {
      w.nv_codes[s] = take(nvfp4_codes_bytes((long long)rows[s], (long long)D));
      w.nv_sf[s] = take(nvfp4_sf_bytes((long long)rows[s], (long long)D));
      w.nv_codes2[s] = take(nvfp4_codes_bytes((long long)rows[s], (long long)g.mlp_hidden));
      w.nv_sf2[s] = take(nvfp4_sf_bytes((long long)rows[s], (long long)g.mlp_hidden));
    }
  }
  w.tc_h0 = w.tc_mprev = w.tc_resid = w.tc_rowpart = w.tc_acc = w.tc_coeffs = w.tc_idx = w.tc_pos = w.tc_nact = w.tc_comp =
      w.tc_rel = 0;
  if (cached) {
    w.tc_h0 = take((size_t)B * NI * D * 4);
    w.tc_mprev = take((size_t)B * NI * D * 4);
    w.tc_resid = take((size_t)B * NI * D * 4);
    w.tc_rowpart = take((size_t)B * NI * 8);
    w.tc_acc = take((size_t)B * 8);
    w.tc_coeffs = take(8 * 8);
    w.tc_idx = take((size_t)B * 4 + 4);      // active_idx[B] followed by n_active (copied to the host together)
    w.tc_nact = w.tc_idx + (size_t)B * 4;
    w.tc_pos = take((size_t)B * 4);
    w.tc_comp = take((size_t)B * 4);
    w.tc_rel = take((size_t)B * 4);
  }
  w.total = o;
  return w;
}

#define CK(ctx, expr)                                  \
  do {                                                 \
    cudaError_t _e = (expr);                           \
    if (_e != cudaSuccess) {                           \
      (ctx)->last_cuda = (int)_e;                      \
      return SPOT_ERR_CUDA;                            \
    }                                                  \
  } while (0)

// SPOT_OPT_TIMING = 2: an event pair around EVERY kernel launch (gap probe: wall time of a rollout minus the summed
// kernel time = what launch gaps cost).  Returns false when the event pool is exhausted or an event call failed.
bool launch_event(spot_ctx* c, cudaStream_t st) {
  if (c->ev_used + 1 > kMaxTimingEvents) return false;
  while (c->ev.size() < c->ev_used + 1) {
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return false;
    c->ev.push_back(e);
  }
  return cudaEventRecord(c->ev[c->ev_used++], st) == cudaSuccess;
}

// LK = CK for a kernel launcher: also counts the launch (reported by spot_get_counters).  Used where the launch stream
// is in scope as `st`.
#define LK(ctx, expr)                                                        \
  do {                                                                       \
    ++(ctx)->n_launches;                                                     \
    const bool _probe = (ctx)->timing == 2 && launch_event((ctx), st);       \
    CK(ctx, expr);                                                           \
    if (_probe && !launch_event((ctx), st)) return SPOT_ERR_CUDA;            \
  } while (0)

// Linear layer dispatch: tcgen05 when the context runs bf16 and every problem qualifies, else SIMT.
spot_status run_gemm(spot_ctx* c, Epilogue epi, GemmProblem* probs, int n, spot_dtype ta, spot_dtype tout,
                     cudaStream_t st) {
  const spot_dtype dt = c->cfg.dtype;
  bool tc = dt == SPOT_BF16 && ta == SPOT_BF16 && (epi == EPI_GATE_RES || tout == SPOT_BF16) && c->gemm_impl != 1;
  for (int i = 0; i < n && tc; ++i)
    if (probs[i].M > 0 && !tcgen05_gemm_supported(probs[i])) tc = false;
  if (tc) {
    const bool timed = c->timing == 1 && c->ev_used + 2 <= kMaxTimingEvents;
    if (timed) {
      while (c->ev.size() < c->ev_used + 2) {
        cudaEvent_t e;
        CK(c, cudaEventCreate(&e));
        c->ev.push_back(e);
      }
      CK(c, cudaEventRecord(c->ev[c->ev_used], st));
    }
    if (c->gemm_impl == 2) LK(c, launch_gemm_tcgen05(epi, probs, n, c->num_sms, st));
    else if (c->gemm_impl == 3) LK(c, launch_gemm_tcgen05_2cta(epi, probs, n, c->num_sms, st));
    else LK(c, launch_gemm_tcgen05_v3(epi, probs, n, c->num_sms, st));   // auto = CTA pairs + TMA-store epilogue
    ++c->gemm_launches;
    if (timed) {
      CK(c, cudaEventRecord(c->ev[c->ev_used + 1], st));
      c->ev_used += 2;
    }
  } else {
    for (int i = 0; i < n; ++i)
      if (probs[i].fp8) return SPOT_ERR_SHAPE;            // E4M3 operands exist on the tcgen05 path only
    for (int i = 0; i < n; ++i) LK(c, launch_gemm_simt(ta, dt, tout, epi, probs[i], st));
  }
  return SPOT_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

const char* spot_status_string(spot_status s) {
  switch (s) {
    case SPOT_OK: return "SPOT_OK";
    case SPOT_ERR_NULL: return "SPOT_ERR_NULL: a required pointer is NULL";
    case SPOT_ERR_SHAPE: return "SPOT_ERR_SHAPE: inconsistent or unsupported sizes";
    case SPOT_ERR_DTYPE: return "SPOT_ERR_DTYPE: unknown dtype";
    case SPOT_ERR_ALIGN: return "SPOT_ERR_ALIGN: pointer not 16-byte aligned";
    case SPOT_ERR_WORKSPACE: return "SPOT_ERR_WORKSPACE: workspace too small";
    case SPOT_ERR_ARCH: return "SPOT_ERR_ARCH: no CUDA device of compute capability 10.x";
    case SPOT_ERR_CUDA: return "SPOT_ERR_CUDA: a CUDA call failed";
    case SPOT_ERR_UNIMPLEMENTED: return "SPOT_ERR_UNIMPLEMENTED";
  }
  return "unknown spot_status";
}

const char* spot_version(void) { return "libspot 0.1 (sm_100a)"; }

int spot_last_cuda_error(const spot_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }

static spot_status validate_config(const spot_config* c) {
  if (c->dtype != SPOT_F32 && c->dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  if (c->n_blocks < 0 || c->hidden <= 0 || c->n_heads <= 0 || c->head_dim <= 0 || c->mlp_hidden <= 0 ||
      c->grid_h <= 0 || c->grid_w <= 0 || c->n_txt < 0 || c->latent_ch <= 0)
    return SPOT_ERR_SHAPE;
  if (c->n_heads * c->head_dim != c->hidden) return SPOT_ERR_SHAPE;
  if (c->head_dim != 64 && c->head_dim != 128) return SPOT_ERR_SHAPE;
  if (c->rope_pairs[0] < 0 || c->rope_pairs[1] < 0 || c->rope_pairs[2] < 0 ||
      c->rope_pairs[0] + c->rope_pairs[1] + c->rope_pairs[2] != c->head_dim / 2)
    return SPOT_ERR_SHAPE;
  const int dq = c->hidden / 128;
  if (c->hidden % 128 || !(dq == 1 || dq == 2 || dq == 4 || dq == 8 || dq == 12 || dq == 16 || dq == 24 || dq == 32))
    return SPOT_ERR_SHAPE;
  if (c->mlp_hidden % 16 || c->latent_ch % 16 || c->txt_dim != c->hidden) return SPOT_ERR_SHAPE;
  if (!(c->rope_theta > 0.f) || !(c->ln_eps >= 0.f) || !(c->rms_eps >= 0.f)) return SPOT_ERR_SHAPE;
  return SPOT_OK;
}

// RoPE table (S5): d_h/2 pairs split over axes (t, h, w); pair i' of an axis with n_a pairs
// has frequency theta^(-i'/n_a).  Text token j sits at max(G_h/2, G_w/2) + j on all axes; image token
// (r, c) at (0, r - ceil(G_h/2), c - ceil(G_w/2)).  Host double math, cast once to fp32.
static void build_rope_host(const spot_config& c, std::vector<float>& cs, std::vector<float>& sn) {
  const int S = c.n_txt + c.grid_h * c.grid_w, half = c.head_dim / 2;
  cs.resize((size_t)S * half);
  sn.resize((size_t)S * half);
  const int base = (c.grid_h / 2 > c.grid_w / 2) ? c.grid_h / 2 : c.grid_w / 2;
  for (int s = 0; s < S; ++s) {
    double pos[3];
    if (s < c.n_txt) {
      pos[0] = pos[1] = pos[2] = (double)(base + s);
    } else {
      const int n = s - c.n_txt, r = n / c.grid_w, col = n % c.grid_w;
      pos[0] = 0.0;
      pos[1] = (double)(r - (c.grid_h + 1) / 2);
      pos[2] = (double)(col - (c.grid_w + 1) / 2);
    }
    int p = 0;
    for (int a = 0; a < 3; ++a)
      for (int i = 0; i < c.rope_pairs[a]; ++i, ++p) {
        const double ang = pos[a] * pow((double)c.rope_theta, -(double)i / (double)c.rope_pairs[a]);
        cs[(size_t)s * half + p] = (float)cos(ang);
        sn[(size_t)s * half + p] = (float)sin(ang);
      }
  }
}

spot_status spot_create(const spot_config* cfg, const spot_weights* w, int max_seqs, spot_ctx** out) {
  if (!cfg || !w || !out) return SPOT_ERR_NULL;
  *out = nullptr;
  spot_status vs = validate_config(cfg);
  if (vs != SPOT_OK) return vs;
  if (max_seqs <= 0) return SPOT_ERR_SHAPE;
  if (cfg->n_blocks > 0 && !w->blocks) return SPOT_ERR_NULL;
  const void* globals[] = {w->time_w1, w->time_b1, w->time_w2, w->time_b2, w->img_in_w, w->img_in_b, w->txt_gain,
                           w->txt_in_w, w->txt_in_b, w->final_mod_w, w->final_mod_b, w->proj_w, w->proj_b};
  for (const void* p : globals) {
    if (!p) return SPOT_ERR_NULL;
    if (!aligned16(p)) return SPOT_ERR_ALIGN;
  }
  for (int b = 0; b < cfg->n_blocks; ++b)
    for (int s = 0; s < 2; ++s) {
      const spot_stream_weights& sw = w->blocks[b].s[s];
      const void* ps[] = {sw.mod_w, sw.mod_b, sw.qkv_w, sw.qkv_b, sw.q_gain, sw.k_gain,
                          sw.out_w, sw.out_b, sw.fc1_w, sw.fc1_b, sw.fc2_w, sw.fc2_b};
      for (const void* p : ps) {
        if (!p) return SPOT_ERR_NULL;
        if (!aligned16(p)) return SPOT_ERR_ALIGN;
      }
    }
  if (device_state() != 1) return SPOT_ERR_ARCH;
  spot_ctx* c = new (std::nothrow) spot_ctx();
  if (!c) return SPOT_ERR_CUDA;
  c->cfg = *cfg;
  c->w = *w;
  c->blocks.assign(w->blocks, w->blocks + cfg->n_blocks);
  c->w.blocks = c->blocks.data();
  c->max_seqs = max_seqs;
  c->last_cuda = 0;
  c->gemm_impl = c->attn_impl = 0;
  c->chunk_seqs = 32;
  c->n_launches = c->gemm_launches = 0;
  c->timing = 0;
  c->fp8 = 0;
  c->nvfp4 = 0;
  c->ev_used = 0;
  c->d_cos = c->d_sin = c->d_partials = c->d_partials2 = nullptr;
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
  std::vector<float> cs, sn;
  build_rope_host(*cfg, cs, sn);
  const size_t E = (size_t)c->n_img() * cfg->latent_ch;
  const size_t n_part = (size_t)max_seqs * ((E + REWARD_CHUNK - 1) / REWARD_CHUNK);
  cudaError_t e = cudaMalloc(&c->d_cos, cs.size() * 4);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_sin, sn.size() * 4);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_partials, n_part * 4);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_partials2, n_part * 4);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_cos, cs.data(), cs.size() * 4, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_sin, sn.data(), sn.size() * 4, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(c->d_cos); cudaFree(c->d_sin); cudaFree(c->d_partials); cudaFree(c->d_partials2);
    delete c;
    return SPOT_ERR_CUDA;
  }
  *out = c;
  return SPOT_OK;
}

spot_status spot_destroy(spot_ctx* ctx) {
  if (!ctx) return SPOT_ERR_NULL;
  cudaFree(ctx->d_cos);
  cudaFree(ctx->d_sin);
  cudaFree(ctx->d_partials);
  cudaFree(ctx->d_partials2);
  for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
  delete ctx;
  return SPOT_OK;
}

spot_status spot_set_option(spot_ctx* ctx, spot_option opt, int value) {
  if (!ctx) return SPOT_ERR_NULL;
  if (opt == SPOT_OPT_GEMM_IMPL) {
    if (value < 0 || value > 4) return SPOT_ERR_SHAPE;
    if (value != 0 && ctx->fp8) return SPOT_ERR_SHAPE;   // the E4M3 Linears exist on the default GEMM only
    ctx->gemm_impl = value;
    return SPOT_OK;
  }
  if (opt == SPOT_OPT_ATTN_IMPL) {
    if (value < 0 || value > 2) return SPOT_ERR_SHAPE;
    ctx->attn_impl = value;
    return SPOT_OK;
  }
  if (opt == SPOT_OPT_CHUNK_SEQS) {
    if (value < 0) return SPOT_ERR_SHAPE;
    ctx->chunk_seqs = value;
    return SPOT_OK;
  }
  if (opt == SPOT_OPT_TIMING) {
    if (value < 0 || value > 2) return SPOT_ERR_SHAPE;
    ctx->timing = value;
    return SPOT_OK;
  }
  if (value != 0 && value != 1) return SPOT_ERR_SHAPE;
  if (opt == SPOT_OPT_FP8) {
    if (value && (ctx->fp8_blocks.size() != ctx->blocks.size() || ctx->cfg.dtype != SPOT_BF16 || ctx->cfg.head_dim != 128 ||
                  ctx->gemm_impl != 0))
      return SPOT_ERR_SHAPE;                     // spot_fp8_prepare first; bf16 configs with d_h = 128, default GEMM only
    ctx->fp8 = value;
    if (!value) ctx->nvfp4 = 0;                  // the 4-bit MLP rides on the FP8 variant
    return SPOT_OK;
  }
  if (opt == SPOT_OPT_NVFP4) {
    if (value && (!ctx->fp8 || ctx->nv4_blocks.size() != ctx->blocks.size() || ctx->cfg.hidden % 256 || ctx->cfg.mlp_hidden % 256))
      return SPOT_ERR_SHAPE;                     // SPOT_OPT_FP8 and spot_nvfp4_prepare first; widths in multiples of 256
    ctx->nvfp4 = value;
    return SPOT_OK;
  }
  if (opt == SPOT_OPT_GEMM_IMPL) ctx->gemm_impl = value;
  else if (opt == SPOT_OPT_TIMING) ctx->timing = value;
  else return SPOT_ERR_SHAPE;
  return SPOT_OK;
}

spot_status spot_get_counters(spot_ctx* ctx, uint64_t* launches, uint64_t* gemm_launches, uint64_t* gemm_timed,
                              double* gemm_ms, int reset) {
  if (!ctx) return SPOT_ERR_NULL;
  double ms = 0.0;
  for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
    float t = 0.f;
    cudaError_t e = cudaEventElapsedTime(&t, ctx->ev[i], ctx->ev[i + 1]);
    if (e != cudaSuccess) { ctx->last_cuda = (int)e; return SPOT_ERR_CUDA; }
    ms += t;
  }
  if (launches) *launches = ctx->n_launches;
  if (gemm_launches) *gemm_launches = ctx->gemm_launches;
  if (gemm_timed) *gemm_timed = ctx->ev_used / 2;
  if (gemm_ms) *gemm_ms = ms;
  if (reset) { ctx->n_launches = ctx->gemm_launches = 0; ctx->ev_used = 0; }
  return SPOT_OK;
}

spot_status spot_workspace_bytes(const spot_ctx* ctx, int n_seqs, int n_steps, size_t* bytes) {
  if (!ctx || !bytes) return SPOT_ERR_NULL;
  if (n_seqs <= 0 || n_seqs > ctx->max_seqs || n_steps < 0) return SPOT_ERR_SHAPE;
  *bytes = carve(ctx, n_seqs, n_steps).total;
  return SPOT_OK;
}

spot_status spot_rope_table(const spot_ctx* ctx, float* h_cos, float* h_sin) {
  if (!ctx || !h_cos || !h_sin) return SPOT_ERR_NULL;
  const size_t n = (size_t)ctx->seq() * (ctx->cfg.head_dim / 2) * 4;
  if (cudaMemcpy(h_cos, ctx->d_cos, n, cudaMemcpyDeviceToHost) != cudaSuccess) return SPOT_ERR_CUDA;
  if (cudaMemcpy(h_sin, ctx->d_sin, n, cudaMemcpyDeviceToHost) != cudaSuccess) return SPOT_ERR_CUDA;
  return SPOT_OK;
}

}  // extern "C"

// ================================================================================================
// internal launch sequences
namespace {

struct StreamMaps {          // row maps of one stream (image or text) inside the joint buffers
  int rows;                  // B * n_sigma
  RowMap y, qkv, wide, h;    // [B,S,D] ybuf, [B,S,3D] qkv, [B,S,F] mlp hidden, [B,n_sigma,D] residual
};

StreamMaps stream_maps(const spot_ctx* c, int B, int stream /*0 img, 1 txt*/) {
  const long long D = c->cfg.hidden, S = c->seq(), F = c->cfg.mlp_hidden;
  const int n = stream == 0 ? c->n_img() : c->cfg.n_txt;
  const long long first = stream == 0 ? c->cfg.n_txt : 0;       // text tokens come first in the joint sequence
  StreamMaps m;
  m.rows = B * n;
  const int rps = n > 0 ? n : 1;
  m.y = RowMap{rps, S * D, first * D, D};
  m.qkv = RowMap{rps, S * 3 * D, first * 3 * D, 3 * D};
  m.wide = RowMap{rps, S * F, first * F, F};
  m.h = RowMap{rps, (long long)n * D, 0, D};
  return m;
}

// One joint block on the fp32 residual streams h_img [B,n_img,D], h_txt [B,n_txt,D] (S4 steps
// 2-8).  mod_img / mod_txt: [6D] fp32 = (shift1, scale1, gate1, shift2, scale2, gate2).  When
// img_only_tail is set (last block of a denoise pass, S16) the text stream's out-proj and MLP,
// whose result nobody reads, are skipped.
// quantised MLP activations per stream (NVFP4 variant): y2 (fc1's operand) and u (fc2's operand, written by fc1's epilogue)
struct Nv4Scratch { uint8_t* codes[2]; uint8_t* sf[2]; uint8_t* codes2[2]; uint8_t* sf2[2]; };

spot_status block_core(spot_ctx* c, int block, int B, float* h_img, float* h_txt, const float* mod_img,
                       const float* mod_txt, void* ybuf, void* big, bool img_only_tail, cudaStream_t st,
                       const Nv4Scratch* nv = nullptr) {
  const spot_config& g = c->cfg;
  const spot_dtype dt = g.dtype;
  const int D = g.hidden, F = g.mlp_hidden, S = c->seq();
  const spot_block_weights& bw = c->blocks[block];
  float* h[2] = {h_img, h_txt};
  const float* mod[2] = {mod_img, mod_txt};
  StreamMaps sm[2] = {stream_maps(c, B, 0), stream_maps(c, B, 1)};
  GemmProblem pr[2];
  // (2) y = LN(h) (1 + scale1) + shift1 ; (3) qkv = y Wqkv^T + b
  // FP8 variant: the activations feeding the four Linears are stored as E4M3 (same row maps: element = byte), the
  // weights come from the quantised copies, accumulators are dequantised per output channel in the epilogue
  const bool f8 = c->fp8 != 0 && dt == SPOT_BF16 && c->gemm_impl == 0 && g.head_dim == 128;
  const spot_dtype adt = f8 ? SPOT_E4M3 : dt;            // storage type of LN output, attention output, MLP hidden
  const spot_ctx::Fp8Block* fb = f8 ? &c->fp8_blocks[block] : nullptr;
  auto use_fp8 = [&](GemmProblem& p, int s, int which) {
    if (!f8) return;
    p.fp8 = 1; p.W = fb->lin[s][which].w; p.w_scale = fb->lin[s][which].scale;
  };
  LnProblem lp[2];
  for (int s = 0; s < 2; ++s) lp[s] = LnProblem{h[s], sm[s].rows, mod[s], mod[s] + D, ybuf, sm[s].y};
  LK(c, launch_ln_modulate2(adt, lp, 2, D, g.ln_eps, st));   // image and text rows in one launch
  for (int s = 0; s < 2; ++s) {
    memset(&pr[s], 0, sizeof(GemmProblem));
    pr[s].A = ybuf; pr[s].a_map = sm[s].y; pr[s].W = bw.s[s].qkv_w; pr[s].bias = bw.s[s].qkv_b;
    pr[s].M = sm[s].rows; pr[s].N = 3 * D; pr[s].K = D; pr[s].out = big; pr[s].out_map = sm[s].qkv;
    use_fp8(pr[s], s, 0);
  }
  // (4)-(5) QK-RMSNorm + RoPE: fused into the epilogue of the QKV projection (v3 kernel, d_h = 128), else K4
  bool fuse_qk = dt == SPOT_BF16 && c->gemm_impl == 0 && g.head_dim == 128;
  for (int s = 0; s < 2; ++s) {
    pr[s].q_gain = bw.s[s].q_gain; pr[s].k_gain = bw.s[s].k_gain; pr[s].cos_t = c->d_cos; pr[s].sin_t = c->d_sin;
    pr[s].pos_off = s == 0 ? g.n_txt : 0; pr[s].rms_eps = g.rms_eps;
    if (pr[s].M > 0 && !(tcgen05_gemm_supported(pr[s]) && tcgen05_v3_qkv_rope_supported(pr[s]))) fuse_qk = false;
  }
  if (f8 && !fuse_qk) return SPOT_ERR_SHAPE;             // the FP8 QKV projection exists only with the fused bf16 q/k/v epilogue
  spot_status rs = run_gemm(c, fuse_qk ? EPI_QKV_ROPE : EPI_BIAS, pr, 2, dt, dt, st);
  if (rs != SPOT_OK) return rs;
  if (!fuse_qk)
    LK(c, launch_qk_norm_rope(dt, big, B, S, g.n_heads, g.head_dim, g.n_txt, bw.s[0].q_gain, bw.s[0].k_gain,
                              bw.s[1].q_gain, bw.s[1].k_gain, c->d_cos, c->d_sin, g.rms_eps, st));
  // (6) joint attention -> ybuf [B,S,D]
  if (dt == SPOT_BF16 && c->attn_impl != 1 && tcgen05_attn_supported(S, g.n_heads, g.head_dim)) {
    if (c->attn_impl == 2) LK(c, launch_attn_tcgen05(big, ybuf, B, S, g.n_heads, g.head_dim, c->num_sms, st));
    else LK(c, launch_attn_tcgen05_v3(big, ybuf, B, S, g.n_heads, g.head_dim, c->num_sms, st, f8));
  }
  else
    LK(c, launch_attn_simt(dt, big, ybuf, B, S, g.n_heads, g.head_dim, st));
  const int ns = img_only_tail ? 1 : 2;
  // (7) h += gate1 * (o Wout^T + b)
  for (int s = 0; s < ns; ++s) {
    memset(&pr[s], 0, sizeof(GemmProblem));
    pr[s].A = ybuf; pr[s].a_map = sm[s].y; pr[s].W = bw.s[s].out_w; pr[s].bias = bw.s[s].out_b;
    pr[s].M = sm[s].rows; pr[s].N = D; pr[s].K = D; pr[s].gate = mod[s] + 2 * D; pr[s].resid = h[s]; pr[s].resid_map = sm[s].h;
    use_fp8(pr[s], s, 1);
  }
  rs = run_gemm(c, EPI_GATE_RES, pr, ns, dt, SPOT_F32, st);
  if (rs != SPOT_OK) return rs;
  // (8) y2 = LN(h)(1 + scale2) + shift2 ; u = GELU(y2 W1^T + b) ; h += gate2 * (u W2^T + b)
  for (int s = 0; s < ns; ++s) lp[s] = LnProblem{h[s], sm[s].rows, mod[s] + 3 * D, mod[s] + 4 * D, ybuf, sm[s].y};
  const bool nv4 = f8 && c->nvfp4 != 0;
  LK(c, launch_ln_modulate2(nv4 ? dt : adt, lp, ns, D, g.ln_eps, st));
  if (nv4) {
    // NVFP4 variant: y2 (bf16) -> E2M1 codes + E4M3 block scales -> fc1 on the block-scaled 4-bit
    // tensor-core path with the GELU epilogue -> u (bf16, dense per stream in `big`) -> codes + scales -> fc2 with the
    // gate-residual epilogue on the fp32 residual stream.
    if (!nv) return SPOT_ERR_WORKSPACE;
    const spot_ctx::Nv4Block& nb = c->nv4_blocks[block];
    Nvfp4Problem np[2];
    for (int s = 0; s < ns; ++s) {
      memset(&np[s], 0, sizeof(Nvfp4Problem));
      np[s].a_codes = nv->codes[s]; np[s].a_sf = nv->sf[s]; np[s].w_codes = nb.lin[s][0].codes; np[s].w_sf = nb.lin[s][0].sf;
      np[s].w_scale = nb.lin[s][0].scale; np[s].bias = bw.s[s].fc1_b; np[s].M = sm[s].rows; np[s].N = F; np[s].K = D; np[s].out = nv->codes2[s];
      if (np[s].M > 0 && !nvfp4_gemm_supported(np[s])) return SPOT_ERR_SHAPE;   // rows in multiples of 128, widths of 256
      LK(c, launch_nvfp4_quantize(ybuf, sm[s].y, sm[s].rows, D, nullptr, nv->codes[s], nv->sf[s], st));
    }
    // fc1's epilogue quantises u itself (codes + scales straight into fc2's operand buffers `u2`): u is never stored
    for (int s = 0; s < ns; ++s) { np[s].out = nv->codes2[s]; np[s].out_sf = nv->sf2[s]; }
    LK(c, launch_gemm_nvfp4(EPI_BIAS_GELU, np, ns, c->num_sms, st));
    for (int s = 0; s < ns; ++s) {
      np[s].a_codes = nv->codes2[s]; np[s].a_sf = nv->sf2[s]; np[s].out_sf = nullptr;
      np[s].w_codes = nb.lin[s][1].codes; np[s].w_sf = nb.lin[s][1].sf; np[s].w_scale = nb.lin[s][1].scale; np[s].bias = bw.s[s].fc2_b;
      np[s].N = D; np[s].K = F; np[s].out = nullptr; np[s].gate = mod[s] + 5 * D; np[s].resid = h[s];
    }
    LK(c, launch_gemm_nvfp4(EPI_GATE_RES, np, ns, c->num_sms, st));
    return SPOT_OK;
  }
  for (int s = 0; s < ns; ++s) {
    memset(&pr[s], 0, sizeof(GemmProblem));
    pr[s].A = ybuf; pr[s].a_map = sm[s].y; pr[s].W = bw.s[s].fc1_w; pr[s].bias = bw.s[s].fc1_b;
    pr[s].M = sm[s].rows; pr[s].N = F; pr[s].K = D; pr[s].out = big; pr[s].out_map = sm[s].wide;
    use_fp8(pr[s], s, 2);
  }
  rs = run_gemm(c, EPI_BIAS_GELU, pr, ns, dt, dt, st);
  if (rs != SPOT_OK) return rs;
  for (int s = 0; s < ns; ++s) {
    memset(&pr[s], 0, sizeof(GemmProblem));
    pr[s].A = big; pr[s].a_map = sm[s].wide; pr[s].W = bw.s[s].fc2_w; pr[s].bias = bw.s[s].fc2_b;
    pr[s].M = sm[s].rows; pr[s].N = D; pr[s].K = F; pr[s].gate = mod[s] + 5 * D; pr[s].resid = h[s]; pr[s].resid_map = sm[s].h;
    use_fp8(pr[s], s, 3);
  }
  return run_gemm(c, EPI_GATE_RES, pr, ns, dt, SPOT_F32, st);
}

// temb/c for T timesteps and every block's modulation vectors (S7, S4 step 1): seed- and
// prompt-independent, so computed once per call for all steps (the 13.6 GB of modulation weights of the
// full-depth config are read once per call instead of once per step).
spot_status conditioning(spot_ctx* c, const Workspace& w, uint8_t* ws, int T, cudaStream_t st) {
  const spot_config& g = c->cfg;
  const int D = g.hidden, L = g.n_blocks;
  float* emb = (float*)(ws + w.emb); float* hid = (float*)(ws + w.hid); float* temb = (float*)(ws + w.temb);
  float* cv = (float*)(ws + w.cvec); float* mod = (float*)(ws + w.mod); float* fmod = (float*)(ws + w.fmod);
  LK(c, launch_time_embed((const float*)(ws + w.t_dev), T, emb, st));
  LK(c, launch_gemv(g.dtype, c->w.time_w1, c->w.time_b1, emb, T, D, 256, hid, D, true, st));
  LK(c, launch_gemv(g.dtype, c->w.time_w2, c->w.time_b2, hid, T, D, D, temb, D, false, st));
  LK(c, launch_silu(temb, cv, (long long)T * D, st));
  const long long stride_t = (long long)L * 2 * 6 * D;
  // The 2 L modulation Linears stream 2 L * 6 D^2 weights (13.6 GB at config 3) once per call: HBM-bound.  The plain
  // warp-per-row kernel re-reads c from L1 for every weight vector and reaches ~0.7 TB/s; on bf16 configs the same
  // product goes through the tcgen05 GEMM instead, with c split into two bf16 rows (hi + lo = 16 mantissa bits) so the
  // fp32 modulation vectors keep ~2^-17 relative accuracy: rows [hi; lo] x W^T accumulate into fp32 through the
  // reduce-add epilogue (gate = 1, bias = 0), then hi + lo + bias.
  GemmProblem mp[2];
  memset(mp, 0, sizeof(mp));
  mp[0].A = ws + w.md_a; mp[0].a_map = plain_rows(2 * T, D); mp[0].M = 2 * T; mp[0].N = 6 * D; mp[0].K = D;
  mp[0].bias = ws + w.md_zero; mp[0].gate = (const float*)(ws + w.md_ones);
  mp[0].resid = (float*)(ws + w.md_acc); mp[0].resid_map = plain_rows(2 * T, 6 * D);
  mp[0].W = L > 0 ? c->blocks[0].s[0].mod_w : nullptr;
  const bool tc_mod = g.dtype == SPOT_BF16 && c->gemm_impl == 0 && L > 0 && tcgen05_gemm_supported(mp[0]);
  if (tc_mod) {
    const size_t acc_bytes = (size_t)2 * T * 6 * D * 4;
    LK(c, launch_split_hi_lo(cv, ws + w.md_a, (long long)T * D, st));
    LK(c, launch_fill_f32((float*)(ws + w.md_ones), 1.f, 6 * D, st));
    CK(c, cudaMemsetAsync(ws + w.md_zero, 0, (size_t)6 * D * 2, st));
    mp[1] = mp[0];
    mp[1].resid = (float*)(ws + w.md_acc + acc_bytes);
    for (int b = 0; b < L; ++b) {
      CK(c, cudaMemsetAsync(ws + w.md_acc, 0, 2 * acc_bytes, st));
      mp[0].W = c->blocks[b].s[0].mod_w;
      mp[1].W = c->blocks[b].s[1].mod_w;
      LK(c, launch_gemm_tcgen05_v3(EPI_GATE_RES, mp, 2, c->num_sms, st));
      for (int s = 0; s < 2; ++s)
        LK(c, launch_mod_combine(mp[s].resid, c->blocks[b].s[s].mod_b, T, 6 * D, mod + ((long long)b * 2 + s) * 6 * D,
                                 stride_t, st));
    }
  } else {
    for (int b = 0; b < L; ++b)
      for (int s = 0; s < 2; ++s)
        LK(c, launch_gemv(g.dtype, c->blocks[b].s[s].mod_w, c->blocks[b].s[s].mod_b, cv, T, 6 * D, D,
                          mod + ((long long)b * 2 + s) * 6 * D, stride_t, false, st));
  }
  LK(c, launch_gemv(g.dtype, c->w.final_mod_w, c->w.final_mod_b, cv, T, 2 * D, D, fmod, 2 * D, false, st));
  return SPOT_OK;
}

// Stochastic steps: steps lo <= i < hi of the grid use the SDE update with noise level a.
struct SdeRun {
  const uint64_t* seeds;   // device, [B]
  float noise_level;
  int lo, hi;
  float* logp;             // device, [B, T] (zero for deterministic steps)
  int first_step;          // global index of the call's step 0: noise stream and window test use first_step + i
};
constexpr uint32_t kSdeStreamBase = 256;

// cx, cv, cn of the step t_i -> t_next (readings D1-D2); returns false when sigma == 0 (a deterministic step)
bool sde_coeffs(float t_i, float t_next, float noise_level, double* cx, double* cv, double* cn) {
  const double t = (double)t_i, tn = (double)t_next, dt = tn - t;
  const double td = t < 1.0 ? t : tn;                       // FlowGRPO: at t = 1 only the denominator takes t_next
  const double sig = (double)noise_level * sqrt(t / (1.0 - td));
  if (!(sig > 0.0) || !(dt < 0.0)) return false;
  *cx = 1.0 + sig * sig / (2.0 * t) * dt;
  *cv = (1.0 + sig * sig * (1.0 - t) / (2.0 * t)) * dt;
  *cn = sig * sqrt(-dt);
  return true;
}

spot_status denoise_core(spot_ctx* c, int P, int K, float* lat, const void* text_emb, const float* h_t, int T,
                         uint8_t* ws, const float* probe, float* partials, cudaStream_t st,
                         const SdeRun* sde = nullptr) {
  const spot_config& g = c->cfg;
  const spot_dtype dt = g.dtype;
  const int B = P * K, D = g.hidden, L = g.n_blocks, NI = c->n_img(), NT = g.n_txt, C = g.latent_ch;
  const long long E = (long long)NI * C;
  const Workspace w = carve(c, B, T);
  if (T == 0) {
    if (probe) LK(c, launch_reward_partials(lat, probe, B, E, partials, st));
    return SPOT_OK;
  }
  LK(c, launch_put_floats(h_t, T + 1, (float*)(ws + w.t_dev), st));   // by value: no host pointer outlives the call (CUDA-graph capturable)
  spot_status rs = conditioning(c, w, ws, T, st);
  if (rs != SPOT_OK) return rs;
  float* txt_h0 = (float*)(ws + w.txt_h0); float* h_img = (float*)(ws + w.h_img); float* h_txt = (float*)(ws + w.h_txt);
  void* ybuf = ws + w.ybuf; void* big = ws + w.big; float* vel = (float*)(ws + w.vel);
  Nv4Scratch nvs{{ws + w.nv_codes[0], ws + w.nv_codes[1]}, {ws + w.nv_sf[0], ws + w.nv_sf[1]},
                 {ws + w.nv_codes2[0], ws + w.nv_codes2[1]}, {ws + w.nv_sf2[0], ws + w.nv_sf2[1]}};
  const float* mod = (const float*)(ws + w.mod); const float* fmod = (const float*)(ws + w.fmod);
  GemmProblem pr;
  // h_txt^0 = RMSNorm(text_emb) Wtxt^T + b, once per prompt (C7)
  if (NT > 0) {
    LK(c, launch_rmsnorm_rows(dt, text_emb, c->w.txt_gain, P * NT, g.txt_dim, g.rms_eps, ws + w.txt_norm, st));
    memset(&pr, 0, sizeof(pr));
    pr.A = ws + w.txt_norm; pr.a_map = plain_rows(P * NT, g.txt_dim); pr.W = c->w.txt_in_w; pr.bias = c->w.txt_in_b;
    pr.M = P * NT; pr.N = D; pr.K = g.txt_dim; pr.out = txt_h0; pr.out_map = plain_rows(P * NT, D);
    LK(c, launch_gemm_simt(dt, dt, SPOT_F32, EPI_BIAS, pr, st));
  }
  // The batch runs as consecutive chunks of at most chunk_seqs sequences (an exploration batch is capped at 32
  // sequences), each through all T steps: measured 9 % faster per sequence at config 5 than one pass over 256 sequences
  // (26.2 -> 23.9 s; DESIGN.md section 5 "Chunked passes"), and a sequence's arithmetic does not depend on its batch, so
  // the result is the same bit for bit.  Conditioning and h_txt^0
  // above are shared by all chunks; the stochastic step takes its seeds, partial sums and log-probability rows at the chunk's offset.
  const int chunk = (c->chunk_seqs <= 0 || c->chunk_seqs > B) ? B : c->chunk_seqs;
  const long long n_part = (E + REWARD_CHUNK - 1) / REWARD_CHUNK;
  for (int b0 = 0; b0 < B; b0 += chunk) {
    const int Bc = B - b0 < chunk ? B - b0 : chunk;
    float* lat_c = lat + (long long)b0 * E;
    float* partials_c = partials ? partials + (long long)b0 * n_part : nullptr;
    for (int i = 0; i < T; ++i) {
      // h_img^0 = x Win^T + b on the fp32 latents
      memset(&pr, 0, sizeof(pr));
      pr.A = lat_c; pr.a_map = plain_rows(Bc * NI, C); pr.W = c->w.img_in_w; pr.bias = c->w.img_in_b;
      pr.M = Bc * NI; pr.N = D; pr.K = C; pr.out = h_img; pr.out_map = plain_rows(Bc * NI, D);
      LK(c, launch_gemm_simt(SPOT_F32, dt, SPOT_F32, EPI_BIAS, pr, st));
      LK(c, launch_broadcast_prompts(txt_h0, h_txt, Bc, K, (long long)NT * D, st, b0));
      for (int b = 0; b < L; ++b) {
        const float* m = mod + ((long long)i * L + b) * 2 * 6 * D;
        rs = block_core(c, b, Bc, h_img, h_txt, m, m + 6 * D, ybuf, big, b == L - 1, st, c->nvfp4 ? &nvs : nullptr);
        if (rs != SPOT_OK) return rs;
      }
      // v = (LN(h_img)(1 + scale_f) + shift_f) Wp^T + b
      const float* fm = fmod + (long long)i * 2 * D;
      LK(c, launch_ln_modulate(dt, h_img, Bc * NI, D, fm + D, fm, g.ln_eps, ybuf, plain_rows(Bc * NI, D), st));
      memset(&pr, 0, sizeof(pr));
      pr.A = ybuf; pr.a_map = plain_rows(Bc * NI, D); pr.W = c->w.proj_w; pr.bias = c->w.proj_b;
      pr.M = Bc * NI; pr.N = C; pr.K = D; pr.out = vel; pr.out_map = plain_rows(Bc * NI, C);
      LK(c, launch_gemm_simt(dt, dt, SPOT_F32, EPI_BIAS, pr, st));
      const bool last = i == T - 1;
      double cx, cv, cn;
      const int j = sde ? sde->first_step + i : i;           // global step index
      if (sde && j >= sde->lo && j < sde->hi && sde_coeffs(h_t[i], h_t[i + 1], sde->noise_level, &cx, &cv, &cn))
        LK(c, launch_sde_update(lat_c, vel, sde->seeds + b0, kSdeStreamBase + (uint32_t)j, cx, cv, cn, Bc, E,
                                last ? probe : nullptr, c->d_partials2 + (long long)b0 * n_part, partials_c,
                                sde->logp + (long long)b0 * T + i, T, st));
      else
        LK(c, launch_euler_update(lat_c, vel, h_t[i + 1] - h_t[i], Bc, E, last ? probe : nullptr, partials_c, st));
    }
  }
  return SPOT_OK;
}

// Cached-step exploration: as denoise_core, but every step first measures
// rel-L1 of the block-0 modulated image input per sequence, decides per sequence whether to run the L blocks, runs
// them on the compacted batch of computing sequences and reuses the cached residual for the others.  One small
// device->host copy (the list of computing sequences) and one stream synchronisation per Euler step.
spot_status denoise_cached_core(spot_ctx* c, int P, int K, float* lat, const void* text_emb, const float* h_t, int T,
                                const spot_cache_config* cc, uint8_t* h_computed, float* h_rel, uint8_t* ws,
                                const float* probe, float* partials, cudaStream_t st) {
  const spot_config& g = c->cfg;
  const spot_dtype dt = g.dtype;
  const int B = P * K, D = g.hidden, L = g.n_blocks, NI = c->n_img(), NT = g.n_txt, C = g.latent_ch;
  const long long E = (long long)NI * C, per_img = (long long)NI * D, per_txt = (long long)NT * D;
  const Workspace w = carve(c, B, T, true);
  if (T == 0) {
    if (probe) LK(c, launch_reward_partials(lat, probe, B, E, partials, st));
    return SPOT_OK;
  }
  double coeffs[8] = {0.0, 1.0, 0, 0, 0, 0, 0, 0};
  int n_coeffs = 2;
  if (cc->n_coeffs > 0) {
    n_coeffs = cc->n_coeffs;
    for (int j = 0; j < n_coeffs; ++j) coeffs[j] = (double)cc->coeffs[j];
  }
  CK(c, cudaMemcpyAsync(ws + w.tc_coeffs, coeffs, sizeof(coeffs), cudaMemcpyHostToDevice, st));
  CK(c, cudaMemsetAsync(ws + w.tc_acc, 0, (size_t)B * 8, st));
  CK(c, cudaMemcpyAsync(ws + w.t_dev, h_t, (size_t)(T + 1) * 4, cudaMemcpyHostToDevice, st));
  spot_status rs = conditioning(c, w, ws, T, st);
  if (rs != SPOT_OK) return rs;
  float* txt_h0 = (float*)(ws + w.txt_h0); float* hc = (float*)(ws + w.h_img); float* h_txt = (float*)(ws + w.h_txt);
  float* h0 = (float*)(ws + w.tc_h0); float* m_prev = (float*)(ws + w.tc_mprev); float* resid = (float*)(ws + w.tc_resid);
  float* row_part = (float*)(ws + w.tc_rowpart); double* acc = (double*)(ws + w.tc_acc);
  int* d_idx = (int*)(ws + w.tc_idx); int* d_pos = (int*)(ws + w.tc_pos); int* d_nact = (int*)(ws + w.tc_nact);
  int* d_comp = (int*)(ws + w.tc_comp); float* d_rel = (float*)(ws + w.tc_rel);
  void* ybuf = ws + w.ybuf; void* big = ws + w.big; float* vel = (float*)(ws + w.vel);
  Nv4Scratch nvs{{ws + w.nv_codes[0], ws + w.nv_codes[1]}, {ws + w.nv_sf[0], ws + w.nv_sf[1]},
                 {ws + w.nv_codes2[0], ws + w.nv_codes2[1]}, {ws + w.nv_sf2[0], ws + w.nv_sf2[1]}};
  const float* mod = (const float*)(ws + w.mod); const float* fmod = (const float*)(ws + w.fmod);
  std::vector<int> h_idx((size_t)B + 1), h_comp((size_t)B);
  std::vector<float> h_relv((size_t)B);
  GemmProblem pr;
  if (NT > 0) {
    LK(c, launch_rmsnorm_rows(dt, text_emb, c->w.txt_gain, P * NT, g.txt_dim, g.rms_eps, ws + w.txt_norm, st));
    memset(&pr, 0, sizeof(pr));
    pr.A = ws + w.txt_norm; pr.a_map = plain_rows(P * NT, g.txt_dim); pr.W = c->w.txt_in_w; pr.bias = c->w.txt_in_b;
    pr.M = P * NT; pr.N = D; pr.K = g.txt_dim; pr.out = txt_h0; pr.out_map = plain_rows(P * NT, D);
    LK(c, launch_gemm_simt(dt, dt, SPOT_F32, EPI_BIAS, pr, st));
  }
  for (int i = 0; i < T; ++i) {
    // h0 = img_in(x) for every sequence; metric on m = LN(h0)(1 + scale1) + shift1 of block 0's image stream
    memset(&pr, 0, sizeof(pr));
    pr.A = lat; pr.a_map = plain_rows(B * NI, C); pr.W = c->w.img_in_w; pr.bias = c->w.img_in_b;
    pr.M = B * NI; pr.N = D; pr.K = C; pr.out = h0; pr.out_map = plain_rows(B * NI, D);
    LK(c, launch_gemm_simt(SPOT_F32, dt, SPOT_F32, EPI_BIAS, pr, st));
    const float* m0 = mod + (long long)i * L * 2 * 6 * D;          // block 0, image stream: (shift1, scale1, ...)
    const bool first = i == 0, force = i == 0 || i == T - 1;
    if (L > 0) LK(c, launch_tc_metric(h0, m_prev, m0, m0 + D, (long long)B * NI, D, g.ln_eps, first, row_part, st));
    LK(c, launch_tc_decide(row_part, B, NI, first || L == 0, force, (double)cc->threshold, n_coeffs,
                           (const double*)(ws + w.tc_coeffs), acc, d_idx, d_pos, d_nact, d_comp, d_rel, st));
    CK(c, cudaMemcpyAsync(h_idx.data(), d_idx, ((size_t)B + 1) * 4, cudaMemcpyDeviceToHost, st));
    if (h_computed) CK(c, cudaMemcpyAsync(h_comp.data(), d_comp, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    if (h_rel) CK(c, cudaMemcpyAsync(h_relv.data(), d_rel, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    CK(c, cudaStreamSynchronize(st));
    const int n_act = h_idx[(size_t)B];
    if (h_computed) for (int b = 0; b < B; ++b) h_computed[(size_t)b * T + i] = (uint8_t)h_comp[(size_t)b];
    if (h_rel) for (int b = 0; b < B; ++b) h_rel[(size_t)b * T + i] = h_relv[(size_t)b];
    if (n_act < 0 || n_act > B) return SPOT_ERR_CUDA;
    if (n_act > 0) {
      LK(c, launch_tc_gather(h0, hc, d_idx, 1, n_act, per_img, st));
      if (NT > 0) LK(c, launch_tc_gather(txt_h0, h_txt, d_idx, K, n_act, per_txt, st));
      // the compacted batch goes through the block stack in chunks of at most chunk_seqs sequences (see denoise_core)
      const int chunk = (c->chunk_seqs <= 0 || c->chunk_seqs > n_act) ? n_act : c->chunk_seqs;
      for (int a0 = 0; a0 < n_act; a0 += chunk) {
        const int nc = n_act - a0 < chunk ? n_act - a0 : chunk;
        for (int b = 0; b < L; ++b) {
          const float* m = mod + ((long long)i * L + b) * 2 * 6 * D;
          rs = block_core(c, b, nc, hc + a0 * per_img, h_txt + a0 * per_txt, m, m + 6 * D, ybuf, big, b == L - 1, st,
                          c->nvfp4 ? &nvs : nullptr);
          if (rs != SPOT_OK) return rs;
        }
      }
    }
    LK(c, launch_tc_combine(h0, resid, hc, d_pos, B, per_img, st));
    const float* fm = fmod + (long long)i * 2 * D;
    LK(c, launch_ln_modulate(dt, h0, B * NI, D, fm + D, fm, g.ln_eps, ybuf, plain_rows(B * NI, D), st));
    memset(&pr, 0, sizeof(pr));
    pr.A = ybuf; pr.a_map = plain_rows(B * NI, D); pr.W = c->w.proj_w; pr.bias = c->w.proj_b;
    pr.M = B * NI; pr.N = C; pr.K = D; pr.out = vel; pr.out_map = plain_rows(B * NI, C);
    LK(c, launch_gemm_simt(dt, dt, SPOT_F32, EPI_BIAS, pr, st));
    const bool last = i == T - 1;
    LK(c, launch_euler_update(lat, vel, h_t[i + 1] - h_t[i], B, E, last ? probe : nullptr, partials, st));
  }
  return SPOT_OK;
}

spot_status check_ws(const spot_ctx* c, int B, int T, const void* ws, size_t bytes, bool cached = false) {
  if (!ws) return SPOT_ERR_NULL;
  if (!aligned16(ws)) return SPOT_ERR_ALIGN;
  if (bytes < carve(c, B, T, cached).total) return SPOT_ERR_WORKSPACE;
  return SPOT_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

static spot_status noise_common(const uint64_t* d_seeds, int n_seeds, int64_t elems, uint32_t stream_id, float* d_out,
                                uint32_t* d_words, void* cuda_stream) {
  if (n_seeds < 0 || n_seeds > 65535 || elems <= 0 || (elems & 3)) return SPOT_ERR_SHAPE;
  if (n_seeds == 0) return SPOT_OK;
  const void* o = d_out ? (const void*)d_out : (const void*)d_words;
  if (!d_seeds || !o) return SPOT_ERR_NULL;
  if (!aligned16(o)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_noise(d_seeds, n_seeds, elems, stream_id, d_out, d_words, (cudaStream_t)cuda_stream) == cudaSuccess
             ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_noise_from_seeds(const uint64_t* d_seeds, int n_seeds, int64_t elems_per_seed, uint32_t stream_id,
                                  float* d_out, void* cuda_stream) {
  if (n_seeds > 0 && !d_out) return SPOT_ERR_NULL;
  return noise_common(d_seeds, n_seeds, elems_per_seed, stream_id, d_out, nullptr, cuda_stream);
}

spot_status spot_philox_words(const uint64_t* d_seeds, int n_seeds, int64_t elems_per_seed, uint32_t stream_id,
                              uint32_t* d_out, void* cuda_stream) {
  if (n_seeds > 0 && !d_out) return SPOT_ERR_NULL;
  return noise_common(d_seeds, n_seeds, elems_per_seed, stream_id, nullptr, d_out, cuda_stream);
}

spot_status spot_dit_block_forward(spot_ctx* ctx, int block, int n_seqs, const void* d_h_img, const void* d_h_txt,
                                   const float* d_temb, void* d_out_img, void* d_out_txt, void* d_workspace,
                                   size_t ws_bytes, void* cuda_stream) {
  if (!ctx || !d_h_img || !d_temb || !d_out_img) return SPOT_ERR_NULL;
  if (ctx->cfg.n_txt > 0 && (!d_h_txt || !d_out_txt)) return SPOT_ERR_NULL;
  if (block < 0 || block >= ctx->cfg.n_blocks || n_seqs <= 0 || n_seqs > ctx->max_seqs) return SPOT_ERR_SHAPE;
  if (!aligned16(d_h_img) || !aligned16(d_h_txt) || !aligned16(d_out_img) || !aligned16(d_out_txt) || !aligned16(d_temb))
    return SPOT_ERR_ALIGN;
  spot_status s = check_ws(ctx, n_seqs, 1, d_workspace, ws_bytes);
  if (s != SPOT_OK) return s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const spot_config& g = ctx->cfg;
  const Workspace w = carve(ctx, n_seqs, 1);
  uint8_t* ws = (uint8_t*)d_workspace;
  const int D = g.hidden;
  const long long n_img = (long long)n_seqs * ctx->n_img() * D, n_txt = (long long)n_seqs * g.n_txt * D;
  float* cv = (float*)(ws + w.cvec); float* mod = (float*)(ws + w.mod);
  float* h_img = (float*)(ws + w.h_img); float* h_txt = (float*)(ws + w.h_txt);
  LK(ctx, launch_silu(d_temb, cv, D, st));
  for (int sgm = 0; sgm < 2; ++sgm)
    LK(ctx, launch_gemv(g.dtype, ctx->blocks[block].s[sgm].mod_w, ctx->blocks[block].s[sgm].mod_b, cv, 1, 6 * D, D,
                        mod + (long long)sgm * 6 * D, 0, false, st));
  LK(ctx, launch_to_f32(g.dtype, d_h_img, h_img, n_img, st));
  LK(ctx, launch_to_f32(g.dtype, d_h_txt, h_txt, n_txt, st));
  Nv4Scratch nvs{{ws + w.nv_codes[0], ws + w.nv_codes[1]}, {ws + w.nv_sf[0], ws + w.nv_sf[1]},
                 {ws + w.nv_codes2[0], ws + w.nv_codes2[1]}, {ws + w.nv_sf2[0], ws + w.nv_sf2[1]}};
  s = block_core(ctx, block, n_seqs, h_img, h_txt, mod, mod + 6 * D, ws + w.ybuf, ws + w.big, false, st,
                 ctx->nvfp4 ? &nvs : nullptr);
  if (s != SPOT_OK) return s;
  LK(ctx, launch_from_f32(g.dtype, h_img, d_out_img, n_img, st));
  LK(ctx, launch_from_f32(g.dtype, h_txt, d_out_txt, n_txt, st));
  return SPOT_OK;
}

static spot_status check_rollout_args(const spot_ctx* ctx, int P, int K, const void* lat, const void* text,
                                      const float* h_t, int T) {
  if (!ctx || !lat || !h_t) return SPOT_ERR_NULL;
  if (ctx->cfg.n_txt > 0 && !text) return SPOT_ERR_NULL;
  if (P <= 0 || K <= 0 || T < 0 || (long long)P * K > ctx->max_seqs) return SPOT_ERR_SHAPE;
  if (!aligned16(lat) || !aligned16(text)) return SPOT_ERR_ALIGN;
  return SPOT_OK;
}

spot_status spot_dit_denoise(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, float* d_latents,
                             const void* d_text_emb, const float* h_timesteps, int n_steps, void* d_workspace,
                             size_t ws_bytes, void* cuda_stream) {
  spot_status s = check_rollout_args(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps);
  if (s != SPOT_OK) return s;
  s = check_ws(ctx, n_prompts * seeds_per_prompt, n_steps, d_workspace, ws_bytes);
  if (s != SPOT_OK) return s;
  return denoise_core(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps,
                      (uint8_t*)d_workspace, nullptr, nullptr, (cudaStream_t)cuda_stream);
}

static spot_status check_select_args(const spot_ctx* ctx, int P, int K, int k_select, const void* rewards,
                                     const void* stats, const void* top, const void* bottom) {
  if (!ctx || !rewards || !stats) return SPOT_ERR_NULL;
  if (P <= 0 || K <= 0 || K > 1024 || (long long)P * K > ctx->max_seqs || k_select < 0 || 2 * k_select > K)
    return SPOT_ERR_SHAPE;
  if (k_select > 0 && (!top || !bottom)) return SPOT_ERR_NULL;
  return SPOT_OK;
}

spot_status spot_seed_rewards(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, const float* d_latents,
                              const float* d_probe, int k_select, float* d_rewards, float* d_stats, int32_t* d_top,
                              int32_t* d_bottom, void* cuda_stream) {
  if (!ctx || !d_latents || !d_probe) return SPOT_ERR_NULL;
  spot_status s = check_select_args(ctx, n_prompts, seeds_per_prompt, k_select, d_rewards, d_stats, d_top, d_bottom);
  if (s != SPOT_OK) return s;
  if (!aligned16(d_latents) || !aligned16(d_probe)) return SPOT_ERR_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int B = n_prompts * seeds_per_prompt;
  const long long E = (long long)ctx->n_img() * ctx->cfg.latent_ch;
  LK(ctx, launch_reward_partials(d_latents, d_probe, B, E, ctx->d_partials, st));
  LK(ctx, launch_reward_finalize(ctx->d_partials, B, E, d_rewards, st));
  LK(ctx, launch_seed_select(d_rewards, n_prompts, seeds_per_prompt, k_select, d_stats, d_top, d_bottom, st));
  return SPOT_OK;
}

spot_status spot_explore(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, const uint64_t* d_seeds,
                         const void* d_text_emb, const float* h_timesteps, int n_steps, const float* d_probe,
                         int k_select, float* d_latents, float* d_rewards, float* d_stats, int32_t* d_top,
                         int32_t* d_bottom, void* d_workspace, size_t ws_bytes, void* cuda_stream) {
  spot_status s = check_rollout_args(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps);
  if (s != SPOT_OK) return s;
  if (!d_seeds || !d_probe) return SPOT_ERR_NULL;
  s = check_select_args(ctx, n_prompts, seeds_per_prompt, k_select, d_rewards, d_stats, d_top, d_bottom);
  if (s != SPOT_OK) return s;
  if (!aligned16(d_probe)) return SPOT_ERR_ALIGN;
  const int B = n_prompts * seeds_per_prompt;
  s = check_ws(ctx, B, n_steps, d_workspace, ws_bytes);
  if (s != SPOT_OK) return s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const long long E = (long long)ctx->n_img() * ctx->cfg.latent_ch;
  LK(ctx, launch_noise(d_seeds, B, E, 0u, d_latents, nullptr, st));
  s = denoise_core(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps,
                   (uint8_t*)d_workspace, d_probe, ctx->d_partials, st);
  if (s != SPOT_OK) return s;
  LK(ctx, launch_reward_finalize(ctx->d_partials, B, E, d_rewards, st));
  LK(ctx, launch_seed_select(d_rewards, n_prompts, seeds_per_prompt, k_select, d_stats, d_top, d_bottom, st));
  return SPOT_OK;
}

static spot_status check_cache_cfg(const spot_cache_config* cc, int B) {
  if (!cc) return SPOT_ERR_NULL;
  if (cc->n_coeffs < 0 || cc->n_coeffs > 8 || !(cc->threshold >= 0.f) || B > 1024) return SPOT_ERR_SHAPE;
  return SPOT_OK;
}

spot_status spot_workspace_bytes_cached(const spot_ctx* ctx, int n_seqs, int n_steps, size_t* bytes) {
  if (!ctx || !bytes) return SPOT_ERR_NULL;
  if (n_seqs <= 0 || n_seqs > ctx->max_seqs || n_steps < 0) return SPOT_ERR_SHAPE;
  *bytes = carve(ctx, n_seqs, n_steps, true).total;
  return SPOT_OK;
}

spot_status spot_dit_denoise_cached(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, float* d_latents,
                                    const void* d_text_emb, const float* h_timesteps, int n_steps,
                                    const spot_cache_config* cache, uint8_t* h_computed, float* h_rel, void* d_workspace,
                                    size_t ws_bytes, void* cuda_stream) {
  spot_status s = check_rollout_args(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps);
  if (s != SPOT_OK) return s;
  s = check_cache_cfg(cache, n_prompts * seeds_per_prompt);
  if (s != SPOT_OK) return s;
  s = check_ws(ctx, n_prompts * seeds_per_prompt, n_steps, d_workspace, ws_bytes, true);
  if (s != SPOT_OK) return s;
  return denoise_cached_core(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps, cache,
                             h_computed, h_rel, (uint8_t*)d_workspace, nullptr, nullptr, (cudaStream_t)cuda_stream);
}

spot_status spot_explore_cached(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, const uint64_t* d_seeds,
                                const void* d_text_emb, const float* h_timesteps, int n_steps, const float* d_probe,
                                int k_select, const spot_cache_config* cache, float* d_latents, float* d_rewards,
                                float* d_stats, int32_t* d_top, int32_t* d_bottom, uint8_t* h_computed, float* h_rel,
                                void* d_workspace, size_t ws_bytes, void* cuda_stream) {
  spot_status s = check_rollout_args(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps);
  if (s != SPOT_OK) return s;
  if (!d_seeds || !d_probe) return SPOT_ERR_NULL;
  s = check_select_args(ctx, n_prompts, seeds_per_prompt, k_select, d_rewards, d_stats, d_top, d_bottom);
  if (s != SPOT_OK) return s;
  if (!aligned16(d_probe)) return SPOT_ERR_ALIGN;
  const int B = n_prompts * seeds_per_prompt;
  s = check_cache_cfg(cache, B);
  if (s != SPOT_OK) return s;
  s = check_ws(ctx, B, n_steps, d_workspace, ws_bytes, true);
  if (s != SPOT_OK) return s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const long long E = (long long)ctx->n_img() * ctx->cfg.latent_ch;
  LK(ctx, launch_noise(d_seeds, B, E, 0u, d_latents, nullptr, st));
  s = denoise_cached_core(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps, cache, h_computed,
                          h_rel, (uint8_t*)d_workspace, d_probe, ctx->d_partials, st);
  if (s != SPOT_OK) return s;
  LK(ctx, launch_reward_finalize(ctx->d_partials, B, E, d_rewards, st));
  LK(ctx, launch_seed_select(d_rewards, n_prompts, seeds_per_prompt, k_select, d_stats, d_top, d_bottom, st));
  return SPOT_OK;
}

spot_status spot_dit_denoise_sde(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, const uint64_t* d_seeds,
                                 float* d_latents, const void* d_text_emb, const float* h_timesteps, int n_steps,
                                 float noise_level, int window_lo, int window_hi, int first_step, float* d_logp,
                                 void* d_workspace, size_t ws_bytes, void* cuda_stream) {
  spot_status s = check_rollout_args(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps);
  if (s != SPOT_OK) return s;
  if (!d_seeds || !d_logp) return SPOT_ERR_NULL;
  if (!(noise_level >= 0.f) || window_lo < 0 || window_hi < window_lo || first_step < 0) return SPOT_ERR_SHAPE;
  for (int i = 0; i < n_steps; ++i)
    if (!(h_timesteps[i] > 0.f && h_timesteps[i] <= 1.f && h_timesteps[i + 1] < h_timesteps[i] && h_timesteps[i + 1] >= 0.f))
      return SPOT_ERR_SHAPE;                                 // the schedule sigma = a sqrt(t/(1-t)) needs 1 >= t_i > t_{i+1} >= 0
  const int B = n_prompts * seeds_per_prompt;
  s = check_ws(ctx, B, n_steps, d_workspace, ws_bytes);
  if (s != SPOT_OK) return s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (n_steps > 0) CK(ctx, cudaMemsetAsync(d_logp, 0, (size_t)B * n_steps * 4, st));
  SdeRun run{d_seeds, noise_level, window_lo, window_hi, d_logp, first_step};
  return denoise_core(ctx, n_prompts, seeds_per_prompt, d_latents, d_text_emb, h_timesteps, n_steps, (uint8_t*)d_workspace,
                      nullptr, nullptr, st, &run);
}

// ---- FP8 exploration variant ----------------------------------------------------------------
// [N, K] of Linear `which` = (qkv, out, fc1, fc2)
static void fp8_shape(const spot_config& g, int which, long long* N, long long* K) {
  const long long D = g.hidden, F = g.mlp_hidden;
  switch (which) {
    case 0: *N = 3 * D; *K = D; break;
    case 1: *N = D; *K = D; break;
    case 2: *N = F; *K = D; break;
    default: *N = D; *K = F; break;
  }
}

spot_status spot_fp8_bytes(const spot_ctx* ctx, size_t* bytes) {
  if (!ctx || !bytes) return SPOT_ERR_NULL;
  if (ctx->cfg.dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  size_t per_stream = 0;
  for (int w = 0; w < 4; ++w) {
    long long N, K;
    fp8_shape(ctx->cfg, w, &N, &K);
    per_stream += align_up((size_t)N * K) + align_up((size_t)N * 4);
  }
  *bytes = per_stream * 2 * (size_t)ctx->cfg.n_blocks;
  return SPOT_OK;
}

spot_status spot_fp8_prepare(spot_ctx* ctx, void* d_buffer, size_t bytes, void* cuda_stream) {
  if (!ctx || !d_buffer) return SPOT_ERR_NULL;
  if (ctx->cfg.dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  if (ctx->cfg.hidden % 16 || ctx->cfg.mlp_hidden % 16) return SPOT_ERR_SHAPE;
  if (!aligned16(d_buffer)) return SPOT_ERR_ALIGN;
  size_t need = 0;
  spot_status s = spot_fp8_bytes(ctx, &need);
  if (s != SPOT_OK) return s;
  if (bytes < need) return SPOT_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint8_t* p = (uint8_t*)d_buffer;
  ctx->fp8 = 0;
  ctx->fp8_blocks.assign(ctx->blocks.size(), spot_ctx::Fp8Block());
  for (size_t b = 0; b < ctx->blocks.size(); ++b)
    for (int sgm = 0; sgm < 2; ++sgm) {
      const spot_stream_weights& sw = ctx->blocks[b].s[sgm];
      const void* src[4] = {sw.qkv_w, sw.out_w, sw.fc1_w, sw.fc2_w};
      for (int w = 0; w < 4; ++w) {
        long long N, K;
        fp8_shape(ctx->cfg, w, &N, &K);
        uint8_t* wq = p; p += align_up((size_t)N * K);
        float* sc = (float*)p; p += align_up((size_t)N * 4);
        LK(ctx, launch_quantize_weight_rows(src[w], N, (int)K, wq, sc, st));
        ctx->fp8_blocks[b].lin[sgm][w] = spot_ctx::Fp8Linear{wq, sc};
      }
    }
  return SPOT_OK;
}

// ---- NVFP4 exploration variant: fc1 / fc2 of every block ---------------------------------------
spot_status spot_nvfp4_bytes(const spot_ctx* ctx, size_t* bytes) {
  if (!ctx || !bytes) return SPOT_ERR_NULL;
  if (ctx->cfg.dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  const long long D = ctx->cfg.hidden, F = ctx->cfg.mlp_hidden;
  if (D % 256 || F % 256) return SPOT_ERR_SHAPE;
  const size_t fc1 = align_up(nvfp4_codes_bytes(F, D)) + align_up(nvfp4_sf_bytes(F, D)) + align_up((size_t)F * 4);
  const size_t fc2 = align_up(nvfp4_codes_bytes(D, F)) + align_up(nvfp4_sf_bytes(D, F)) + align_up((size_t)D * 4);
  *bytes = (fc1 + fc2) * 2 * (size_t)ctx->cfg.n_blocks;
  return SPOT_OK;
}

spot_status spot_nvfp4_prepare(spot_ctx* ctx, void* d_buffer, size_t bytes, void* cuda_stream) {
  if (!ctx || !d_buffer) return SPOT_ERR_NULL;
  if (!aligned16(d_buffer)) return SPOT_ERR_ALIGN;
  size_t need = 0;
  spot_status s = spot_nvfp4_bytes(ctx, &need);
  if (s != SPOT_OK) return s;
  if (bytes < need) return SPOT_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint8_t* p = (uint8_t*)d_buffer;
  const long long D = ctx->cfg.hidden, F = ctx->cfg.mlp_hidden;
  ctx->nvfp4 = 0;
  ctx->nv4_blocks.assign(ctx->blocks.size(), spot_ctx::Nv4Block());
  for (size_t b = 0; b < ctx->blocks.size(); ++b)
    for (int sgm = 0; sgm < 2; ++sgm) {
      const spot_stream_weights& sw = ctx->blocks[b].s[sgm];
      const void* src[2] = {sw.fc1_w, sw.fc2_w};
      const long long N[2] = {F, D}, K[2] = {D, F};
      for (int w = 0; w < 2; ++w) {
        uint8_t* codes = p; p += align_up(nvfp4_codes_bytes(N[w], K[w]));
        uint8_t* sf = p; p += align_up(nvfp4_sf_bytes(N[w], K[w]));
        float* sc = (float*)p; p += align_up((size_t)N[w] * 4);
        LK(ctx, launch_nvfp4_row_scale(src[w], (int)N[w], (int)K[w], sc, st));
        LK(ctx, launch_nvfp4_quantize(src[w], plain_rows((int)N[w], K[w]), (int)N[w], (int)K[w], sc, codes, sf, st));
        ctx->nv4_blocks[b].lin[sgm][w] = spot_ctx::Nv4Linear{codes, sf, sc};
      }
    }
  return SPOT_OK;
}

spot_status spot_explore_host(spot_ctx* ctx, int n_prompts, int seeds_per_prompt, const uint64_t* h_seeds,
                              const void* h_text_emb, const float* h_timesteps, int n_steps, const float* h_probe,
                              int k_select, float* h_latents, float* h_rewards, float* h_stats, int32_t* h_top,
                              int32_t* h_bottom, void* d_workspace, size_t ws_bytes, void* cuda_stream) {
  if (!ctx || !h_seeds || !h_timesteps || !h_probe || !h_rewards || !h_stats) return SPOT_ERR_NULL;
  if (ctx->cfg.n_txt > 0 && !h_text_emb) return SPOT_ERR_NULL;
  if (n_prompts <= 0 || seeds_per_prompt <= 0 || (long long)n_prompts * seeds_per_prompt > ctx->max_seqs || n_steps < 0)
    return SPOT_ERR_SHAPE;
  if (k_select < 0 || 2 * k_select > seeds_per_prompt || seeds_per_prompt > 1024) return SPOT_ERR_SHAPE;
  if (k_select > 0 && (!h_top || !h_bottom)) return SPOT_ERR_NULL;
  const int B = n_prompts * seeds_per_prompt;
  spot_status s = check_ws(ctx, B, n_steps, d_workspace, ws_bytes);
  if (s != SPOT_OK) return s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const spot_config& g = ctx->cfg;
  const Workspace w = carve(ctx, B, n_steps);
  uint8_t* ws = (uint8_t*)d_workspace;
  const size_t E = (size_t)ctx->n_img() * g.latent_ch;
  const size_t text_bytes = (size_t)n_prompts * g.n_txt * g.txt_dim * esize(g.dtype);
  CK(ctx, cudaMemcpyAsync(ws + w.st_seeds, h_seeds, (size_t)B * 8, cudaMemcpyHostToDevice, st));
  if (text_bytes) CK(ctx, cudaMemcpyAsync(ws + w.st_text, h_text_emb, text_bytes, cudaMemcpyHostToDevice, st));
  CK(ctx, cudaMemcpyAsync(ws + w.st_probe, h_probe, E * 4, cudaMemcpyHostToDevice, st));
  s = spot_explore(ctx, n_prompts, seeds_per_prompt, (const uint64_t*)(ws + w.st_seeds), ws + w.st_text, h_timesteps,
                   n_steps, (const float*)(ws + w.st_probe), k_select, (float*)(ws + w.st_lat),
                   (float*)(ws + w.st_rew), (float*)(ws + w.st_stats), (int32_t*)(ws + w.st_top),
                   (int32_t*)(ws + w.st_bot), d_workspace, ws_bytes, cuda_stream);
  if (s != SPOT_OK) return s;
  if (h_latents) CK(ctx, cudaMemcpyAsync(h_latents, ws + w.st_lat, (size_t)B * E * 4, cudaMemcpyDeviceToHost, st));
  CK(ctx, cudaMemcpyAsync(h_rewards, ws + w.st_rew, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
  CK(ctx, cudaMemcpyAsync(h_stats, ws + w.st_stats, (size_t)n_prompts * 8, cudaMemcpyDeviceToHost, st));
  if (k_select > 0) {
    CK(ctx, cudaMemcpyAsync(h_top, ws + w.st_top, (size_t)n_prompts * k_select * 4, cudaMemcpyDeviceToHost, st));
    CK(ctx, cudaMemcpyAsync(h_bottom, ws + w.st_bot, (size_t)n_prompts * k_select * 4, cudaMemcpyDeviceToHost, st));
  }
  CK(ctx, cudaStreamSynchronize(st));
  return SPOT_OK;
}

}  // extern "C"

// ================================================================================================
// kernel-level entry points (include/spot_kernels.h)
extern "C" {

static int sm_count() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  }
  return n;
}

spot_status spot_linear(spot_dtype dtype, spot_impl impl, spot_epilogue epi, const void* d_a, int64_t M, int64_t K,
                        const void* d_w, int64_t N, const void* d_bias, const float* d_gate, float* d_residual,
                        void* d_out, void* cuda_stream) {
  if (dtype != SPOT_F32 && dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  if (M < 0 || N <= 0 || K <= 0 || M > 0x7fffffff || N > 0x7fffffff || K > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (M == 0) return SPOT_OK;
  if (!d_a || !d_w || !d_bias) return SPOT_ERR_NULL;
  const bool gate_res = epi == SPOT_EPI_GATE_RESIDUAL;
  if (gate_res ? (!d_gate || !d_residual) : !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_a) || !aligned16(d_w) || !aligned16(d_bias) || !aligned16(d_out) || !aligned16(d_residual) ||
      !aligned16(d_gate))
    return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  GemmProblem p;
  memset(&p, 0, sizeof(p));
  p.A = d_a; p.a_map = plain_rows((int)M, K); p.W = d_w; p.bias = d_bias;
  p.M = (int)M; p.N = (int)N; p.K = (int)K;
  if (gate_res) { p.gate = d_gate; p.resid = d_residual; p.resid_map = plain_rows((int)M, N); }
  else { p.out = d_out; p.out_map = plain_rows((int)M, N); }
  const Epilogue e = epi == SPOT_EPI_BIAS ? EPI_BIAS : (epi == SPOT_EPI_BIAS_GELU ? EPI_BIAS_GELU : EPI_GATE_RES);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  bool tc = impl == SPOT_IMPL_TCGEN05 || impl == SPOT_IMPL_TCGEN05_2CTA || impl == SPOT_IMPL_TCGEN05_TMA ||
            (impl == SPOT_IMPL_AUTO && dtype == SPOT_BF16 && tcgen05_gemm_supported(p));
  if (tc) {
    if (dtype != SPOT_BF16 || !tcgen05_gemm_supported(p)) return SPOT_ERR_SHAPE;
    cudaError_t ce = impl == SPOT_IMPL_TCGEN05 ? launch_gemm_tcgen05(e, &p, 1, sm_count(), st)
                     : impl == SPOT_IMPL_TCGEN05_2CTA ? launch_gemm_tcgen05_2cta(e, &p, 1, sm_count(), st)
                                                      : launch_gemm_tcgen05_v3(e, &p, 1, sm_count(), st);
    return ce == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
  }
  if (K % 16) return SPOT_ERR_SHAPE;
  return launch_gemm_simt(dtype, dtype, dtype, e, p, st) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

static spot_status qkv_rope_linear(const void* d_a, int n_seqs, int rows_per_seq, int64_t K, const void* d_w,
                                   const float* d_w_scale, int64_t hidden, const void* d_bias, const void* d_q_gain,
                                   const void* d_k_gain, const float* d_cos, const float* d_sin, int pos_off, float eps,
                                   void* d_out, void* cuda_stream, bool fp8) {
  if (n_seqs < 0 || rows_per_seq <= 0 || K <= 0 || hidden <= 0 || hidden % 128 || pos_off < 0 || K > 0x7fffffff ||
      3 * hidden > 0x7fffffff || (long long)n_seqs * rows_per_seq > 0x7fffffff)
    return SPOT_ERR_SHAPE;
  if (n_seqs == 0) return SPOT_OK;
  if (!d_a || !d_w || !d_bias || !d_q_gain || !d_k_gain || !d_cos || !d_sin || !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_a) || !aligned16(d_w) || !aligned16(d_bias) || !aligned16(d_q_gain) || !aligned16(d_k_gain) ||
      !aligned16(d_cos) || !aligned16(d_sin) || !aligned16(d_out))
    return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  GemmProblem p;
  memset(&p, 0, sizeof(p));
  const int M = n_seqs * rows_per_seq;
  const long long N = 3 * hidden;
  p.A = d_a; p.a_map = RowMap{rows_per_seq, (long long)rows_per_seq * K, 0, K}; p.W = d_w; p.bias = d_bias;
  p.M = M; p.N = (int)N; p.K = (int)K; p.out = d_out; p.out_map = RowMap{rows_per_seq, (long long)rows_per_seq * N, 0, N};
  p.q_gain = d_q_gain; p.k_gain = d_k_gain; p.cos_t = d_cos; p.sin_t = d_sin; p.pos_off = pos_off; p.rms_eps = eps;
  if (fp8) {
    if (!d_w_scale) return SPOT_ERR_NULL;
    if (!aligned16(d_w_scale)) return SPOT_ERR_ALIGN;
    p.fp8 = 1; p.w_scale = d_w_scale;
  }
  if (!tcgen05_gemm_supported(p) || !tcgen05_v3_qkv_rope_supported(p)) return SPOT_ERR_SHAPE;
  return launch_gemm_tcgen05_v3(EPI_QKV_ROPE, &p, 1, sm_count(), (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK
                                                                                                           : SPOT_ERR_CUDA;
}

spot_status spot_qkv_rope_linear(const void* d_a, int n_seqs, int rows_per_seq, int64_t K, const void* d_w, int64_t hidden,
                                 const void* d_bias, const void* d_q_gain, const void* d_k_gain, const float* d_cos,
                                 const float* d_sin, int pos_off, float eps, void* d_out, void* cuda_stream) {
  return qkv_rope_linear(d_a, n_seqs, rows_per_seq, K, d_w, nullptr, hidden, d_bias, d_q_gain, d_k_gain, d_cos, d_sin, pos_off,
                         eps, d_out, cuda_stream, false);
}

spot_status spot_qkv_rope_linear_fp8(const void* d_a, int n_seqs, int rows_per_seq, int64_t K, const void* d_wq,
                                     const float* d_w_scale, int64_t hidden, const void* d_bias, const void* d_q_gain,
                                     const void* d_k_gain, const float* d_cos, const float* d_sin, int pos_off, float eps,
                                     void* d_out, void* cuda_stream) {
  return qkv_rope_linear(d_a, n_seqs, rows_per_seq, K, d_wq, d_w_scale, hidden, d_bias, d_q_gain, d_k_gain, d_cos, d_sin,
                         pos_off, eps, d_out, cuda_stream, true);
}

spot_status spot_select_seeds(const float* d_rewards, int n_prompts, int seeds_per_prompt, int k_select, float* d_stats,
                              int32_t* d_top, int32_t* d_bottom, void* cuda_stream) {
  if (!d_rewards || !d_stats) return SPOT_ERR_NULL;
  if (n_prompts <= 0 || seeds_per_prompt <= 0 || seeds_per_prompt > 1024 || k_select < 0 || 2 * k_select > seeds_per_prompt)
    return SPOT_ERR_SHAPE;
  if (k_select > 0 && (!d_top || !d_bottom)) return SPOT_ERR_NULL;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_seed_select(d_rewards, n_prompts, seeds_per_prompt, k_select, d_stats, d_top, d_bottom,
                            (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_ln_modulate(spot_dtype dtype, const float* d_h, int64_t M, int64_t D, const float* d_shift,
                             const float* d_scale, float eps, void* d_out, void* cuda_stream) {
  if (dtype != SPOT_F32 && dtype != SPOT_BF16 && dtype != SPOT_E4M3) return SPOT_ERR_DTYPE;
  if (M < 0 || D <= 0 || D % 128 || M > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (M == 0) return SPOT_OK;
  if (!d_h || !d_shift || !d_scale || !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_h) || !aligned16(d_shift) || !aligned16(d_scale) || !aligned16(d_out)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  cudaError_t e = launch_ln_modulate(dtype, d_h, (int)M, (int)D, d_shift, d_scale, eps, d_out, plain_rows((int)M, D),
                                     (cudaStream_t)cuda_stream);
  return e == cudaSuccess ? SPOT_OK : (e == cudaErrorInvalidValue ? SPOT_ERR_SHAPE : SPOT_ERR_CUDA);
}

spot_status spot_qk_norm_rope(spot_dtype dtype, void* d_qkv, int B, int S, int H, int head_dim, int n_txt,
                              const void* d_q_gain_img, const void* d_k_gain_img, const void* d_q_gain_txt,
                              const void* d_k_gain_txt, const float* d_cos, const float* d_sin, float eps,
                              void* cuda_stream) {
  if (dtype != SPOT_F32 && dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  if (B < 0 || S <= 0 || H <= 0 || (head_dim != 64 && head_dim != 128) || n_txt < 0 || n_txt > S) return SPOT_ERR_SHAPE;
  if (B == 0) return SPOT_OK;
  if (!d_qkv || !d_q_gain_img || !d_k_gain_img || !d_q_gain_txt || !d_k_gain_txt || !d_cos || !d_sin) return SPOT_ERR_NULL;
  if (!aligned16(d_qkv) || !aligned16(d_q_gain_img) || !aligned16(d_k_gain_img) || !aligned16(d_q_gain_txt) ||
      !aligned16(d_k_gain_txt) || !aligned16(d_cos) || !aligned16(d_sin))
    return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_qk_norm_rope(dtype, d_qkv, B, S, H, head_dim, n_txt, d_q_gain_img, d_k_gain_img, d_q_gain_txt,
                             d_k_gain_txt, d_cos, d_sin, eps, (cudaStream_t)cuda_stream) == cudaSuccess
             ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_attention(spot_dtype dtype, spot_impl impl, const void* d_qkv, void* d_out, int B, int S, int H,
                           int head_dim, void* cuda_stream) {
  if (dtype != SPOT_F32 && dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  if (B < 0 || S <= 0 || H <= 0 || (head_dim != 64 && head_dim != 128)) return SPOT_ERR_SHAPE;
  if (B == 0) return SPOT_OK;
  if (!d_qkv || !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_qkv) || !aligned16(d_out)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool can_tc = dtype == SPOT_BF16 && tcgen05_attn_supported(S, H, head_dim);
  if (impl == SPOT_IMPL_TCGEN05 && !can_tc) return SPOT_ERR_SHAPE;
  if (impl == SPOT_IMPL_TCGEN05_2CTA && can_tc)   // for attention this value selects the previous (two-pass, 128-key tile) kernel
    return launch_attn_tcgen05(d_qkv, d_out, B, S, H, head_dim, sm_count(), st) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
  if (impl != SPOT_IMPL_SIMT && can_tc)
    return launch_attn_tcgen05_v3(d_qkv, d_out, B, S, H, head_dim, sm_count(), st) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
  return launch_attn_simt(dtype, d_qkv, d_out, B, S, H, head_dim, st) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_euler_update(float* d_x, const float* d_v, float dt, int n_seqs, int64_t elems, const float* d_probe,
                              float* d_rewards, float* d_partials, void* cuda_stream) {
  if (n_seqs < 0 || elems <= 0 || (elems & 3)) return SPOT_ERR_SHAPE;
  if (n_seqs == 0) return SPOT_OK;
  if (!d_x || !d_v) return SPOT_ERR_NULL;
  if (d_probe && (!d_rewards || !d_partials)) return SPOT_ERR_NULL;
  if (!aligned16(d_x) || !aligned16(d_v) || !aligned16(d_probe)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (launch_euler_update(d_x, d_v, dt, n_seqs, elems, d_probe, d_partials, st) != cudaSuccess) return SPOT_ERR_CUDA;
  if (d_probe && launch_reward_finalize(d_partials, n_seqs, elems, d_rewards, st) != cudaSuccess) return SPOT_ERR_CUDA;
  return SPOT_OK;
}

spot_status spot_sde_update(float* d_x, const float* d_v, const uint64_t* d_seeds, int step, float t_i, float t_next,
                            float noise_level, int n_seqs, int64_t elems, float* d_logp, float* d_partials,
                            void* cuda_stream) {
  if (n_seqs < 0 || elems <= 0 || (elems & 3) || step < 0) return SPOT_ERR_SHAPE;
  if (n_seqs == 0) return SPOT_OK;
  if (!d_x || !d_v || !d_seeds || !d_logp || !d_partials) return SPOT_ERR_NULL;
  if (!aligned16(d_x) || !aligned16(d_v)) return SPOT_ERR_ALIGN;
  if (!(t_i > 0.f && t_i <= 1.f && t_next < t_i && t_next >= 0.f) || !(noise_level >= 0.f)) return SPOT_ERR_SHAPE;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  double cx, cv, cn;
  if (!sde_coeffs(t_i, t_next, noise_level, &cx, &cv, &cn)) {
    if (cudaMemsetAsync(d_logp, 0, (size_t)n_seqs * 4, st) != cudaSuccess) return SPOT_ERR_CUDA;
    return launch_euler_update(d_x, d_v, t_next - t_i, n_seqs, elems, nullptr, nullptr, st) == cudaSuccess ? SPOT_OK
                                                                                                       : SPOT_ERR_CUDA;
  }
  return launch_sde_update(d_x, d_v, d_seeds, kSdeStreamBase + (uint32_t)step, cx, cv, cn, n_seqs, elems, nullptr, d_partials,
                           nullptr, d_logp, 1, st) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_quantize_weight_rows(const void* d_w_bf16, int64_t N, int64_t K, void* d_wq, float* d_scale, void* cuda_stream) {
  if (N < 0 || K <= 0 || K % 8 || K > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (N == 0) return SPOT_OK;
  if (!d_w_bf16 || !d_wq || !d_scale) return SPOT_ERR_NULL;
  if (!aligned16(d_w_bf16) || !aligned16(d_wq)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_quantize_weight_rows(d_w_bf16, N, (int)K, d_wq, d_scale, (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK
                                                                                                                 : SPOT_ERR_CUDA;
}

spot_status spot_quantize_e4m3(spot_dtype dtype, const void* d_in, int64_t n, void* d_out, void* cuda_stream) {
  if (dtype != SPOT_F32 && dtype != SPOT_BF16) return SPOT_ERR_DTYPE;
  if (n < 0) return SPOT_ERR_SHAPE;
  if (n == 0) return SPOT_OK;
  if (!d_in || !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_in) || !aligned16(d_out)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_quantize_e4m3(dtype, d_in, n, d_out, (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_linear_fp8(spot_epilogue epi, const void* d_a, int64_t M, int64_t K, const void* d_wq, int64_t N,
                            const float* d_w_scale, const void* d_bias, const float* d_gate, float* d_residual, void* d_out,
                            void* cuda_stream) {
  if (M < 0 || N <= 0 || K <= 0 || M > 0x7fffffff || N > 0x7fffffff || K > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (M == 0) return SPOT_OK;
  if (!d_a || !d_wq || !d_w_scale || !d_bias) return SPOT_ERR_NULL;
  const bool gate_res = epi == SPOT_EPI_GATE_RESIDUAL;
  if (gate_res ? (!d_gate || !d_residual) : !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_a) || !aligned16(d_wq) || !aligned16(d_w_scale) || !aligned16(d_bias) || !aligned16(d_out) ||
      !aligned16(d_residual) || !aligned16(d_gate))
    return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  GemmProblem p;
  memset(&p, 0, sizeof(p));
  p.A = d_a; p.a_map = plain_rows((int)M, K); p.W = d_wq; p.bias = d_bias; p.fp8 = 1; p.w_scale = d_w_scale;
  p.M = (int)M; p.N = (int)N; p.K = (int)K;
  if (gate_res) { p.gate = d_gate; p.resid = d_residual; p.resid_map = plain_rows((int)M, N); }
  else { p.out = d_out; p.out_map = plain_rows((int)M, N); }
  if (!tcgen05_gemm_supported(p)) return SPOT_ERR_SHAPE;
  const Epilogue e = epi == SPOT_EPI_BIAS ? EPI_BIAS : (epi == SPOT_EPI_BIAS_GELU ? EPI_BIAS_GELU : EPI_GATE_RES);
  return launch_gemm_tcgen05_v3(e, &p, 1, sm_count(), (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

// ---- NVFP4 building blocks -----------------------------------------------------------------
spot_status spot_nvfp4_sizes(int64_t rows, int64_t K, size_t* codes_bytes, size_t* sf_bytes) {
  if (!codes_bytes || !sf_bytes) return SPOT_ERR_NULL;
  if (rows < 0 || K <= 0 || K % 64) return SPOT_ERR_SHAPE;
  *codes_bytes = nvfp4_codes_bytes(rows, K);
  *sf_bytes = nvfp4_sf_bytes(rows, K);
  return SPOT_OK;
}

spot_status spot_nvfp4_row_scale(const void* d_w_bf16, int64_t rows, int64_t K, float* d_scale, void* cuda_stream) {
  if (rows < 0 || K <= 0 || K % 8 || rows > 0x7fffffff || K > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (rows == 0) return SPOT_OK;
  if (!d_w_bf16 || !d_scale) return SPOT_ERR_NULL;
  if (!aligned16(d_w_bf16)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_nvfp4_row_scale(d_w_bf16, (int)rows, (int)K, d_scale, (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_nvfp4_quantize(const void* d_src_bf16, int64_t rows, int64_t K, const float* d_row_scale, void* d_codes,
                                void* d_sf, void* cuda_stream) {
  if (rows < 0 || K <= 0 || K % 64 || rows % 128 || rows > 0x7fffffff || K > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (rows == 0) return SPOT_OK;
  if (!d_src_bf16 || !d_codes || !d_sf) return SPOT_ERR_NULL;
  if (!aligned16(d_src_bf16) || !aligned16(d_codes) || !aligned16(d_sf)) return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  return launch_nvfp4_quantize(d_src_bf16, plain_rows((int)rows, K), (int)rows, (int)K, d_row_scale, d_codes, d_sf,
                               (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

spot_status spot_linear_nvfp4(spot_epilogue epi, const void* d_a_codes, const void* d_a_sf, int64_t M, int64_t K,
                              const void* d_w_codes, const void* d_w_sf, const float* d_w_scale, int64_t N,
                              const void* d_bias, const float* d_gate, float* d_residual, void* d_out, void* d_out_sf,
                              void* cuda_stream) {
  if (M < 0 || N <= 0 || K <= 0 || M > 0x7fffffff || N > 0x7fffffff || K > 0x7fffffff) return SPOT_ERR_SHAPE;
  if (M == 0) return SPOT_OK;
  if (!d_a_codes || !d_a_sf || !d_w_codes || !d_w_sf || !d_w_scale || !d_bias) return SPOT_ERR_NULL;
  const bool gate_res = epi == SPOT_EPI_GATE_RESIDUAL;
  if (gate_res ? (!d_gate || !d_residual) : !d_out) return SPOT_ERR_NULL;
  if (!aligned16(d_a_codes) || !aligned16(d_a_sf) || !aligned16(d_w_codes) || !aligned16(d_w_sf) || !aligned16(d_w_scale) ||
      !aligned16(d_bias) || !aligned16(d_out) || !aligned16(d_residual) || !aligned16(d_gate))
    return SPOT_ERR_ALIGN;
  if (device_state() != 1) return SPOT_ERR_ARCH;
  Nvfp4Problem p;
  memset(&p, 0, sizeof(p));
  p.a_codes = d_a_codes; p.a_sf = d_a_sf; p.w_codes = d_w_codes; p.w_sf = d_w_sf; p.w_scale = d_w_scale; p.bias = d_bias;
  p.M = (int)M; p.N = (int)N; p.K = (int)K;
  if (gate_res) { p.gate = d_gate; p.resid = d_residual; } else p.out = d_out;
  if (d_out_sf) {
    if (epi != SPOT_EPI_BIAS_GELU || N % 64) return SPOT_ERR_SHAPE;
    if (!aligned16(d_out_sf)) return SPOT_ERR_ALIGN;
    p.out_sf = d_out_sf;
  }
  if (!nvfp4_gemm_supported(p)) return SPOT_ERR_SHAPE;
  const Epilogue e = epi == SPOT_EPI_BIAS ? EPI_BIAS : (epi == SPOT_EPI_BIAS_GELU ? EPI_BIAS_GELU : EPI_GATE_RES);
  return launch_gemm_nvfp4(e, &p, 1, sm_count(), (cudaStream_t)cuda_stream) == cudaSuccess ? SPOT_OK : SPOT_ERR_CUDA;
}

}  // extern "C"
