// elementwise.cu - the HBM-bound kernels: K3 ln_modulate, K4 qk_norm_rope, K6 euler_update(+reward),
// K7 time embedding / skinny Linear, K8 seed selection, and small plumbing kernels.
// Readings S4-S12 of DESIGN.md; paper passages are cited at each kernel.
#include <cuda_fp8.h>
#include <string.h>

#include "kernels.h"

namespace {

// ------------------------------------------------------------------------------------------------
// K7: sinusoidal-256 embedding e(t) = [cos(a f_i) ; sin(a f_i)], a = 1000 t, f_i = 10000^(-i/128)
// (S7).  T is tiny; computed in double so the fp32 result is correctly rounded.
__global__ void time_embed_kernel(const float* __restrict__ t, int T, float* __restrict__ e) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= T * 128) return;
  int step = i / 128, f = i % 128;
  double a = 1000.0 * (double)t[step];
  double freq = exp(-log(10000.0) * (double)f / 128.0);
  e[step * 256 + f] = (float)cos(a * freq);
  e[step * 256 + 128 + f] = (float)sin(a * freq);
}

// out[t, n] = act(sum_k W[n,k] X[t,k] + b[n]); one warp per output row n, X rows fp32 (L1/L2 resident),
// W streamed once with 16-byte loads.  Used for the time MLP and the per-block modulation Linear
// (13.6 GB of weights per call at config 3: HBM-bound, once per call).
template <typename TW, int TT>
__global__ void __launch_bounds__(256) gemv_kernel(const TW* __restrict__ W, const TW* __restrict__ b,
                                                   const float* __restrict__ X, int T, int N, int K,
                                                   float* __restrict__ out, long long out_stride_t, int silu_out) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= N) return;
  constexpr int V = 16 / sizeof(TW);           // elements per 16-byte load
  const TW* wrow = W + (long long)warp * K;
  for (int t0 = 0; t0 < T; t0 += TT) {
    float acc[TT];
#pragma unroll
    for (int t = 0; t < TT; ++t) acc[t] = 0.f;
    for (int k = lane * V; k < K; k += 32 * V) {
      float w[V];
      uint4 raw = *reinterpret_cast<const uint4*>(wrow + k);
      const TW* rw = reinterpret_cast<const TW*>(&raw);
#pragma unroll
      for (int j = 0; j < V; ++j) w[j] = to_f32(rw[j]);
#pragma unroll
      for (int t = 0; t < TT; ++t) {
        if (t0 + t < T) {
          const float* x = X + (long long)(t0 + t) * K + k;
#pragma unroll
          for (int j = 0; j < V; j += 4) {
            float4 xv = *reinterpret_cast<const float4*>(x + j);
            acc[t] = fmaf(w[j], xv.x, acc[t]);
            acc[t] = fmaf(w[j + 1], xv.y, acc[t]);
            acc[t] = fmaf(w[j + 2], xv.z, acc[t]);
            acc[t] = fmaf(w[j + 3], xv.w, acc[t]);
          }
        }
      }
    }
#pragma unroll
    for (int t = 0; t < TT; ++t) {
      float s = warp_sum(acc[t]);
      if (lane == 0 && t0 + t < T) {
        s += to_f32(b[warp]);
        out[(long long)(t0 + t) * out_stride_t + warp] = silu_out ? silu_f(s) : s;
      }
    }
  }
}

__global__ void silu_kernel(const float* __restrict__ in, float* __restrict__ out, long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = silu_f(in[i]);
}

// ------------------------------------------------------------------------------------------------
// K3: y = LN(h) * (1 + scale) + shift; LN over D, biased variance, no affine (S4, "adaLN-
// modulated" in north_star (b)).  One warp per row; the row (fp32 residual stream) is read once into
// registers (NV float4 per lane), mean and variance are two exact passes over registers, the
// output is written once in the activation dtype.  Algorithmic bytes: 4 D read + sizeof(T) D write.
// Up to two problems (the image and the text stream of a block) share one launch: rows [0, M0) belong to p[0].
// Launched with LN_ROWS_PER_CTA warps per CTA; for rows of up to 3072 elements the register cap of 6 resident CTAs
// (168: the 96 row registers plus a window of the scale / shift loads) keeps 12 warps on an SM.
constexpr int LN_ROWS_PER_CTA = 2;
template <typename TO, int NV>
__global__ void __launch_bounds__(32 * LN_ROWS_PER_CTA, NV <= 24 ? 6 : 4) ln_modulate_kernel(const LnProblem p0, const LnProblem p1, int D, float eps) {
  int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  const bool second = row >= p0.M;
  if (second) row -= p0.M;
  // field-by-field selects (constant-bank operands + SEL); a reference to `second ? p1 : p0` makes the compiler copy
  // both parameter structs to local memory and costs 13 % of this bandwidth-bound kernel
  if (row >= (second ? p1.M : p0.M)) return;
  const float* __restrict__ h = second ? p1.h : p0.h;
  const float* __restrict__ shift = second ? p1.shift : p0.shift;
  const float* __restrict__ scale = second ? p1.scale : p0.scale;
  TO* __restrict__ out = reinterpret_cast<TO*>(second ? p1.out : p0.out);
  RowMap omap;
  omap.rows_per_seq = second ? p1.out_map.rows_per_seq : p0.out_map.rows_per_seq;
  omap.seq_stride = second ? p1.out_map.seq_stride : p0.out_map.seq_stride;
  omap.offset = second ? p1.out_map.offset : p0.out_map.offset;
  omap.ld = second ? p1.out_map.ld : p0.out_map.ld;
  const float4* src = reinterpret_cast<const float4*>(h + (long long)row * D);
  float4 v[NV];
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    v[i] = __ldg(src + lane + 32 * i);
    s += (v[i].x + v[i].y) + (v[i].z + v[i].w);
  }
  const float mean = warp_sum(s) / (float)D;
  float q = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    float a = v[i].x - mean, b = v[i].y - mean, c = v[i].z - mean, d = v[i].w - mean;
    q += (a * a + b * b) + (c * c + d * d);
  }
  const float rstd = rsqrtf(warp_sum(q) / (float)D + eps);
  TO* dst = out + omap.row(row);
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int col = 4 * (lane + 32 * i);
    float4 sc = __ldg(reinterpret_cast<const float4*>(scale + col));   // read-only path: not ordered behind the stores to `out`
    float4 sh = __ldg(reinterpret_cast<const float4*>(shift + col));   // (the pointers are selected values, so __restrict__ is lost)
    float y0 = (v[i].x - mean) * rstd * (1.f + sc.x) + sh.x;
    float y1 = (v[i].y - mean) * rstd * (1.f + sc.y) + sh.y;
    float y2 = (v[i].z - mean) * rstd * (1.f + sc.z) + sh.z;
    float y3 = (v[i].w - mean) * rstd * (1.f + sc.w) + sh.w;
    if constexpr (sizeof(TO) == 4) {
      *reinterpret_cast<float4*>(dst + col) = make_float4(y0, y1, y2, y3);
    } else if constexpr (sizeof(TO) == 1) {               // E4M3, unit scale, saturating (DESIGN.md section 13 reading Q3)
      const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(y0, y1), __NV_SATFINITE, __NV_E4M3);
      const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(y2, y3), __NV_SATFINITE, __NV_E4M3);
      *reinterpret_cast<uint32_t*>(dst + col) = lo | (hi << 16);
    } else {
      __nv_bfloat162 p0 = __floats2bfloat162_rn(y0, y1), p1 = __floats2bfloat162_rn(y2, y3);
      uint2 pk = make_uint2(*reinterpret_cast<uint32_t*>(&p0), *reinterpret_cast<uint32_t*>(&p1));
      *reinterpret_cast<uint2*>(dst + col) = pk;
    }
  }
}

// RMSNorm over rows with a gain (text_emb -> txt_in input, S4/C7); once per call.
template <typename T>
__global__ void __launch_bounds__(256) rmsnorm_rows_kernel(const T* __restrict__ in, const T* __restrict__ gain,
                                                           int M, int D, float eps, T* __restrict__ out) {
  const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (row >= M) return;
  const T* src = in + (long long)row * D;
  float q = 0.f;
  for (int k = lane; k < D; k += 32) { float x = to_f32(src[k]); q += x * x; }
  const float r = rsqrtf(warp_sum(q) / (float)D + eps);
  for (int k = lane; k < D; k += 32) out[(long long)row * D + k] = from_f32<T>(to_f32(src[k]) * r * to_f32(gain[k]));
}

}  // namespace

namespace {

// ------------------------------------------------------------------------------------------------
// K4: q <- RoPE(RMSNorm(q) * g_q), k likewise, in place on qkv [B, S, 3, H, d_h] (north_star (c);
// DESIGN.md S4 step 4-5, S5).  A warp owns HPW consecutive heads of one token: lanes 0-15 hold q,
// lanes 16-31 hold k, EPL = d_h / 16 consecutive elements per lane (16 bytes for bf16 d_h = 128, and
// for fp32 d_h = 64), so every global access is a 128-bit load/store and the RMS reduction is 4
// shuffles.  The HPW row loads are issued back to back before any arithmetic (HPW x 16 B in flight
// per thread), and the gain and the rotation pair of the token are read once per warp, as 128-bit
// loads, and reused for the HPW heads.
// Algorithmic bytes: read + write of q and k = 4 * sizeof(T) * d_h per (token, head).
template <typename T, int EPL, int HPW>
__global__ void __launch_bounds__(256) qk_norm_rope_kernel(T* __restrict__ qkv, long long n_warps, int S, int H,
                                                           int n_txt, const T* __restrict__ qg_img,
                                                           const T* __restrict__ kg_img, const T* __restrict__ qg_txt,
                                                           const T* __restrict__ kg_txt, const float* __restrict__ cos_t,
                                                           const float* __restrict__ sin_t, float eps) {
  constexpr int DH = EPL * 16;
  constexpr bool VEC = sizeof(T) * EPL == 16;
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= n_warps) return;
  const int lane = threadIdx.x & 31, part = lane >> 4, sub = lane & 15;
  const int groups = H / HPW;
  const long long tok = w / groups;
  const int head0 = (int)(w - tok * groups) * HPW, s = (int)(tok % S);
  T* ptr = qkv + (tok * 3 + part) * (long long)(H * DH) + head0 * DH + sub * EPL;
  const T* gain = (s < n_txt ? (part ? kg_txt : qg_txt) : (part ? kg_img : qg_img)) + sub * EPL;
  const float* cs = cos_t + (long long)s * (DH / 2) + sub * (EPL / 2);
  const float* sn = sin_t + (long long)s * (DH / 2) + sub * (EPL / 2);
  float x[HPW][EPL], g[EPL], c[EPL / 2], d[EPL / 2];
  if constexpr (VEC) {
    uint4 raw[HPW];
#pragma unroll
    for (int h = 0; h < HPW; ++h) raw[h] = *reinterpret_cast<const uint4*>(ptr + h * DH);
    const uint4 graw = __ldg(reinterpret_cast<const uint4*>(gain));
#pragma unroll
    for (int j = 0; j < EPL; ++j) g[j] = to_f32(reinterpret_cast<const T*>(&graw)[j]);
#pragma unroll
    for (int h = 0; h < HPW; ++h)
#pragma unroll
      for (int j = 0; j < EPL; ++j) x[h][j] = to_f32(reinterpret_cast<const T*>(&raw[h])[j]);
  } else if constexpr (sizeof(T) * EPL == 32) {  // fp32, d_h = 128: two 128-bit accesses per lane and row
    static_assert(sizeof(T) == 4, "32 bytes per lane is the fp32 d_h = 128 case");
#pragma unroll
    for (int h = 0; h < HPW; ++h)
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const float4 v = *reinterpret_cast<const float4*>(ptr + h * DH + 4 * k);
        x[h][4 * k] = v.x; x[h][4 * k + 1] = v.y; x[h][4 * k + 2] = v.z; x[h][4 * k + 3] = v.w;
      }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(gain) + k);
      g[4 * k] = v.x; g[4 * k + 1] = v.y; g[4 * k + 2] = v.z; g[4 * k + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int h = 0; h < HPW; ++h)
#pragma unroll
      for (int j = 0; j < EPL; ++j) x[h][j] = to_f32(ptr[h * DH + j]);
#pragma unroll
    for (int j = 0; j < EPL; ++j) g[j] = to_f32(gain[j]);
  }
  if constexpr (EPL % 8 == 0) {  // EPL / 2 floats per table = whole float4s, 16-byte aligned
#pragma unroll
    for (int j = 0; j < EPL / 8; ++j) {
      const float4 cv = __ldg(reinterpret_cast<const float4*>(cs) + j);
      const float4 dv = __ldg(reinterpret_cast<const float4*>(sn) + j);
      c[4 * j] = cv.x; c[4 * j + 1] = cv.y; c[4 * j + 2] = cv.z; c[4 * j + 3] = cv.w;
      d[4 * j] = dv.x; d[4 * j + 1] = dv.y; d[4 * j + 2] = dv.z; d[4 * j + 3] = dv.w;
    }
  } else {
#pragma unroll
    for (int j = 0; j < EPL / 2; ++j) { c[j] = __ldg(cs + j); d[j] = __ldg(sn + j); }
  }
#pragma unroll
  for (int h = 0; h < HPW; ++h) {
    float q = 0.f;
#pragma unroll
    for (int j = 0; j < EPL; ++j) q += x[h][j] * x[h][j];
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    const float r = rsqrtf(q / (float)DH + eps);
    float y[EPL];
#pragma unroll
    for (int j = 0; j < EPL / 2; ++j) {
      float a = x[h][2 * j] * r * g[2 * j], b = x[h][2 * j + 1] * r * g[2 * j + 1];
      y[2 * j] = a * c[j] - b * d[j];
      y[2 * j + 1] = a * d[j] + b * c[j];
    }
    if constexpr (VEC) {
      uint4 o;
#pragma unroll
      for (int j = 0; j < EPL; ++j) reinterpret_cast<T*>(&o)[j] = from_f32<T>(y[j]);
      *reinterpret_cast<uint4*>(ptr + h * DH) = o;
    } else if constexpr (sizeof(T) * EPL == 32) {
#pragma unroll
      for (int k = 0; k < 2; ++k)
        *reinterpret_cast<float4*>(ptr + h * DH + 4 * k) = make_float4(y[4 * k], y[4 * k + 1], y[4 * k + 2], y[4 * k + 3]);
    } else {
#pragma unroll
      for (int j = 0; j < EPL; ++j) ptr[h * DH + j] = from_f32<T>(y[j]);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// K6: x <- x + dt * v ("refines a latent representation over a fixed number of denoising
// steps"; S8) and, when probe != nullptr, the partial sums of r_b = <p, x_b> (PAPER.md:61
// "per-sample scalar reward r_k"; S9) in a fixed order: block (b, chunk) reduces REWARD_CHUNK
// elements thread-serially, then by a shuffle tree, then over 8 warps in index order.  No atomics, so
// the reward is bit-identical run to run and independent of the batch (determinism contract).
template <bool UPDATE>
__global__ void __launch_bounds__(256) euler_reward_kernel(float* __restrict__ x, const float* __restrict__ v,
                                                           float dt, long long E, const float* __restrict__ probe,
                                                           float* __restrict__ partials, int n_chunks) {
  const int b = blockIdx.y, chunk = blockIdx.x;
  const long long base = (long long)b * E;
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < REWARD_CHUNK / (256 * 4); ++i) {
    long long e = (long long)chunk * REWARD_CHUNK + (i * 256 + threadIdx.x) * 4;
    if (e < E) {
      float4 xv = *reinterpret_cast<float4*>(x + base + e);
      if (UPDATE) {
        float4 vv = *reinterpret_cast<const float4*>(v + base + e);
        xv.x = fmaf(dt, vv.x, xv.x); xv.y = fmaf(dt, vv.y, xv.y);
        xv.z = fmaf(dt, vv.z, xv.z); xv.w = fmaf(dt, vv.w, xv.w);
        *reinterpret_cast<float4*>(x + base + e) = xv;
      }
      if (probe) {
        float4 p = *reinterpret_cast<const float4*>(probe + e);
        acc += (p.x * xv.x + p.y * xv.y) + (p.z * xv.z + p.w * xv.w);
      }
    }
  }
  if (probe) {
    __shared__ float ws[8];
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
      float s = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) s += ws[i];
      partials[(long long)b * n_chunks + chunk] = s;
    }
  }
}

__global__ void reward_finalize_kernel(const float* __restrict__ partials, int B, int n_chunks, double inv_norm,
                                       float* __restrict__ rewards) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  double s = 0.0;
  for (int i = 0; i < n_chunks; ++i) s += (double)partials[(long long)b * n_chunks + i];
  rewards[b] = (float)(s * inv_norm);
}

// K8: per-prompt mean, population std, top-k / bottom-k ("top-k/bottom-k strategy ...
// retaining the highest- and lowest-scoring seeds", :67 "top and bottom K/2", :175 sigma_g; DESIGN.md
// S10-S11: ties -> lower index first).  One block per prompt, rank by counting (K <= 1024).
__global__ void __launch_bounds__(1024) seed_select_kernel(const float* __restrict__ rewards, int K, int k_select,
                                                           float* __restrict__ stats, int32_t* __restrict__ top,
                                                           int32_t* __restrict__ bottom) {
  __shared__ float r[1024];
  const int p = blockIdx.x, i = threadIdx.x;
  if (i < K) r[i] = rewards[(long long)p * K + i];
  __syncthreads();
  if (i < K) {
    int above = 0, below = 0;
    const float ri = r[i];
    for (int j = 0; j < K; ++j) {
      float rj = r[j];
      above += (rj > ri) || (rj == ri && j < i);
      below += (rj < ri) || (rj == ri && j < i);
    }
    if (above < k_select) top[(long long)p * k_select + above] = i;
    if (below < k_select) bottom[(long long)p * k_select + below] = i;
  }
  if (i == 0) {
    double m = 0.0, q = 0.0;
    for (int j = 0; j < K; ++j) m += (double)r[j];
    m /= (double)K;
    for (int j = 0; j < K; ++j) { double d = (double)r[j] - m; q += d * d; }
    stats[2 * p] = (float)m;
    stats[2 * p + 1] = (float)sqrt(q / (double)K);
  }
}

// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void to_f32_kernel(const T* __restrict__ in, float* __restrict__ out, long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < n; i += stride) out[i] = to_f32(in[i]);
}
template <typename T>
__global__ void from_f32_kernel(const float* __restrict__ in, T* __restrict__ out, long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < n; i += stride) out[i] = from_f32<T>(in[i]);
}
// dst[b, :] = src[b / K, :]  (the prompt's text stream h_txt^0 is shared by its K seeds)
__global__ void broadcast_prompts_kernel(const float4* __restrict__ src, float4* __restrict__ dst, int K,
                                         long long n4, long long total4, int first_seq) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < total4; i += stride) {
    long long b = i / n4, e = i - b * n4;
    dst[i] = src[((b + first_seq) / K) * n4 + e];   // dst row b holds sequence first_seq + b of the call
  }
}

inline int grid_for(long long n, int block, int cap = 148 * 16) {
  long long g = (n + block - 1) / block;
  return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

}  // namespace

// ================================================================================================
// launchers
cudaError_t launch_time_embed(const float* d_t, int T, float* d_e, cudaStream_t st) {
  if (T <= 0) return cudaSuccess;
  time_embed_kernel<<<(T * 128 + 127) / 128, 128, 0, st>>>(d_t, T, d_e);
  return cudaGetLastError();
}

cudaError_t launch_gemv(spot_dtype wdt, const void* W, const void* b, const float* X, int T, int N, int K,
                        float* out, long long out_stride_t, bool silu_out, cudaStream_t st) {
  if (T <= 0 || N <= 0) return cudaSuccess;
  const int grid = (N + 7) / 8;
  if (wdt == SPOT_F32) {
    if (K % 4) return cudaErrorInvalidValue;
    gemv_kernel<float, 4><<<grid, 256, 0, st>>>((const float*)W, (const float*)b, X, T, N, K, out, out_stride_t, silu_out);
  } else {
    if (K % 8) return cudaErrorInvalidValue;
    gemv_kernel<bf16, 4><<<grid, 256, 0, st>>>((const bf16*)W, (const bf16*)b, X, T, N, K, out, out_stride_t, silu_out);
  }
  return cudaGetLastError();
}

cudaError_t launch_silu(const float* in, float* out, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  silu_kernel<<<(int)((n + 255) / 256), 256, 0, st>>>(in, out, n);
  return cudaGetLastError();
}

template <typename TO>
static cudaError_t ln_dispatch(const LnProblem& p0, const LnProblem& p1, int D, float eps, cudaStream_t st) {
  // 2 rows per CTA, 6 CTAs = 12 warps per SM (the launch bounds cap the kernel at 168 registers; left alone the compiler
  // hoists every scale / shift load and takes 248, i.e. 8 warps): 5.94 TB/s at config 3, against 5.59 uncapped, 4.95 with one
  // 256-thread CTA and 4.55 with a CTA per row spread over 256 threads; with the cap in place 1, 2 or 4 rows per CTA (12
  // warps per SM each) time the same to 0.1 us: the kernel sits on the DRAM roof
  constexpr int blk = 32 * LN_ROWS_PER_CTA;
  const int wpb = blk / 32, grid = (p0.M + p1.M + wpb - 1) / wpb;
#define LN_CASE(nv)                                                                                     \
  case nv:                                                                                              \
    ln_modulate_kernel<TO, nv><<<grid, blk, 0, st>>>(p0, p1, D, eps);                                   \
    break;
  switch (D / 128) {
    LN_CASE(1) LN_CASE(2) LN_CASE(4) LN_CASE(8) LN_CASE(12) LN_CASE(16) LN_CASE(24) LN_CASE(32)
    default: return cudaErrorInvalidValue;
  }
#undef LN_CASE
  return cudaGetLastError();
}

cudaError_t launch_ln_modulate2(spot_dtype odt, const LnProblem* probs, int n_probs, int D, float eps, cudaStream_t st) {
  if (n_probs < 1 || n_probs > 2 || D % 128) return cudaErrorInvalidValue;
  LnProblem p0 = probs[0], p1;
  memset(&p1, 0, sizeof(p1));
  if (n_probs == 2) p1 = probs[1];
  if (p0.M < 0 || p1.M < 0) return cudaErrorInvalidValue;
  if (p0.M == 0) { p0 = p1; p1.M = 0; }
  if (p0.M == 0) return cudaSuccess;
  if (odt == SPOT_E4M3) return ln_dispatch<uint8_t>(p0, p1, D, eps, st);
  return odt == SPOT_F32 ? ln_dispatch<float>(p0, p1, D, eps, st) : ln_dispatch<bf16>(p0, p1, D, eps, st);
}

cudaError_t launch_ln_modulate(spot_dtype odt, const float* h, int M, int D, const float* shift, const float* scale,
                               float eps, void* out, RowMap out_map, cudaStream_t st) {
  if (M <= 0) return cudaSuccess;
  LnProblem p{h, M, shift, scale, out, out_map};
  return launch_ln_modulate2(odt, &p, 1, D, eps, st);
}

cudaError_t launch_rmsnorm_rows(spot_dtype dt, const void* in, const void* gain, int M, int D, float eps, void* out,
                                cudaStream_t st) {
  if (M <= 0) return cudaSuccess;
  const int grid = (M + 7) / 8;
  if (dt == SPOT_F32)
    rmsnorm_rows_kernel<float><<<grid, 256, 0, st>>>((const float*)in, (const float*)gain, M, D, eps, (float*)out);
  else
    rmsnorm_rows_kernel<bf16><<<grid, 256, 0, st>>>((const bf16*)in, (const bf16*)gain, M, D, eps, (bf16*)out);
  return cudaGetLastError();
}

cudaError_t launch_qk_norm_rope(spot_dtype dt, void* qkv, int B, int S, int H, int dh, int n_txt,
                                const void* qg_img, const void* kg_img, const void* qg_txt, const void* kg_txt,
                                const float* cos_t, const float* sin_t, float eps, cudaStream_t st) {
  const long long n_heads = (long long)B * S * H;
  if (n_heads <= 0) return cudaSuccess;
  const int hpw = H % 4 == 0 ? 4 : H % 2 == 0 ? 2 : 1;  // heads per warp
  const long long n = n_heads / hpw;
  const long long blocks = (n + 7) / 8;
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
#define QK_LAUNCH(T, EPL, HPW)                                                                                  \
  qk_norm_rope_kernel<T, EPL, HPW><<<(int)blocks, 256, 0, st>>>((T*)qkv, n, S, H, n_txt, (const T*)qg_img,      \
                                                                (const T*)kg_img, (const T*)qg_txt,             \
                                                                (const T*)kg_txt, cos_t, sin_t, eps)
#define QK_CASE(T, EPL)                                                                                        \
  do {                                                                                                         \
    if (hpw == 4) QK_LAUNCH(T, EPL, 4);                                                                        \
    else if (hpw == 2) QK_LAUNCH(T, EPL, 2);                                                                   \
    else QK_LAUNCH(T, EPL, 1);                                                                                 \
  } while (0)
  if (dt == SPOT_F32 && dh == 64) QK_CASE(float, 4);
  else if (dt == SPOT_F32 && dh == 128) QK_CASE(float, 8);
  else if (dt == SPOT_BF16 && dh == 64) QK_CASE(bf16, 4);
  else if (dt == SPOT_BF16 && dh == 128) QK_CASE(bf16, 8);
  else return cudaErrorInvalidValue;
#undef QK_LAUNCH
#undef QK_CASE
  return cudaGetLastError();
}

static inline int reward_chunks(long long E) { return (int)((E + REWARD_CHUNK - 1) / REWARD_CHUNK); }

cudaError_t launch_euler_update(float* x, const float* v, float dt, int B, long long E, const float* probe,
                                float* partials, cudaStream_t st) {
  if (B <= 0 || E <= 0) return cudaSuccess;
  const int nc = reward_chunks(E);
  euler_reward_kernel<true><<<dim3(nc, B), 256, 0, st>>>(x, v, dt, E, probe, partials, nc);
  return cudaGetLastError();
}

cudaError_t launch_reward_partials(const float* x, const float* probe, int B, long long E, float* partials,
                                   cudaStream_t st) {
  if (B <= 0 || E <= 0) return cudaSuccess;
  const int nc = reward_chunks(E);
  euler_reward_kernel<false><<<dim3(nc, B), 256, 0, st>>>(const_cast<float*>(x), nullptr, 0.f, E, probe, partials, nc);
  return cudaGetLastError();
}

cudaError_t launch_reward_finalize(const float* partials, int B, long long E, float* rewards, cudaStream_t st) {
  if (B <= 0) return cudaSuccess;
  reward_finalize_kernel<<<(B + 127) / 128, 128, 0, st>>>(partials, B, reward_chunks(E), 1.0 / sqrt((double)E), rewards);
  return cudaGetLastError();
}

cudaError_t launch_seed_select(const float* rewards, int P, int K, int k_select, float* stats, int32_t* top,
                               int32_t* bottom, cudaStream_t st) {
  if (P <= 0) return cudaSuccess;
  if (K > 1024 || K <= 0) return cudaErrorInvalidValue;
  seed_select_kernel<<<P, ((K + 31) / 32) * 32, 0, st>>>(rewards, K, k_select, stats, top, bottom);
  return cudaGetLastError();
}

cudaError_t launch_to_f32(spot_dtype dt, const void* in, float* out, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  if (dt == SPOT_F32) return cudaMemcpyAsync(out, in, n * 4, cudaMemcpyDeviceToDevice, st);
  to_f32_kernel<bf16><<<grid_for(n, 256), 256, 0, st>>>((const bf16*)in, out, n);
  return cudaGetLastError();
}

cudaError_t launch_from_f32(spot_dtype dt, const float* in, void* out, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  if (dt == SPOT_F32) return cudaMemcpyAsync(out, in, n * 4, cudaMemcpyDeviceToDevice, st);
  from_f32_kernel<bf16><<<grid_for(n, 256), 256, 0, st>>>(in, (bf16*)out, n);
  return cudaGetLastError();
}

cudaError_t launch_broadcast_prompts(const float* src, float* dst, int B, int K, long long n_per_prompt, cudaStream_t st,
                                     int first_seq) {
  const long long n4 = n_per_prompt / 4, total4 = n4 * B;
  if (total4 <= 0) return cudaSuccess;
  broadcast_prompts_kernel<<<grid_for(total4, 256), 256, 0, st>>>((const float4*)src, (float4*)dst, K, n4, total4, first_seq);
  return cudaGetLastError();
}

namespace {

// c [rows, D] fp32 -> A [2 * rows, D] bf16: rows 0..rows-1 = hi = bf16(c), rows rows..2 rows-1 = lo = bf16(c - hi), so that
// hi + lo carries 16 mantissa bits of c through a bf16 tensor-core GEMM (used for the modulation Linears, K7)
__global__ void split_hi_lo_kernel(const float* __restrict__ c, bf16* __restrict__ a, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float x = c[i];
  const bf16 hi = __float2bfloat16_rn(x);
  a[i] = hi;
  a[n + i] = __float2bfloat16_rn(x - __bfloat162float(hi));
}

__global__ void fill_f32_kernel(float* __restrict__ p, float v, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// up to 64 host floats travel as KERNEL ARGUMENTS: no host pointer is read after the launch call returns, so a rollout
// captured into a CUDA graph carries its timestep grid with it
struct Floats64 { float v[64]; };
__global__ void put_floats_kernel(Floats64 a, int n, float* __restrict__ p) {
  if ((int)threadIdx.x < n) p[threadIdx.x] = a.v[threadIdx.x];
}

// out[t * stride_t + n] = acc[t, n] + acc[T + t, n] + bias[n]   (hi and lo halves of the split GEMM, then the bias)
template <typename TB>
__global__ void mod_combine_kernel(const float* __restrict__ acc, const TB* __restrict__ bias, int T, int N,
                                   float* __restrict__ out, long long stride_t) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)T * N) return;
  const int t = (int)(i / N), n = (int)(i - (long long)t * N);
  out[(long long)t * stride_t + n] = (acc[(long long)t * N + n] + acc[(long long)(T + t) * N + n]) + to_f32(bias[n]);
}

}  // namespace

cudaError_t launch_split_hi_lo(const float* c, void* a_bf16, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  split_hi_lo_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(c, (bf16*)a_bf16, n);
  return cudaGetLastError();
}

cudaError_t launch_put_floats(const float* h_src, int n, float* d_dst, cudaStream_t st) {
  for (int i0 = 0; i0 < n; i0 += 64) {
    Floats64 a;
    const int m = n - i0 < 64 ? n - i0 : 64;
    for (int i = 0; i < 64; ++i) a.v[i] = i < m ? h_src[i0 + i] : 0.f;
    put_floats_kernel<<<1, 64, 0, st>>>(a, m, d_dst + i0);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_fill_f32(float* p, float v, long long n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  fill_f32_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, v, n);
  return cudaGetLastError();
}

cudaError_t launch_mod_combine(const float* acc, const void* bias_bf16, int T, int N, float* out, long long stride_t,
                               cudaStream_t st) {
  const long long n = (long long)T * N;
  if (n <= 0) return cudaSuccess;
  mod_combine_kernel<bf16><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(acc, (const bf16*)bias_bf16, T, N, out, stride_t);
  return cudaGetLastError();
}
