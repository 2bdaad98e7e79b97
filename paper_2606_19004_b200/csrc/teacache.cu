// teacache.cu - kernels of the cached-step exploration variant ("we control effective denoising
// steps via a caching strategy ... caches and reuses intermediate transformer outputs across adjacent denoising
// steps when their residual difference falls below a threshold", readings T1-T5).
//
// Per Euler step the rule needs, per sequence, rel = mean|m_i - m_{i-1}| / mean|m_{i-1}| of the block-0 modulated
// image input m = LN(h0)(1 + scale1) + shift1, an accumulate-and-compare decision, and either the L blocks (for the
// sequences that compute) or h0 + cached residual (for those that skip).  Sequences decide independently (a request
// is one prompt x one seed), so the batch becomes ragged: the computing sequences are gathered into a compact
// batch, run through the ordinary block kernels, and scattered back.  All of this is HBM-bound and runs once per
// Euler step (three passes over [B, N_img, D] fp32 against 60 blocks of GEMMs), so the kernels are plain
// coalesced float4 loops; reductions use a fixed order (no atomics): bit-identical run to run.
#include "kernels.h"

namespace {

// One warp per image-token row: m = LN(h0)(1 + scale) + shift (fp32, exact two-pass statistics as K3), the row's
// sum|m - m_prev| and sum|m_prev| -> row_part[row] = (sd, sp), then m_prev <- m.  first != 0: m_prev is unset, sums = 0.
__global__ void __launch_bounds__(256) tc_metric_kernel(const float* __restrict__ h0, float* __restrict__ m_prev,
                                                        const float* __restrict__ shift, const float* __restrict__ scale,
                                                        long long rows, int D, float eps, int first,
                                                        float2* __restrict__ row_part) {
  const long long row = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (row >= rows) return;
  const int lane = threadIdx.x & 31;
  const float4* x = reinterpret_cast<const float4*>(h0 + row * D);
  float4* mp = reinterpret_cast<float4*>(m_prev + row * D);
  const float4* sh = reinterpret_cast<const float4*>(shift);
  const float4* sc = reinterpret_cast<const float4*>(scale);
  const int n4 = D >> 2;
  float s = 0.f;
  for (int i = lane; i < n4; i += 32) { const float4 v = x[i]; s += (v.x + v.y) + (v.z + v.w); }
  const float mean = warp_sum(s) / (float)D;
  float q = 0.f;
  for (int i = lane; i < n4; i += 32) {
    const float4 v = x[i];
    const float a = v.x - mean, b = v.y - mean, c = v.z - mean, d = v.w - mean;
    q += (a * a + b * b) + (c * c + d * d);
  }
  const float rstd = rsqrtf(warp_sum(q) / (float)D + eps);
  float sd = 0.f, sp = 0.f;
  for (int i = lane; i < n4; i += 32) {
    const float4 v = x[i], a = sh[i], g = sc[i];
    float4 m;
    m.x = (v.x - mean) * rstd * (1.f + g.x) + a.x;
    m.y = (v.y - mean) * rstd * (1.f + g.y) + a.y;
    m.z = (v.z - mean) * rstd * (1.f + g.z) + a.z;
    m.w = (v.w - mean) * rstd * (1.f + g.w) + a.w;
    if (!first) {
      const float4 p = mp[i];
      sd += (fabsf(m.x - p.x) + fabsf(m.y - p.y)) + (fabsf(m.z - p.z) + fabsf(m.w - p.w));
      sp += (fabsf(p.x) + fabsf(p.y)) + (fabsf(p.z) + fabsf(p.w));
    }
    mp[i] = m;
  }
  sd = warp_sum(sd);
  sp = warp_sum(sp);
  if (lane == 0) row_part[row] = make_float2(sd, sp);
}

// One block, thread b = sequence b: rel_b in fp64 from the row partials (fixed order), the accumulate / compare /
// reset rule, then thread 0 builds the compact list of computing sequences in index order.
//   force != 0 (first and last step): every sequence computes and acc <- 0.
//   outputs: active_idx[0 .. n_active), pos[b] (position in the compact batch or -1), n_active[0],
//            computed[b] (0/1), rel[b] (NaN-free: 0 on the first step), acc[b] updated.
__global__ void __launch_bounds__(1024) tc_decide_kernel(const float2* __restrict__ row_part, int B, int rows_per_seq,
                                                         int first, int force, double threshold, int n_coeffs,
                                                         const double* __restrict__ coeffs, double* __restrict__ acc,
                                                         int* __restrict__ active_idx, int* __restrict__ pos,
                                                         int* __restrict__ n_active, int* __restrict__ computed,
                                                         float* __restrict__ rel_out) {
  __shared__ int flag[1024];
  const int b = threadIdx.x;
  if (b < B) {
    double rel = 0.0;
    if (!first) {
      double sd = 0.0, sp = 0.0;
      const float2* p = row_part + (long long)b * rows_per_seq;
      for (int r = 0; r < rows_per_seq; ++r) { sd += (double)p[r].x; sp += (double)p[r].y; }
      rel = sd / sp;
    }
    int compute;
    if (force) {
      compute = 1;
      acc[b] = 0.0;
    } else {
      double pv = 0.0, rp = 1.0;
      for (int j = 0; j < n_coeffs; ++j) { pv += coeffs[j] * rp; rp *= rel; }
      const double a = acc[b] + pv;
      compute = !(a < threshold);
      acc[b] = compute ? 0.0 : a;
    }
    flag[b] = compute;
    computed[b] = compute;
    rel_out[b] = (float)rel;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int n = 0;
    for (int i = 0; i < B; ++i) {
      if (flag[i]) { active_idx[n] = i; pos[i] = n; ++n; }
      else pos[i] = -1;
    }
    n_active[0] = n;
  }
}

// dst[j, :] = src[idx[j] / div, :] for j < n (div = 1: gather sequences; div = K: text rows of the sequence's prompt)
__global__ void __launch_bounds__(256) tc_gather_kernel(const float4* __restrict__ src, float4* __restrict__ dst,
                                                        const int* __restrict__ idx, int div, long long n4_per_seq,
                                                        long long total4) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total4) return;
  const long long j = i / n4_per_seq, e = i - j * n4_per_seq;
  dst[i] = src[(long long)(idx[j] / div) * n4_per_seq + e];
}

// For every sequence b: computing (pos[b] = j >= 0): R_b <- hc_j - h0_b ; h0_b <- hc_j      (cache the residual)
//                       skipping  (pos[b] < 0):       h0_b <- h0_b + R_b                    (reuse it)
__global__ void __launch_bounds__(256) tc_combine_kernel(float4* __restrict__ h0, float4* __restrict__ resid,
                                                         const float4* __restrict__ hc, const int* __restrict__ pos,
                                                         long long n4_per_seq, long long total4) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total4) return;
  const long long b = i / n4_per_seq, e = i - b * n4_per_seq;
  const int j = pos[b];
  float4 x = h0[i];
  if (j >= 0) {
    const float4 y = hc[(long long)j * n4_per_seq + e];
    resid[i] = make_float4(y.x - x.x, y.y - x.y, y.z - x.z, y.w - x.w);
    h0[i] = y;
  } else {
    const float4 r = resid[i];
    h0[i] = make_float4(x.x + r.x, x.y + r.y, x.z + r.z, x.w + r.w);
  }
}

}  // namespace

cudaError_t launch_tc_metric(const float* h0, float* m_prev, const float* shift, const float* scale, long long rows, int D,
                             float eps, bool first, float* row_part, cudaStream_t st) {
  if (rows <= 0) return cudaSuccess;
  if (D % 4) return cudaErrorInvalidValue;
  const long long blocks = (rows + 7) / 8;
  tc_metric_kernel<<<(unsigned)blocks, 256, 0, st>>>(h0, m_prev, shift, scale, rows, D, eps, first ? 1 : 0,
                                                     reinterpret_cast<float2*>(row_part));
  return cudaGetLastError();
}

cudaError_t launch_tc_decide(const float* row_part, int B, int rows_per_seq, bool first, bool force, double threshold,
                             int n_coeffs, const double* d_coeffs, double* acc, int* active_idx, int* pos, int* n_active,
                             int* computed, float* rel, cudaStream_t st) {
  if (B <= 0 || B > 1024) return cudaErrorInvalidValue;
  tc_decide_kernel<<<1, 1024, 0, st>>>(reinterpret_cast<const float2*>(row_part), B, rows_per_seq, first ? 1 : 0, force ? 1 : 0,
                                       threshold, n_coeffs, d_coeffs, acc, active_idx, pos, n_active, computed, rel);
  return cudaGetLastError();
}

cudaError_t launch_tc_gather(const float* src, float* dst, const int* idx, int div, int n, long long n_per_seq,
                             cudaStream_t st) {
  if (n <= 0 || n_per_seq <= 0) return cudaSuccess;
  if (n_per_seq % 4 || div <= 0) return cudaErrorInvalidValue;
  const long long n4 = n_per_seq / 4, total4 = n4 * n;
  tc_gather_kernel<<<(unsigned)((total4 + 255) / 256), 256, 0, st>>>(reinterpret_cast<const float4*>(src),
                                                                     reinterpret_cast<float4*>(dst), idx, div, n4, total4);
  return cudaGetLastError();
}

cudaError_t launch_tc_combine(float* h0, float* resid, const float* hc, const int* pos, int B, long long n_per_seq,
                              cudaStream_t st) {
  if (B <= 0 || n_per_seq <= 0) return cudaSuccess;
  if (n_per_seq % 4) return cudaErrorInvalidValue;
  const long long n4 = n_per_seq / 4, total4 = n4 * B;
  tc_combine_kernel<<<(unsigned)((total4 + 255) / 256), 256, 0, st>>>(reinterpret_cast<float4*>(h0),
                                                                      reinterpret_cast<float4*>(resid),
                                                                      reinterpret_cast<const float4*>(hc), pos, n4, total4);
  return cudaGetLastError();
}
