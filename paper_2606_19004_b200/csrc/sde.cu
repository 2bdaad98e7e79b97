// sde.cu - stochastic sampler step with per-step log-probability ("The algorithm backbone is FlowGRPO",
// Table 2 "SDE window", readings D1-D4):
//     x <- cx * x + cv * v + cn * xi ,  xi ~ N(0, I) from Philox stream 256 + step of the sequence's seed,
//     log p = -mean(xi^2) / 2 - log(cn) - log(2 pi) / 2
// with cx = 1 + sigma^2/(2 t) dt, cv = (1 + sigma^2 (1 - t)/(2 t)) dt, cn = sigma sqrt(-dt) computed by the caller.
// One kernel: the noise is generated in registers (the Philox block of element e/4 is exactly the float4 the thread
// updates), so the step moves the same 12 B/element as the deterministic Euler update (K6) - HBM-bound - and the
// reductions (sum xi^2, and <probe, x> on the last step) use K6's fixed-order partial sums: deterministic,
// batch-independent.
#include <math.h>

#include "kernels.h"
#include "philox.cuh"

namespace {

__global__ void __launch_bounds__(256) sde_update_kernel(float* __restrict__ x, const float* __restrict__ v,
                                                         const uint64_t* __restrict__ seeds, uint32_t stream_id, float cx,
                                                         float cv, float cn, long long E, const float* __restrict__ probe,
                                                         float* __restrict__ lp_partials, float* __restrict__ rw_partials,
                                                         int n_chunks) {
  const int b = blockIdx.y, chunk = blockIdx.x;
  const long long base = (long long)b * E;
  const uint64_t seed = seeds[b];
  const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
  float acc2 = 0.f, accr = 0.f;
#pragma unroll
  for (int i = 0; i < REWARD_CHUNK / (256 * 4); ++i) {
    const long long e = (long long)chunk * REWARD_CHUNK + (i * 256 + threadIdx.x) * 4;
    if (e < E) {
      const unsigned long long j = (unsigned long long)(e >> 2);
      const uint4 w = philox4x32_10(make_uint4((uint32_t)j, (uint32_t)(j >> 32), stream_id, 0u), key);
      const float2 za = box_muller(w.x, w.y), zb = box_muller(w.z, w.w);
      float4 xv = *reinterpret_cast<float4*>(x + base + e);
      const float4 vv = *reinterpret_cast<const float4*>(v + base + e);
      xv.x = fmaf(cn, za.x, fmaf(cv, vv.x, cx * xv.x));
      xv.y = fmaf(cn, za.y, fmaf(cv, vv.y, cx * xv.y));
      xv.z = fmaf(cn, zb.x, fmaf(cv, vv.z, cx * xv.z));
      xv.w = fmaf(cn, zb.y, fmaf(cv, vv.w, cx * xv.w));
      *reinterpret_cast<float4*>(x + base + e) = xv;
      acc2 += (za.x * za.x + za.y * za.y) + (zb.x * zb.x + zb.y * zb.y);
      if (probe) {
        const float4 p = *reinterpret_cast<const float4*>(probe + e);
        accr += (p.x * xv.x + p.y * xv.y) + (p.z * xv.z + p.w * xv.w);
      }
    }
  }
  __shared__ float ws2[8], wsr[8];
  acc2 = warp_sum(acc2);
  accr = warp_sum(accr);
  if ((threadIdx.x & 31) == 0) { ws2[threadIdx.x >> 5] = acc2; wsr[threadIdx.x >> 5] = accr; }
  __syncthreads();
  if (threadIdx.x == 0) {
    float s2 = 0.f, sr = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { s2 += ws2[i]; sr += wsr[i]; }
    lp_partials[(long long)b * n_chunks + chunk] = s2;
    if (probe) rw_partials[(long long)b * n_chunks + chunk] = sr;
  }
}

// logp[b * stride] = -(sum xi^2) / (2 E) - log(cn) - log(2 pi)/2, partials summed in index order in fp64
__global__ void sde_logp_finalize_kernel(const float* __restrict__ partials, int B, int n_chunks, double inv_2e,
                                         double log_term, float* __restrict__ logp, long long stride) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  double s = 0.0;
  for (int i = 0; i < n_chunks; ++i) s += (double)partials[(long long)b * n_chunks + i];
  logp[(long long)b * stride] = (float)(-s * inv_2e - log_term);
}

}  // namespace

cudaError_t launch_sde_update(float* x, const float* v, const uint64_t* seeds, uint32_t stream_id, double cx, double cv,
                              double cn, int B, long long E, const float* probe, float* lp_partials, float* rw_partials,
                              float* logp, long long logp_stride, cudaStream_t st) {
  if (B <= 0 || E <= 0) return cudaSuccess;
  if (E % 4 || !(cn > 0.0)) return cudaErrorInvalidValue;
  const int nc = (int)((E + REWARD_CHUNK - 1) / REWARD_CHUNK);
  sde_update_kernel<<<dim3(nc, B), 256, 0, st>>>(x, v, seeds, stream_id, (float)cx, (float)cv, (float)cn, E, probe,
                                                 lp_partials, rw_partials, nc);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double cnf = (double)(float)cn;                       // the coefficient the kernel actually used
  sde_logp_finalize_kernel<<<(B + 127) / 128, 128, 0, st>>>(lp_partials, B, nc, 0.5 / (double)E,
                                                            log(cnf) + 0.9189385332046727, logp, logp_stride);
  return cudaGetLastError();
}
