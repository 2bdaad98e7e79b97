// fp8.cu - quantisation kernels of the low-precision (FP8 E4M3) exploration variant ("a cheap exploratory
// rollout e.g., with reduced denoising steps or a quantized model", readings Q1-Q4):
//   weights      per output channel n: s_n = max_k |W_nk| / 448 (1 for a zero row), Wq_nk = e4m3(W_nk / s_n)   (once)
//   activations  unit scale: xq = e4m3(x), round-to-nearest-even, saturating at +-448
// Both are HBM-bound streaming kernels; the weight pass runs once per weight set (20.4 G parameters at config 3).
#include <cuda_fp8.h>

#include "kernels.h"

namespace {

__device__ __forceinline__ uint32_t pack4_e4m3(float a, float b, float c, float d) {
  const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3);
  const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(c, d), __NV_SATFINITE, __NV_E4M3);
  return lo | (hi << 16);
}

// one block per row of W [N, K] (K % 8 == 0): row maximum (fixed-order tree), then the scaled conversion
__global__ void __launch_bounds__(256) quantize_weight_rows_kernel(const bf16* __restrict__ w, int K, uint8_t* __restrict__ wq,
                                                                  float* __restrict__ scale) {
  const long long row = blockIdx.x;
  const uint4* src = reinterpret_cast<const uint4*>(w + row * K);
  const int n8 = K >> 3;
  float m = 0.f;
  for (int i = threadIdx.x; i < n8; i += 256) {
    const uint4 raw = src[i];
    const bf16* e = reinterpret_cast<const bf16*>(&raw);
#pragma unroll
    for (int j = 0; j < 8; ++j) m = fmaxf(m, fabsf(__bfloat162float(e[j])));
  }
  __shared__ float red[8];
  m = warp_max(m);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  float amax = red[0];
#pragma unroll
  for (int i = 1; i < 8; ++i) amax = fmaxf(amax, red[i]);
  const float s = amax > 0.f ? amax / 448.f : 1.f;
  if (threadIdx.x == 0) scale[row] = s;
  uint2* dst = reinterpret_cast<uint2*>(wq + row * K);
  for (int i = threadIdx.x; i < n8; i += 256) {
    const uint4 raw = src[i];
    const bf16* e = reinterpret_cast<const bf16*>(&raw);
    float v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __bfloat162float(e[j]) / s;       // IEEE division: the oracle divides too
    dst[i] = make_uint2(pack4_e4m3(v[0], v[1], v[2], v[3]), pack4_e4m3(v[4], v[5], v[6], v[7]));
  }
}

template <typename T>
__global__ void __launch_bounds__(256) quantize_e4m3_kernel(const T* __restrict__ in, uint8_t* __restrict__ out, long long n) {
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (i >= n) return;
  float v[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) v[j] = i + j < n ? to_f32(in[i + j]) : 0.f;
  if (i + 3 < n) {
    *reinterpret_cast<uint32_t*>(out + i) = pack4_e4m3(v[0], v[1], v[2], v[3]);
  } else {
    const uint32_t p = pack4_e4m3(v[0], v[1], v[2], v[3]);
    for (int j = 0; i + j < n; ++j) out[i + j] = (uint8_t)(p >> (8 * j));
  }
}

}  // namespace

cudaError_t launch_quantize_weight_rows(const void* w_bf16, long long N, int K, void* wq, float* scale, cudaStream_t st) {
  if (N <= 0) return cudaSuccess;
  if (K <= 0 || K % 8 || N > 0x7fffffffLL) return cudaErrorInvalidValue;
  quantize_weight_rows_kernel<<<(unsigned)N, 256, 0, st>>>((const bf16*)w_bf16, K, (uint8_t*)wq, scale);
  return cudaGetLastError();
}

cudaError_t launch_quantize_e4m3(spot_dtype dt, const void* in, long long n, void* out, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  const long long blocks = (n + 1023) / 1024;
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
  if (dt == SPOT_F32) quantize_e4m3_kernel<float><<<(unsigned)blocks, 256, 0, st>>>((const float*)in, (uint8_t*)out, n);
  else quantize_e4m3_kernel<bf16><<<(unsigned)blocks, 256, 0, st>>>((const bf16*)in, (uint8_t*)out, n);
  return cudaGetLastError();
}
