// nvfp4.cu - quantisers of the NVFP4 exploration variant (readings N2-N4; "a cheap
// exploratory rollout ... with a quantized model").  NVFP4 = E2M1 values in blocks of 16 consecutive elements along K,
// one E4M3 scale factor per block; weights carry a second-level fp32 scale per output channel.
//
// Output layout = what the block-scaled tensor-core GEMM (gemm_nvfp4.cu) consumes without further shuffling:
//   codes   [rows, K / 2] bytes, element k in the low (k even) / high (k odd) nibble - K-major, TMA-loadable;
//   scales  in "atoms" of 512 bytes = the scale factors of 128 rows x 64 elements of K (one K = 64 MMA step):
//           byte (r % 32) * 16 + ((r % 128) / 32) * 4 + (b % 4) of atom (r / 128) * (K / 64) + b / 4 holds the scale
//           of row r, block b - 32 rows x 16 bytes, exactly the shape tcgen05.cp 32x128b.warpx4 moves to tensor memory.
// Every value that decides a code is formed in fp32 with IEEE division, as oracle/nvfp4.py does (a 4-bit code is an
// integer decided by floating point; both sides take the decision in the same precision).
#include <cuda_fp8.h>

#include "kernels.h"

namespace {

__device__ __forceinline__ float e4m3_round(float v, uint8_t* code) {      // nearest E4M3 (RNE, saturating) as fp32 + its byte
  const __nv_fp8_storage_t c = __nv_cvt_float_to_fp8(v, __NV_SATFINITE, __NV_E4M3);
  *code = (uint8_t)c;
  return __half2float(__half(__nv_cvt_fp8_to_halfraw(c, __NV_E4M3)));
}

// eight fp32 -> eight E2M1 codes in one 32-bit word, element i in nibble i (RNE, ties to the even code, saturating)
__device__ __forceinline__ uint32_t e2m1x8(const float* v) {
  uint32_t r;
  asm("{\n\t.reg .b8 b0, b1, b2, b3;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b0, %2, %1;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b1, %4, %3;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b2, %6, %5;\n\t"
      "cvt.rn.satfinite.e2m1x2.f32 b3, %8, %7;\n\t"
      "mov.b32 %0, {b0, b1, b2, b3};\n\t}\n"
      : "=r"(r)
      : "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]));
  return r;
}

__device__ __forceinline__ void load16(const bf16* p, float* x) {
  const uint4 a = __ldg(reinterpret_cast<const uint4*>(p)), b = __ldg(reinterpret_cast<const uint4*>(p) + 1);
  const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    x[2 * i] = __uint_as_float(w[i] << 16);
    x[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
}

// One thread = one row x 64 elements of K (4 blocks): 128 bytes in, 32 bytes of codes + 4 scale bytes out.
// row_scale != nullptr: the row is divided by row_scale[r] first (weights, reading N4).
__global__ void __launch_bounds__(256)
nvfp4_quantize_kernel(const bf16* __restrict__ src, RowMap map, int rows, int K, const float* __restrict__ row_scale,
                      uint8_t* __restrict__ codes, uint8_t* __restrict__ sf) {
  const int groups = K >> 6;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)rows * groups) return;
  const int r = (int)(idx / groups), g = (int)(idx - (long long)r * groups);
  const bf16* p = src + map.row(r) + (long long)g * 64;
  const float rs = row_scale ? row_scale[r] : 1.f;
  uint32_t packed[8];
  uint8_t sfb[4];
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    float x[16];
    load16(p + b * 16, x);
    float amax = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      if (row_scale) x[i] = __fdiv_rn(x[i], rs);
      amax = fmaxf(amax, fabsf(x[i]));
    }
    const float s = e4m3_round(__fdiv_rn(amax, 6.f), &sfb[b]);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = s > 0.f ? __fdiv_rn(x[i], s) : 0.f;
    packed[2 * b] = e2m1x8(x);
    packed[2 * b + 1] = e2m1x8(x + 8);
  }
  uint4* cp = reinterpret_cast<uint4*>(codes + (long long)r * (K >> 1) + g * 32);
  cp[0] = make_uint4(packed[0], packed[1], packed[2], packed[3]);
  cp[1] = make_uint4(packed[4], packed[5], packed[6], packed[7]);
  const long long atom = (long long)(r >> 7) * groups + g;
  *reinterpret_cast<uint32_t*>(sf + atom * 512 + (r & 31) * 16 + ((r & 127) >> 5) * 4) =
      (uint32_t)sfb[0] | ((uint32_t)sfb[1] << 8) | ((uint32_t)sfb[2] << 16) | ((uint32_t)sfb[3] << 24);
}

// s_n = max_k |W_nk| / (6 * 448), 1 for a zero row (reading N4); one warp per row
__global__ void __launch_bounds__(256)
nvfp4_row_scale_kernel(const bf16* __restrict__ w, int rows, int K, float* __restrict__ scale) {
  const int r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (r >= rows) return;
  float amax = 0.f;
  for (int k = lane * 8; k < K; k += 256) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(w + (long long)r * K + k));
    const uint32_t u[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i)
      amax = fmaxf(amax, fmaxf(fabsf(__uint_as_float(u[i] << 16)), fabsf(__uint_as_float(u[i] & 0xffff0000u))));
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  if (lane == 0) scale[r] = amax > 0.f ? __fdiv_rn(amax, 2688.f) : 1.f;
}

}  // namespace

size_t nvfp4_codes_bytes(long long rows, long long K) { return (size_t)(rows * (K / 2)); }
size_t nvfp4_sf_bytes(long long rows, long long K) { return (size_t)(((rows + 127) / 128) * (K / 64) * 512); }

cudaError_t launch_nvfp4_quantize(const void* src_bf16, RowMap map, int rows, int K, const float* row_scale, void* codes,
                                  void* sf, cudaStream_t st) {
  if (rows <= 0) return cudaSuccess;
  if (K % 64 || rows % 128) return cudaErrorInvalidValue;
  const long long n = (long long)rows * (K / 64);
  nvfp4_quantize_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(static_cast<const bf16*>(src_bf16), map, rows, K, row_scale,
                                                                   static_cast<uint8_t*>(codes), static_cast<uint8_t*>(sf));
  return cudaGetLastError();
}

cudaError_t launch_nvfp4_row_scale(const void* w_bf16, int rows, int K, float* scale, cudaStream_t st) {
  if (rows <= 0) return cudaSuccess;
  if (K % 8) return cudaErrorInvalidValue;
  nvfp4_row_scale_kernel<<<(rows + 7) / 8, 256, 0, st>>>(static_cast<const bf16*>(w_bf16), rows, K, scale);
  return cudaGetLastError();
}
