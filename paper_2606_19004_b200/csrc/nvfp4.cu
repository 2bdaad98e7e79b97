// nvfp4.cu - quantisers of the NVFP4 exploration variant (readings N2-N4; "a cheap
// exploratory rollout ... with a quantized model").  NVFP4 = E2M1 values in blocks of 16 consecutive elements along K,
// one E4M3 scale factor per block; weights carry a second-level fp32 scale per output channel.
//
// Output layout = what the block-scaled tensor-core GEMM (gemm_nvfp4.cu) consumes without further shuffling:
//   codes   [rows, K / 2] bytes, element k in the low (k even) / high (k odd) nibble - K-major, TMA-loadable;
//   scales  in "atoms" of 512 bytes = the scale factors of 128 rows x 64 elements of K (one K = 64 MMA step):
//           byte (r % 32) * 16 + ((r % 128) / 32) * 4 + (b % 4) of atom (r / 128) * (K / 64) + b / 4 holds the scale
//           of row r, block b - 32 rows x 16 bytes, exactly the shape tcgen05.cp 32x128b.warpx4 moves to tensor memory.
// Every value that decides a code is the correctly rounded fp32 quotient oracle/nvfp4.py forms (a 4-bit code is an integer
// decided by floating point; both sides take the decision in the same precision) - see nvfp4_math.cuh for how.
#include "kernels.h"
#include "nvfp4_math.cuh"

namespace {

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
  uint32_t packed[8], sfb[4];
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    float x[16];
    load16(p + b * 16, x);
    if (row_scale) {
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = __fdiv_rn(x[i], rs);
    }
    nvfp4::quantize_block16(x, &sfb[b], &packed[2 * b], &packed[2 * b + 1]);
  }
  uint4* cp = reinterpret_cast<uint4*>(codes + (long long)r * (K >> 1) + g * 32);
  cp[0] = make_uint4(packed[0], packed[1], packed[2], packed[3]);
  cp[1] = make_uint4(packed[4], packed[5], packed[6], packed[7]);
  const long long atom = (long long)(r >> 7) * groups + g;
  *reinterpret_cast<uint32_t*>(sf + atom * 512 + (r & 31) * 16 + ((r & 127) >> 5) * 4) =
      sfb[0] | (sfb[1] << 8) | (sfb[2] << 16) | (sfb[3] << 24);
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
