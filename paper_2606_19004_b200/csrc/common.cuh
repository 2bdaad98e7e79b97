// common.cuh - shared device/host helpers of libspot (CUDA path only; shares nothing with oracle/).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/spot.h"

typedef __nv_bfloat16 bf16;

// Row addressing for activations that live in "per-sequence" buffers: logical row m of a
// [M, ld] matrix sits at element offset (m / rows_per_seq) * seq_stride + offset + (m % rows_per_seq) * ld.
// A plain row-major matrix is {rows_per_seq = M, seq_stride = 0, offset = 0, ld}.
struct RowMap {
  int rows_per_seq;
  long long seq_stride;
  long long offset;
  long long ld;
  __host__ __device__ __forceinline__ long long row(int m) const {
    int b = m / rows_per_seq;
    return (long long)b * seq_stride + offset + (long long)(m - b * rows_per_seq) * ld;
  }
};
static inline RowMap plain_rows(int M, long long ld) { RowMap r{M > 0 ? M : 1, 0, 0, ld}; return r; }

// EPI_QKV_ROPE: the QKV projection with K4 fused: +bias, then per-head RMSNorm * gain and the rotary
// rotation on the q and k heads (v heads: +bias only), bf16 out (tcgen05 v3 kernel only, head_dim 128)
enum Epilogue { EPI_BIAS = 0, EPI_BIAS_GELU = 1, EPI_GATE_RES = 2, EPI_QKV_ROPE = 3 };

// One GEMM problem C = epi(A W^T + bias); A rows addressed through a_map (K contiguous), W [N, K].
struct GemmProblem {
  const void* A;
  RowMap a_map;
  const void* W;
  const void* bias;     // [N], element type of W
  int M, N, K;
  void* out;            // EPI_BIAS / EPI_BIAS_GELU: output matrix (type TOUT)
  RowMap out_map;
  const float* gate;    // EPI_GATE_RES: [N] fp32
  float* resid;         // EPI_GATE_RES: fp32 residual stream, updated in place
  RowMap resid_map;
  // EPI_QKV_ROPE only: N = 3 * hidden, columns [q | k | v], heads of 128; row r of a sequence sits at joint
  // position pos_off + r of the rotary table cos_t / sin_t [S, 64] fp32; gains [128] in the element type of W
  const void* q_gain;
  const void* k_gain;
  const float* cos_t;
  const float* sin_t;
  int pos_off;
  float rms_eps;
  // FP8 variant (tcgen05 v3 kernel only): A and W hold E4M3 bytes (a_map in elements = bytes),
  // w_scale [N] fp32 = per-output-channel dequantisation scale applied to the accumulator before the bias;
  // EPI_BIAS / EPI_BIAS_GELU then write E4M3 (out_map in bytes), EPI_QKV_ROPE bf16, EPI_GATE_RES the fp32 residual
  int fp8;
  const float* w_scale;
};

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f32<bf16>(float v) { return __float2bfloat16_rn(v); }

__device__ __forceinline__ float gelu_tanh_f(float x) {
  const float k0 = 0.7978845608028654f;   // sqrt(2/pi)
  float inner = k0 * (x + 0.044715f * x * x * x);
  return 0.5f * x * (1.0f + tanhf(inner));
}
__device__ __forceinline__ float silu_f(float x) { return x / (1.0f + expf(-x)); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

#define SPOT_CUDA_TRY(expr)                         \
  do {                                              \
    cudaError_t _e = (expr);                        \
    if (_e != cudaSuccess) return _e;               \
  } while (0)
