// nvfp4_math.cuh - the arithmetic that decides NVFP4 codes, shared by the quantiser (nvfp4.cu) and the fused GEMM epilogue
// (gemm_nvfp4.cu).  DESIGN.md section 13b, reading N3: sf_b = e4m3(max_b |x| / 6), q_k = e2m1(x_k / sf_b), every value that
// decides a code formed in fp32 with IEEE (round-to-nearest) division, as oracle/nvfp4.py forms it.
#pragma once
#include <cuda_fp8.h>
#include <stdint.h>

namespace nvfp4 {

// nearest E4M3 value (RNE, saturating) of v as fp32, and its byte
__device__ __forceinline__ float e4m3_round(float v, uint32_t* code) {
  const __nv_fp8_storage_t c = __nv_cvt_float_to_fp8(v, __NV_SATFINITE, __NV_E4M3);
  *code = (uint32_t)c;
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

// x / sf for a divisor that is an E4M3 value, correctly rounded, without the 16 branchy div.rn.f32 sequences per block:
// every positive E4M3 value is (1 + k/8) * 2^e, so with y = RN(1 / sf) (one IEEE reciprocal per block) the Markstein step
//     q = RN(x * y);  r = x - sf * q (exact in one FMA);  q' = RN(q + r * y)
// returns RN(x / sf).  For the eight significands this is checked EXHAUSTIVELY over all 2^23 significands of x against the
// host's IEEE division (tests/test_nvfp4_division.py); powers of two scale both sides exactly.  Where the quotient
// underflows both sides give a value far below E2M1's first rounding boundary (0.25), i.e. code 0.
struct BlockDivisor {
  float sf, y;
  __device__ __forceinline__ explicit BlockDivisor(float sf_) {
    sf = sf_;
    y = sf_ > 0.f ? __frcp_rn(sf_) : 0.f;                          // sf = 0: every quotient is 0
  }
  __device__ __forceinline__ BlockDivisor(float sf_, float y_) {
    sf = sf_;
    y = y_;
  }
  __device__ __forceinline__ float operator()(float x) const {
    const float q = __fmul_rn(x, y);
    return fmaf(fmaf(-sf, q, x), y, q);
  }
};

// one block of 16 values -> its E4M3 scale byte and two words of E2M1 codes
__device__ __forceinline__ void quantize_block16(const float* x, uint32_t* sf_code, uint32_t* lo, uint32_t* hi) {
  float amax = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) amax = fmaxf(amax, fabsf(x[i]));
  const BlockDivisor six(6.f, 0x1.555556p-3f);   // RN(1 / 6);                                 // amax / 6: the same step with sf = 1.5 * 4
  const BlockDivisor div(e4m3_round(six(amax), sf_code));
  float q[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) q[i] = div(x[i]);
  *lo = e2m1x8(q);
  *hi = e2m1x8(q + 8);
}

}  // namespace nvfp4
