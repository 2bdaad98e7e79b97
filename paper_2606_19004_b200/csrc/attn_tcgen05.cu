// attn_tcgen05.cu - K5: flash-style joint text+image attention O = softmax(Q K^T / sqrt(d_h)) V over all S
// keys, no mask (north_star (d); S4 step 6, S6), bf16, d_h = 128.
//
// One CTA = one 128-row query tile of one (sequence, head); it streams the S keys in tiles of 128:
//   warp 0      TMA producer: Q once, then K_j / V_j tiles (2-stage rings), all from ONE 3-D tensor map over
//               qkv [B, S, 3*H*d_h] (box 64 x 128 x 1, 128-byte swizzle; rows past S are zero-filled)
//   warp 1      TMEM allocator + MMA issuer: S_j = Q K_j^T (tcgen05.mma M128 N128 K16 x 8, K-major operands)
//               into one of two TMEM score buffers, and O += P_j V_j (V as MN-major B operand) into a TMEM
//               accumulator; S_{j+1} is issued before P_j V_j so the tensor pipe works during softmax_j
//   warps 2-5   softmax: thread = one query row; tcgen05.ld of the 128 scores, row max, exp2 with the scale
//               folded into one FFMA, row sum, bf16 P written to shared memory in the swizzled K-major layout
//               the MMA reads.  Online softmax with LAZY rescaling: the running reference maximum is only
//               raised (and O in TMEM corrected by tcgen05.ld/st) when a row's maximum grows by more than 8
//               (log2 units), decided per warp with a vote; P stays <= 2^8, the final O / l is exact.
// Tensor-pipe bound (+ MUFU ex2): 4 S^2 d_h FLOP per (sequence, head).
#include <string.h>

#include "kernels.h"
#include "tcgen05.cuh"

namespace {

constexpr int DH = 128, BQ = 128, BKV = 128, KV_STAGES = 2;
constexpr uint32_t SUB_BYTES = 128 * 64 * 2;          // one [128 x 64] bf16 sub-tile, 128-byte rows
constexpr uint32_t TILE_BYTES = 2 * SUB_BYTES;        // [128 x 128]
constexpr uint32_t OFF_Q = 0, OFF_K = TILE_BYTES, OFF_V = OFF_K + KV_STAGES * TILE_BYTES,
                   OFF_P = OFF_V + KV_STAGES * TILE_BYTES, OFF_BAR = OFF_P + TILE_BYTES;
constexpr uint32_t ATT_SMEM = OFF_BAR + 256 + 1024;
constexpr int ATT_THREADS = 192;
constexpr float RESCALE_THRESHOLD = 8.0f;

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__global__ void __launch_bounds__(ATT_THREADS, 1)
attn_tcgen05_kernel(const __grid_constant__ CUtensorMap tm_qkv, bf16* __restrict__ out, int S, int H, float scale_log2) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw_addr = ptx::smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 1023u) & ~1023u;
  uint8_t* base_ptr = smem_raw + (base - raw_addr);
  const uint32_t bar = base + OFF_BAR;
  const uint32_t q_full = bar;
  auto k_full = [&](int s) { return bar + 8u * (1 + s); };
  auto k_empty = [&](int s) { return bar + 8u * (3 + s); };
  auto v_full = [&](int s) { return bar + 8u * (5 + s); };
  auto v_empty = [&](int s) { return bar + 8u * (7 + s); };
  auto s_full = [&](int s) { return bar + 8u * (9 + s); };
  auto s_empty = [&](int s) { return bar + 8u * (11 + s); };
  const uint32_t p_full = bar + 8u * 13, pv_done = bar + 8u * 14, tmem_slot = bar + 8u * 15;
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(base_ptr + OFF_BAR + 8 * 15);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q0 = blockIdx.x * BQ, head = blockIdx.y, seq = blockIdx.z;
  const int n_kv = (S + BKV - 1) / BKV;
  const int col_q = head * DH, col_k = (H + head) * DH, col_v = (2 * H + head) * DH;

  if (warp == 0 && lane == 0) ptx::prefetch_tmap(&tm_qkv);
  if (warp == 1) {
    if (lane == 0) {
      ptx::mbar_init(q_full, 1);
      for (int s = 0; s < 2; ++s) {
        ptx::mbar_init(k_full(s), 1); ptx::mbar_init(k_empty(s), 1);
        ptx::mbar_init(v_full(s), 1); ptx::mbar_init(v_empty(s), 1);
        ptx::mbar_init(s_full(s), 1); ptx::mbar_init(s_empty(s), 4);
      }
      ptx::mbar_init(p_full, 4); ptx::mbar_init(pv_done, 1);
      ptx::fence_barrier_init();
    }
    __syncwarp();
    ptx::tmem_alloc(tmem_slot, 512);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  const uint32_t tmem_s0 = tmem_base, tmem_o = tmem_base + 256;       // S buffers at columns 0 and 128

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      ptx::mbar_arrive_expect_tx(q_full, TILE_BYTES);
      ptx::tma_load_3d(base + OFF_Q, &tm_qkv, q_full, col_q, q0, seq);
      ptx::tma_load_3d(base + OFF_Q + SUB_BYTES, &tm_qkv, q_full, col_q + 64, q0, seq);
      for (int j = 0; j < n_kv; ++j) {
        const int st = j & 1;
        const uint32_t ph = (uint32_t)(j >> 1) & 1u;
        ptx::mbar_wait(k_empty(st), ph ^ 1);
        ptx::mbar_arrive_expect_tx(k_full(st), TILE_BYTES);
        ptx::tma_load_3d(base + OFF_K + st * TILE_BYTES, &tm_qkv, k_full(st), col_k, j * BKV, seq);
        ptx::tma_load_3d(base + OFF_K + st * TILE_BYTES + SUB_BYTES, &tm_qkv, k_full(st), col_k + 64, j * BKV, seq);
        ptx::mbar_wait(v_empty(st), ph ^ 1);
        ptx::mbar_arrive_expect_tx(v_full(st), TILE_BYTES);
        ptx::tma_load_3d(base + OFF_V + st * TILE_BYTES, &tm_qkv, v_full(st), col_v, j * BKV, seq);
        ptx::tma_load_3d(base + OFF_V + st * TILE_BYTES + SUB_BYTES, &tm_qkv, v_full(st), col_v + 64, j * BKV, seq);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc_qk = ptx::make_idesc_bf16(BQ, BKV, 0, 0);   // A = Q (K-major), B = K (K-major)
      constexpr uint32_t idesc_pv = ptx::make_idesc_bf16(BQ, DH, 0, 1);    // A = P (K-major), B = V (MN-major)
      auto issue_qk = [&](int j) {
        const int st = j & 1;
        ptx::mbar_wait(k_full(st), (uint32_t)(j >> 1) & 1u);
        ptx::mbar_wait(s_empty(st), ((uint32_t)(j >> 1) & 1u) ^ 1u);
        ptx::tc_fence_after();
        const uint32_t qa = base + OFF_Q, ka = base + OFF_K + st * TILE_BYTES;
#pragma unroll
        for (int k = 0; k < DH / 16; ++k) {
          const uint32_t off = (k >> 2) * SUB_BYTES + (k & 3) * 32;
          ptx::mma_f16_ss(tmem_s0 + st * BKV, ptx::make_smem_desc(qa + off, 16, 1024),
                          ptx::make_smem_desc(ka + off, 16, 1024), idesc_qk, k ? 1u : 0u);
        }
        ptx::mma_commit(k_empty(st));
        ptx::mma_commit(s_full(st));
      };
      ptx::mbar_wait(q_full, 0);
      issue_qk(0);
      for (int j = 0; j < n_kv; ++j) {
        if (j + 1 < n_kv) issue_qk(j + 1);
        const int st = j & 1;
        ptx::mbar_wait(v_full(st), (uint32_t)(j >> 1) & 1u);
        ptx::mbar_wait(p_full, (uint32_t)j & 1u);
        ptx::tc_fence_after();
        const uint32_t pa = base + OFF_P, va = base + OFF_V + st * TILE_BYTES;
#pragma unroll
        for (int k = 0; k < BKV / 16; ++k) {
          const uint64_t da = ptx::make_smem_desc(pa + (k >> 2) * SUB_BYTES + (k & 3) * 32, 16, 1024);
          const uint64_t db = ptx::make_smem_desc(va + k * 2048, SUB_BYTES, 1024);   // 16 keys = 2 x 1024-byte groups
          ptx::mma_f16_ss(tmem_o, da, db, idesc_pv, (j | k) ? 1u : 0u);
        }
        ptx::mma_commit(v_empty(st));
        ptx::mma_commit(pv_done);
      }
    }
  } else {
    // ===================== softmax / correction / epilogue (128 threads, one query row each) ===========
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    float m_ref = -INFINITY, l = 0.f;
    uint8_t* p_row = base_ptr + OFF_P + row * 128;
    for (int j = 0; j < n_kv; ++j) {
      const int st = j & 1;
      ptx::mbar_wait(s_full(st), (uint32_t)(j >> 1) & 1u);
      ptx::tc_fence_after();
      uint32_t sv[4][32];
#pragma unroll
      for (int c = 0; c < 4; ++c) ptx::tmem_ld_32x32(tmem_s0 + st * BKV + c * 32 + lane_addr, sv[c]);
      ptx::tmem_ld_wait();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(s_empty(st));
      const int valid = S - j * BKV;                       // keys of this tile that exist (>= 128 except the last)
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          float s = __uint_as_float(sv[c][i]);
          if (valid < BKV && c * 32 + i >= valid) { s = -INFINITY; sv[c][i] = __float_as_uint(s); }
          mx = fmaxf(mx, s);
        }
      // lazy rescale, decided per warp
      const bool need = (mx - m_ref) * scale_log2 > RESCALE_THRESHOLD;     // true on the first tile (m_ref = -inf)
      if (__any_sync(0xffffffffu, need)) {
        const float m_new = fmaxf(m_ref, mx);
        if (j > 0) {
          const float alpha = ex2_approx((m_ref - m_new) * scale_log2);
          l *= alpha;
          ptx::mbar_wait(pv_done, (uint32_t)(j - 1) & 1u);                 // O must be quiescent
          ptx::tc_fence_after();
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t ov[32];
            ptx::tmem_ld_32x32(tmem_o + c * 32 + lane_addr, ov);
            ptx::tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) ov[i] = __float_as_uint(__uint_as_float(ov[i]) * alpha);
            ptx::tmem_st_32x32(tmem_o + c * 32 + lane_addr, ov);
          }
          ptx::tmem_st_wait();
        }
        m_ref = m_new;
      }
      const float mc = m_ref * scale_log2;
      if (j > 0) ptx::mbar_wait(pv_done, (uint32_t)(j - 1) & 1u);          // P buffer free again
      float sum = 0.f;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
#pragma unroll
        for (int g = 0; g < 4; ++g) {                                      // 8 keys = one 16-byte chunk
          float p[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            p[i] = ex2_approx(fmaf(__uint_as_float(sv[c][g * 8 + i]), scale_log2, -mc));
            sum += p[i];
          }
          uint4 pk;
          __nv_bfloat162 b0 = __floats2bfloat162_rn(p[0], p[1]), b1 = __floats2bfloat162_rn(p[2], p[3]);
          __nv_bfloat162 b2 = __floats2bfloat162_rn(p[4], p[5]), b3 = __floats2bfloat162_rn(p[6], p[7]);
          pk.x = *reinterpret_cast<uint32_t*>(&b0); pk.y = *reinterpret_cast<uint32_t*>(&b1);
          pk.z = *reinterpret_cast<uint32_t*>(&b2); pk.w = *reinterpret_cast<uint32_t*>(&b3);
          const int key_chunk = c * 4 + g;                                  // 0..15 : keys key_chunk*8 ..
          const int sub = key_chunk >> 3, ch = key_chunk & 7;
          *reinterpret_cast<uint4*>(p_row + sub * SUB_BYTES + ((ch ^ (row & 7)) << 4)) = pk;
        }
      }
      l += sum;
      ptx::fence_proxy_async_smem();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full);
    }
    // epilogue: O / l -> bf16
    ptx::mbar_wait(pv_done, (uint32_t)(n_kv - 1) & 1u);
    ptx::tc_fence_after();
    const float inv = 1.f / l;
    const bool row_ok = q0 + row < S;
    bf16* orow = out + ((long long)seq * S + q0 + row) * (long long)(H * DH) + head * DH;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      uint32_t ov[32];
      ptx::tmem_ld_32x32(tmem_o + c * 32 + lane_addr, ov);
      ptx::tmem_ld_wait();
      if (row_ok) {
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          uint4 pk;
          __nv_bfloat162 b0 = __floats2bfloat162_rn(__uint_as_float(ov[g * 8]) * inv, __uint_as_float(ov[g * 8 + 1]) * inv);
          __nv_bfloat162 b1 = __floats2bfloat162_rn(__uint_as_float(ov[g * 8 + 2]) * inv, __uint_as_float(ov[g * 8 + 3]) * inv);
          __nv_bfloat162 b2 = __floats2bfloat162_rn(__uint_as_float(ov[g * 8 + 4]) * inv, __uint_as_float(ov[g * 8 + 5]) * inv);
          __nv_bfloat162 b3 = __floats2bfloat162_rn(__uint_as_float(ov[g * 8 + 6]) * inv, __uint_as_float(ov[g * 8 + 7]) * inv);
          pk.x = *reinterpret_cast<uint32_t*>(&b0); pk.y = *reinterpret_cast<uint32_t*>(&b1);
          pk.z = *reinterpret_cast<uint32_t*>(&b2); pk.w = *reinterpret_cast<uint32_t*>(&b3);
          *reinterpret_cast<uint4*>(orow + c * 32 + g * 8) = pk;
        }
      }
    }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem_base, 512); }
}

}  // namespace

bool tcgen05_attn_supported(int S, int H, int dh) {
  return dh == DH && S > 0 && H > 0 && spot_get_encode_tiled() != nullptr;
}

cudaError_t launch_attn_tcgen05(const void* qkv, void* out, int B, int S, int H, int dh, int num_sms, cudaStream_t st) {
  (void)num_sms;
  if (dh != DH) return cudaErrorInvalidValue;
  if (B <= 0) return cudaSuccess;
  CUtensorMap tm;
  memset(&tm, 0, sizeof(tm));
  const uint64_t dims[3] = {(uint64_t)3 * H * DH, (uint64_t)S, (uint64_t)B};
  const uint64_t strides[2] = {(uint64_t)3 * H * DH * 2, (uint64_t)S * 3 * H * DH * 2};
  const uint32_t box[3] = {64, 128, 1};
  SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm, qkv, 3, dims, strides, box));
  static bool attr_set = false;
  if (!attr_set) {
    SPOT_CUDA_TRY(cudaFuncSetAttribute(attn_tcgen05_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ATT_SMEM));
    attr_set = true;
  }
  dim3 grid((S + BQ - 1) / BQ, H, B);
  const float scale_log2 = 1.4426950408889634f / sqrtf((float)DH);
  attn_tcgen05_kernel<<<grid, ATT_THREADS, ATT_SMEM, st>>>(tm, (bf16*)out, S, H, scale_log2);
  return cudaGetLastError();
}
