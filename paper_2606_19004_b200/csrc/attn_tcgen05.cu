// attn_tcgen05.cu - K5: flash-style joint text+image attention O = softmax(Q K^T / sqrt(d_h)) V over all S
// keys, no mask (north_star (d); S4 step 6, S6), bf16, d_h = 128.
//
// One CTA = TWO 128-row query tiles (A, B) of one (sequence, head), processed in ping-pong so that the
// softmax of one tile overlaps the tensor-core work of the other.  Keys are streamed in tiles of 128:
//   warp 0      TMA producer: Q_A, Q_B once, then K_j / V_j tiles (2-stage rings), all from ONE 3-D tensor map
//               over qkv [B, S, 3*H*d_h] (box 64 x 128 x 1, 128-byte swizzle; rows past S are zero-filled)
//   warp 1      TMEM allocator + MMA issuer (one thread):
//                 S_t = Q_t K_j^T   tcgen05.mma M128 N128 K16 x 8, both operands K-major in shared memory
//                 O_t += P_t V_j    A operand = P_t read from TENSOR MEMORY, B = V_j as MN-major shared memory
//               issue order per key tile: PV_A(j), S_A(j+1), PV_B(j), S_B(j+1)
//   warps 2-5   softmax warpgroup of tile A, warps 6-9 of tile B: thread = one query row; two tcgen05.ld passes over the 128
//               scores (row max, then exp), exp2 with the scale folded into one FFMA, row sum, P packed to bf16 and written
//               back with tcgen05.st over the columns S_t occupied (P never touches shared memory).
//               Online softmax with LAZY rescaling: the reference maximum is raised (and O_t in TMEM corrected)
//               only when a row's maximum grows by more than 2^8, decided per warp by a vote; the final O / l is
//               exact because P and l always use the same reference.
// TMEM columns: [0,128) S_A/P_A, [128,256) S_B/P_B, [256,384) O_A, [384,512) O_B.
// Tensor-pipe bound (+ MUFU ex2): 4 S^2 d_h FLOP per (sequence, head).
#include <string.h>

#include "kernels.h"
#include "tcgen05.cuh"

namespace {

constexpr int DH = 128, BQ = 128, BKV = 128, KV_STAGES = 2, QT = 2;
constexpr uint32_t SUB_BYTES = 128 * 64 * 2;          // one [128 x 64] bf16 sub-tile, 128-byte rows
constexpr uint32_t TILE_BYTES = 2 * SUB_BYTES;        // [128 x 128]
constexpr uint32_t OFF_Q = 0, OFF_K = QT * TILE_BYTES, OFF_V = OFF_K + KV_STAGES * TILE_BYTES,
                   OFF_BAR = OFF_V + KV_STAGES * TILE_BYTES;
constexpr uint32_t ATT_SMEM = OFF_BAR + 256 + 1024;
constexpr int ATT_THREADS = 64 + QT * 128;    // warps 0-1: TMA, MMA; warps 2-5 / 6-9: softmax warpgroups
constexpr float RESCALE_THRESHOLD = 8.0f;

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// D[tmem] (+)= A[tmem] * B[smem desc]
__device__ __forceinline__ void mma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                           uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
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
  auto s_full = [&](int t) { return bar + 8u * (9 + t); };
  auto p_full = [&](int t) { return bar + 8u * (11 + t); };
  auto pv_done = [&](int t) { return bar + 8u * (13 + t); };
  const uint32_t tmem_slot = bar + 8u * 15;
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(base_ptr + OFF_BAR + 8 * 15);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q0 = blockIdx.x * (QT * BQ), head = blockIdx.y, seq = blockIdx.z;
  const int n_kv = (S + BKV - 1) / BKV;
  const int col_q = head * DH, col_k = (H + head) * DH, col_v = (2 * H + head) * DH;

  if (warp == 0 && lane == 0) ptx::prefetch_tmap(&tm_qkv);
  if (warp == 1) {
    if (lane == 0) {
      ptx::mbar_init(q_full, 1);
      for (int s = 0; s < 2; ++s) {
        ptx::mbar_init(k_full(s), 1); ptx::mbar_init(k_empty(s), 1);
        ptx::mbar_init(v_full(s), 1); ptx::mbar_init(v_empty(s), 1);
        ptx::mbar_init(s_full(s), 1); ptx::mbar_init(p_full(s), 4); ptx::mbar_init(pv_done(s), 1);
      }
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

  if (warp == 0) {
    // ===================== TMA producer =====================
    // (elect.sync, not `lane == 0`: the compiler then issues UTMALDG / UTCHMMA straight from uniform registers instead
    //  of wrapping each one in a per-lane ELECT / BRA.U.ANY loop - see "single-thread issue paths" in tcgen05.cuh)
    if (ptx::elect_one()) {
      ptx::mbar_arrive_expect_tx(q_full, QT * TILE_BYTES);
#pragma unroll
      for (int t = 0; t < QT; ++t) {
        ptx::tma_load_3d(base + OFF_Q + t * TILE_BYTES, &tm_qkv, q_full, col_q, q0 + t * BQ, seq);
        ptx::tma_load_3d(base + OFF_Q + t * TILE_BYTES + SUB_BYTES, &tm_qkv, q_full, col_q + 64, q0 + t * BQ, seq);
      }
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
    if (ptx::elect_one()) {
      constexpr uint32_t idesc_qk = ptx::make_idesc_bf16(BQ, BKV, 0, 0);   // A = Q (K-major smem), B = K (K-major smem)
      constexpr uint32_t idesc_pv = ptx::make_idesc_bf16(BQ, DH, 0, 1);    // A = P (TMEM), B = V (MN-major smem)
      auto issue_qk = [&](int t, int j) {
        const int st = j & 1;
        const uint32_t qa = base + OFF_Q + t * TILE_BYTES, ka = base + OFF_K + st * TILE_BYTES;
#pragma unroll
        for (int k = 0; k < DH / 16; ++k) {
          const uint32_t off = (k >> 2) * SUB_BYTES + (k & 3) * 32;
          ptx::mma_f16_ss(tmem_base + t * BKV, ptx::make_smem_desc(qa + off, 16, 1024),
                          ptx::make_smem_desc(ka + off, 16, 1024), idesc_qk, k ? 1u : 0u);
        }
        ptx::mma_commit(s_full(t));
        if (t == QT - 1) ptx::mma_commit(k_empty(st));
      };
      ptx::mbar_wait(q_full, 0);
      ptx::mbar_wait(k_full(0), 0);
      ptx::tc_fence_after();
      issue_qk(0, 0);
      issue_qk(1, 0);
      for (int j = 0; j < n_kv; ++j) {
        const int st = j & 1;
        ptx::mbar_wait(v_full(st), (uint32_t)(j >> 1) & 1u);
#pragma unroll
        for (int t = 0; t < QT; ++t) {
          ptx::mbar_wait(p_full(t), (uint32_t)j & 1u);
          ptx::tc_fence_after();
          const uint32_t va = base + OFF_V + st * TILE_BYTES;
#pragma unroll
          for (int k = 0; k < BKV / 16; ++k)        // 16 keys = 8 packed TMEM columns of P, 2 x 1024-byte groups of V
            mma_f16_ts(tmem_base + 256 + t * DH, tmem_base + t * BKV + k * 8,
                       ptx::make_smem_desc(va + k * 2048, SUB_BYTES, 1024), idesc_pv, (j | k) ? 1u : 0u);
          ptx::mma_commit(pv_done(t));
          if (t == QT - 1) ptx::mma_commit(v_empty(st));
          if (j + 1 < n_kv) {
            if (t == 0) { ptx::mbar_wait(k_full((j + 1) & 1), (uint32_t)((j + 1) >> 1) & 1u); ptx::tc_fence_after(); }
            issue_qk(t, j + 1);
          }
        }
      }
    }
  } else {
    // ===================== softmax / correction / epilogue: 2 warpgroups x 128 rows =====================
    const int t = (warp - 2) >> 2;                      // query tile of this warpgroup
    const int quarter = warp & 3;                       // TMEM lane quarter this warp may access
    const int row = quarter * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const uint32_t tmem_s = tmem_base + t * BKV + lane_addr, tmem_o = tmem_base + 256 + t * DH + lane_addr;
    float m_ref = -INFINITY, l = 0.f;
    for (int j = 0; j < n_kv; ++j) {
      ptx::mbar_wait(s_full(t), (uint32_t)j & 1u);     // also implies PV_t(j-1) has completed (in-order pipe)
      ptx::tc_fence_after();
      const int valid = S - j * BKV;                   // keys of this tile that exist (>= 128 except the last)
      // pass 1 over TMEM: row maximum (two passes keep the live registers at 64 scores instead of 128)
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t sv[32];
        ptx::tmem_ld_32x32(tmem_s + c * 32, sv);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 32; ++i)
          if (valid >= BKV || c * 32 + i < valid) mx = fmaxf(mx, __uint_as_float(sv[i]));
      }
      const bool need = (mx - m_ref) * scale_log2 > RESCALE_THRESHOLD;     // true on the first tile (m_ref = -inf)
      if (__any_sync(0xffffffffu, need)) {
        const float m_new = fmaxf(m_ref, mx);
        if (j > 0) {
          const float alpha = ex2_approx((m_ref - m_new) * scale_log2);
          l *= alpha;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t ov[32];
            ptx::tmem_ld_32x32(tmem_o + c * 32, ov);
            ptx::tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) ov[i] = __float_as_uint(__uint_as_float(ov[i]) * alpha);
            ptx::tmem_st_32x32(tmem_o + c * 32, ov);
          }
        }
        m_ref = m_new;
      }
      const float mc = m_ref * scale_log2;
      float sum = 0.f;
      // pass 2: 64 keys at a time -> exp2 -> 32 packed bf16x2 columns written over the consumed score columns
#pragma unroll
      for (int hlf = 0; hlf < 2; ++hlf) {
        uint32_t sv[2][32];
        ptx::tmem_ld_32x32(tmem_s + hlf * 64, sv[0]);
        ptx::tmem_ld_32x32(tmem_s + hlf * 64 + 32, sv[1]);
        ptx::tmem_ld_wait();
        uint32_t pk[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const int c = i >> 4, e = (i & 15) * 2, key = hlf * 64 + 2 * i;
          float p0 = ex2_approx(fmaf(__uint_as_float(sv[c][e]), scale_log2, -mc));
          float p1 = ex2_approx(fmaf(__uint_as_float(sv[c][e + 1]), scale_log2, -mc));
          if (valid < BKV) { if (key >= valid) p0 = 0.f; if (key + 1 >= valid) p1 = 0.f; }
          sum += p0 + p1;
          pk[i] = pack_bf16(p0, p1);
        }
        ptx::tmem_st_32x32(tmem_s + hlf * 32, pk);
      }
      l += sum;
      ptx::tmem_st_wait();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full(t));
    }
    // epilogue: O / l -> bf16
    ptx::mbar_wait(pv_done(t), (uint32_t)(n_kv - 1) & 1u);
    ptx::tc_fence_after();
    const float inv = 1.f / l;
    const int qrow = q0 + t * BQ + row;
    const bool row_ok = qrow < S;
    bf16* orow = out + ((long long)seq * S + qrow) * (long long)(H * DH) + head * DH;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      uint32_t ov[32];
      ptx::tmem_ld_32x32(tmem_o + c * 32, ov);
      ptx::tmem_ld_wait();
      if (row_ok) {
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          uint4 pk;
          pk.x = pack_bf16(__uint_as_float(ov[g * 8]) * inv, __uint_as_float(ov[g * 8 + 1]) * inv);
          pk.y = pack_bf16(__uint_as_float(ov[g * 8 + 2]) * inv, __uint_as_float(ov[g * 8 + 3]) * inv);
          pk.z = pack_bf16(__uint_as_float(ov[g * 8 + 4]) * inv, __uint_as_float(ov[g * 8 + 5]) * inv);
          pk.w = pack_bf16(__uint_as_float(ov[g * 8 + 6]) * inv, __uint_as_float(ov[g * 8 + 7]) * inv);
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
  dim3 grid((S + QT * BQ - 1) / (QT * BQ), H, B);
  const float scale_log2 = 1.4426950408889634f / sqrtf((float)DH);
  attn_tcgen05_kernel<<<grid, ATT_THREADS, ATT_SMEM, st>>>(tm, (bf16*)out, S, H, scale_log2);
  return cudaGetLastError();
}
