// attn_tcgen05_v3.cu - K5, third version: flash-style joint text+image attention O = softmax(Q K^T / sqrt(d_h)) V over
// all S keys, no mask (north_star (d); S4 step 6, S6), bf16, d_h = 128.
//
// What changed against attn_tcgen05.cu (v2) and why (its ncu capture in round 1: tensor pipe 37 % active):
//   * v2 read every score tile from tensor memory TWICE (row max, then exp) and its S tile aliased P, so the chain
//     S -> softmax -> P -> PV -> next S of a query tile was serial.  TMEM reads are the scarce resource (the 128 x 128
//     fp32 S tile is 64 KB), so v3 streams keys in tiles of 64: a thread's 64 scores fit in registers (ONE pass), and
//     each query tile owns TWO 64-column S buffers, so Q K_{j+2}^T is issued right behind P_j V_j and the softmax
//     warps never wait for the tensor pipe in steady state.
//   * same warp roles: warp 0 TMA producer (Q once, then K_j / V_j through 4-stage rings, all from one 3-D tensor map
//     over qkv [B, S, 3*H*d_h], box 64 x 64), warp 1 TMEM allocator + single-thread MMA issuer, warps 2-5 / 6-9 the
//     softmax warpgroups of query tiles A / B (thread = one query row).
//   * S_t = Q_t K_j^T: tcgen05.mma M128 N64 K16 x 8 (both operands K-major shared memory); O_t += P_t V_j: M128 N128
//     K16 x 4 with P read from tensor memory (bf16, written over the consumed score columns) and V as MN-major B.
//   * online softmax with lazy rescaling as v2 (threshold 2^8, per-warp vote, O corrected in TMEM only then).
//   * PERSISTENT: one CTA per SM walks the list of work items (sequence, head, pair of query tiles).  A CTA's fixed
//     cost (launch, TMEM allocation, first loads, pipeline fill, O read-out) measured 8.2 us against 1.5-2.3 us per 128
//     keys, i.e. a quarter of the run time at S = 1280; now TMEM is allocated once, the producer runs ahead into the
//     next item's Q / K / V, the next item's first Q K^T overlap the read-out of O, and only the first P V of an item
//     waits for that read-out (o_free).
// TMEM columns: [0,64) S_A0, [64,128) S_A1, [128,192) S_B0, [192,256) S_B1, [256,384) O_A, [384,512) O_B.
// Tensor-pipe + MUFU bound: 4 S^2 d_h FLOP and S^2 ex2 per (sequence, head).
#include <cuda_fp8.h>
#include <string.h>

#include <stdlib.h>

#include "kernels.h"
#include "tcgen05.cuh"

namespace {

constexpr int DH = 128, BQ = 128, BKV = 64, KV_STAGES = 4, QT = 2;
constexpr uint32_t Q_SUB = 128 * 128;                  // [128 rows x 64 cols] bf16, 128-byte rows
constexpr uint32_t Q_TILE = 2 * Q_SUB;                 // [128 x 128]
constexpr uint32_t KV_SUB = 64 * 128;                  // [64 rows x 64 cols]
constexpr uint32_t KV_TILE = 2 * KV_SUB;               // [64 x 128]
constexpr uint32_t OFF_Q = 0, OFF_K = QT * Q_TILE, OFF_V = OFF_K + KV_STAGES * KV_TILE, OFF_BAR = OFF_V + KV_STAGES * KV_TILE;
// epilogue staging: one [32 rows x 128 bytes] buffer per softmax warp, 128-byte swizzled, handed to TMA stores
constexpr uint32_t OFF_STG = OFF_BAR + 1024, STG_BYTES = 32 * 128;
constexpr uint32_t ATT_SMEM = OFF_STG + QT * 4 * STG_BYTES + 1024;        // 226 KB of the 227 KB a CTA may have
constexpr int ATT_THREADS = 64 + QT * 128;
constexpr float RESCALE_THRESHOLD = 8.0f;

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// D[tmem] (+)= A[tmem] * B[smem desc]
__device__ __forceinline__ void mma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
}

// OUT8: O is stored as E4M3 bytes (unit scale, saturating) - the A operand of the FP8 out-projection.
template <bool OUT8>
__global__ void __launch_bounds__(ATT_THREADS, 1)
attn_tcgen05_v3_kernel(const __grid_constant__ CUtensorMap tm_qkv, const __grid_constant__ CUtensorMap tm_out, int S, int H,
                       int n_items, float scale_log2, int kv_policy) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw_addr = ptx::smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 1023u) & ~1023u;
  uint8_t* base_ptr = smem_raw + (base - raw_addr);
  const uint32_t bar = base + OFF_BAR;
  const uint32_t q_full = bar, q_empty = bar + 8u * 31;
  auto k_full = [&](int s) { return bar + 8u * (1 + s); };
  auto k_empty = [&](int s) { return bar + 8u * (5 + s); };
  auto v_full = [&](int s) { return bar + 8u * (9 + s); };
  auto v_empty = [&](int s) { return bar + 8u * (13 + s); };
  auto s_full = [&](int t, int b) { return bar + 8u * (17 + 2 * t + b); };
  auto p_full = [&](int t, int b) { return bar + 8u * (21 + 2 * t + b); };
  auto pv_done = [&](int t) { return bar + 8u * (25 + t); };
  auto o_final = [&](int t) { return bar + 8u * (27 + t); };      // all P V of query tile t of this item have completed
  auto o_free = [&](int t) { return bar + 8u * (29 + t); };       // the epilogue has read O_t: the next item may overwrite it
  const uint32_t tmem_slot = bar + 8u * 32;
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(base_ptr + OFF_BAR + 8 * 32);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_kv = (S + BKV - 1) / BKV;
  const int n_qt = (S + QT * BQ - 1) / (QT * BQ);           // work item = (sequence, head, pair of query tiles)

  if (warp == 0 && lane == 0) { ptx::prefetch_tmap(&tm_qkv); ptx::prefetch_tmap(&tm_out); }
  if (warp == 1) {
    if (lane == 0) {
      ptx::mbar_init(q_full, 1);
      ptx::mbar_init(q_empty, 1);
      for (int s = 0; s < KV_STAGES; ++s) {
        ptx::mbar_init(k_full(s), 1); ptx::mbar_init(k_empty(s), 1);
        ptx::mbar_init(v_full(s), 1); ptx::mbar_init(v_empty(s), 1);
      }
      for (int t = 0; t < QT; ++t) {
        for (int b = 0; b < 2; ++b) { ptx::mbar_init(s_full(t, b), 1); ptx::mbar_init(p_full(t, b), 4); }
        ptx::mbar_init(pv_done(t), 1);
        ptx::mbar_init(o_final(t), 1);
        ptx::mbar_init(o_free(t), 4);
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

  // Every role walks the same list of items (w = blockIdx.x, blockIdx.x + gridDim.x, ...) and counts key tiles with
  // one running index g = it * n_kv + j across items: ring stage g % 4, S/P buffer g & 1, barrier parities from g.
  if (warp == 0) {
    // ===================== TMA producer =====================
    // (elect.sync, not `lane == 0`: the compiler then issues UTMALDG / UTCHMMA straight from uniform registers instead
    //  of wrapping each one in a per-lane ELECT / BRA.U.ANY loop - see "single-thread issue paths" in tcgen05.cuh)
    if (ptx::elect_one()) {
      int it = 0;
      const uint64_t pol_kv = ptx::l2_policy(kv_policy);   // K / V tiles are re-read by the item's other query tiles
      for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++it) {
        const int x = w % n_qt, head = (w / n_qt) % H, seq = w / (n_qt * H);
        const int q0 = x * (QT * BQ);
        const int col_q = head * DH, col_k = (H + head) * DH, col_v = (2 * H + head) * DH;
        ptx::mbar_wait(q_empty, (uint32_t)(it & 1) ^ 1u);    // the last Q K^T of the previous item has read Q
        ptx::mbar_arrive_expect_tx(q_full, QT * Q_TILE);
#pragma unroll
        for (int t = 0; t < QT; ++t)
#pragma unroll
          for (int hf = 0; hf < 2; ++hf)                    // d_h halves (64 columns = 128 bytes)
#pragma unroll
            for (int rh = 0; rh < 2; ++rh)                  // row halves (box = 64 rows)
              ptx::tma_load_3d(base + OFF_Q + t * Q_TILE + hf * Q_SUB + rh * KV_SUB, &tm_qkv, q_full, col_q + hf * 64,
                               q0 + t * BQ + rh * 64, seq);
        for (int j = 0; j < n_kv; ++j) {
          const int g = it * n_kv + j, st = g % KV_STAGES;
          const uint32_t ph = (uint32_t)(g / KV_STAGES) & 1u;
          ptx::mbar_wait(k_empty(st), ph ^ 1);
          ptx::mbar_arrive_expect_tx(k_full(st), KV_TILE);
          ptx::tma_load_3d_hint(base + OFF_K + st * KV_TILE, &tm_qkv, k_full(st), col_k, j * BKV, seq, pol_kv);
          ptx::tma_load_3d_hint(base + OFF_K + st * KV_TILE + KV_SUB, &tm_qkv, k_full(st), col_k + 64, j * BKV, seq, pol_kv);
          ptx::mbar_wait(v_empty(st), ph ^ 1);
          ptx::mbar_arrive_expect_tx(v_full(st), KV_TILE);
          ptx::tma_load_3d_hint(base + OFF_V + st * KV_TILE, &tm_qkv, v_full(st), col_v, j * BKV, seq, pol_kv);
          ptx::tma_load_3d_hint(base + OFF_V + st * KV_TILE + KV_SUB, &tm_qkv, v_full(st), col_v + 64, j * BKV, seq, pol_kv);
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (ptx::elect_one()) {
      constexpr uint32_t idesc_qk = ptx::make_idesc_bf16(BQ, BKV, 0, 0);   // A = Q (K-major smem), B = K_j (K-major smem)
      constexpr uint32_t idesc_pv = ptx::make_idesc_bf16(BQ, DH, 0, 1);    // A = P (TMEM), B = V_j (MN-major smem)
      auto issue_qk = [&](int t, int g) {                                  // S_t(g) -> buffer g & 1
        const int st = g % KV_STAGES;
        const uint32_t qa = base + OFF_Q + t * Q_TILE, ka = base + OFF_K + st * KV_TILE;
        const uint32_t d = tmem_base + (uint32_t)(t * 128 + (g & 1) * 64);
#pragma unroll
        for (int k = 0; k < DH / 16; ++k)
          ptx::mma_f16_ss(d, ptx::make_smem_desc(qa + (k >> 2) * Q_SUB + (k & 3) * 32, 16, 1024),
                          ptx::make_smem_desc(ka + (k >> 2) * KV_SUB + (k & 3) * 32, 16, 1024), idesc_qk, k ? 1u : 0u);
        ptx::mma_commit(s_full(t, g & 1));
        if (t == QT - 1) ptx::mma_commit(k_empty(st));
      };
      int it = 0;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++it) {
        const int g0 = it * n_kv;
        ptx::mbar_wait(q_full, (uint32_t)(it & 1));
        for (int j = 0; j < 2 && j < n_kv; ++j) {           // the S buffers are free: every P of the previous item was
          const int g = g0 + j;                             // consumed by a P V issued before (in-order tensor pipe)
          ptx::mbar_wait(k_full(g % KV_STAGES), (uint32_t)(g / KV_STAGES) & 1u);
          ptx::tc_fence_after();
          issue_qk(0, g);
          issue_qk(1, g);
          if (j == n_kv - 1) ptx::mma_commit(q_empty);
        }
        for (int j = 0; j < n_kv; ++j) {
          const int g = g0 + j, st = g % KV_STAGES;
          ptx::mbar_wait(v_full(st), (uint32_t)(g / KV_STAGES) & 1u);
#pragma unroll
          for (int t = 0; t < QT; ++t) {
            ptx::mbar_wait(p_full(t, g & 1), (uint32_t)(g >> 1) & 1u);
            if (j == 0) ptx::mbar_wait(o_free(t), (uint32_t)(it & 1) ^ 1u);   // the previous item's epilogue has read O_t
            ptx::tc_fence_after();
            const uint32_t va = base + OFF_V + st * KV_TILE;
            const uint32_t p_tmem = tmem_base + (uint32_t)(t * 128 + (g & 1) * 64);
#pragma unroll
            for (int k = 0; k < BKV / 16; ++k)      // 16 keys = 8 packed TMEM columns of P, 16 rows (2048 bytes) of V
              mma_f16_ts(tmem_base + 256 + t * DH, p_tmem + k * 8, ptx::make_smem_desc(va + k * 2048, KV_SUB, 1024), idesc_pv,
                         (j | k) ? 1u : 0u);
            ptx::mma_commit(pv_done(t));
            if (j == n_kv - 1) ptx::mma_commit(o_final(t));
            if (t == QT - 1) ptx::mma_commit(v_empty(st));
            if (j + 2 < n_kv) {
              const int g2 = g + 2;
              if (t == 0) { ptx::mbar_wait(k_full(g2 % KV_STAGES), (uint32_t)(g2 / KV_STAGES) & 1u); ptx::tc_fence_after(); }
              issue_qk(t, g2);                      // overwrites the buffer P_t(g) sat in: ordered behind PV_t(g) in the pipe
              if (t == QT - 1 && j + 2 == n_kv - 1) ptx::mma_commit(q_empty);   // last Q K^T of the item: Q may be replaced
            }
          }
        }
      }
    }
  } else {
    // ===================== softmax / correction / epilogue: 2 warpgroups x 128 rows =====================
    const int t = (warp - 2) >> 2;                      // query tile of this warpgroup
    const int quarter = warp & 3;                       // TMEM lane quarter this warp may access
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const uint32_t tmem_s = tmem_base + t * 128 + lane_addr, tmem_o = tmem_base + 256 + t * DH + lane_addr;
    int it = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++it) {
      const int x = w % n_qt, head = (w / n_qt) % H, seq = w / (n_qt * H);
      const int q0 = x * (QT * BQ);
      float m_ref = -INFINITY, l = 0.f;
      for (int j = 0; j < n_kv; ++j) {
        const int g = it * n_kv + j, b = g & 1;
        ptx::mbar_wait(s_full(t, b), (uint32_t)(g >> 1) & 1u);
        ptx::tc_fence_after();
        const int valid = S - j * BKV;                   // keys of this tile that exist (>= 64 except the last)
        uint32_t sv[2][32];
        ptx::tmem_ld_32x32(tmem_s + b * 64, sv[0]);
        ptx::tmem_ld_32x32(tmem_s + b * 64 + 32, sv[1]);
        ptx::tmem_ld_wait();
        // full tiles (all but possibly the last) take a mask-free path: per-element validity tests cost 3 of the 8
        // instructions per score (ncu: 526 SASS instructions per tile and warp with them, 64 FMNMX + 64 FFMA + 64 MUFU
        // + 64 FADD + 32 F2FP without) and the softmax warps are issue-bound
        float mx = -INFINITY;
        if (valid >= BKV) {
#pragma unroll
          for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int i = 0; i < 32; i += 2)
              mx = fmaxf(mx, fmaxf(__uint_as_float(sv[c][i]), __uint_as_float(sv[c][i + 1])));
        } else {
#pragma unroll
          for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (c * 32 + i < valid) mx = fmaxf(mx, __uint_as_float(sv[c][i]));
        }
        const bool need = (mx - m_ref) * scale_log2 > RESCALE_THRESHOLD;     // true on the first tile (m_ref = -inf)
        if (__any_sync(0xffffffffu, need)) {
          const float m_new = fmaxf(m_ref, mx);
          if (j > 0) {
            ptx::mbar_wait(pv_done(t), (uint32_t)(g - 1) & 1u);             // O_t holds P V of tiles 0 .. j-1 of this item
            ptx::tc_fence_after();
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
        uint32_t pk[32];
        if (valid >= BKV) {
          float sum1 = 0.f;                                  // two independent accumulation chains
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const int c = i >> 4, e = (i & 15) * 2;
            const float p0 = ex2_approx(fmaf(__uint_as_float(sv[c][e]), scale_log2, -mc));
            const float p1 = ex2_approx(fmaf(__uint_as_float(sv[c][e + 1]), scale_log2, -mc));
            sum += p0;
            sum1 += p1;
            pk[i] = pack_bf16(p0, p1);
          }
          sum += sum1;
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const int c = i >> 4, e = (i & 15) * 2, key = 2 * i;
            float p0 = ex2_approx(fmaf(__uint_as_float(sv[c][e]), scale_log2, -mc));
            float p1 = ex2_approx(fmaf(__uint_as_float(sv[c][e + 1]), scale_log2, -mc));
            if (key >= valid) p0 = 0.f;
            if (key + 1 >= valid) p1 = 0.f;
            sum += p0 + p1;
            pk[i] = pack_bf16(p0, p1);
          }
        }
        ptx::tmem_st_32x32(tmem_s + b * 64, pk);
        l += sum;
        ptx::tmem_st_wait();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(p_full(t, b));
      }
      // epilogue: O / l -> bf16 (or E4M3).  (pv_done's parity is only unambiguous one phase back - the softmax of tile g
      // runs at most one P V ahead of it - so the end of the item's LAST P V has its own barrier.)
      // A thread owns a query ROW, so storing from registers sends 32 scattered 16-byte pieces per instruction (measured:
      // 4400-6000 cycles per item and query tile, 12-18 % of an S = 1280 item).  Instead each warp stages its 32 rows x
      // 128 bytes in 128-byte-swizzled shared memory and one lane hands them to a TMA store, which also clips rows >= S.
      ptx::mbar_wait(o_final(t), (uint32_t)(it & 1));
      ptx::tc_fence_after();
      const float inv = 1.f / l;
      const int row0 = q0 + t * BQ + quarter * 32;        // first row of this warp
      const uint32_t stg = base + OFF_STG + (uint32_t)(warp - 2) * STG_BYTES;
      const uint32_t stg_row = stg + (uint32_t)lane * 128u;
      const int sw = lane & 7;
      auto send = [&](int col) {                          // staging buffer -> out[seq, row0 .. row0 + 31, col ..]
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (ptx::elect_one()) {                           // the same lane every time: it owns the bulk async-groups
          if (row0 < S) ptx::tma_store_3d(&tm_out, stg, col, row0, seq);
          ptx::bulk_commit();
        }
      };
      auto acquire = [&]() {                              // the TMA engine has read the previous contents
        ptx::bulk_wait_read<0>();
        __syncwarp();
      };
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t ov[32];
        ptx::tmem_ld_32x32(tmem_o + c * 32, ov);
        ptx::tmem_ld_wait();
        if (c == 3) {                                     // O_t is in registers: the next item's first P V may overwrite it
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(o_free(t));
        }
        if (OUT8) {                                       // 128 E4M3 bytes per row: one buffer, one store
          if (c == 0) acquire();
#pragma unroll
          for (int g4 = 0; g4 < 2; ++g4) {
            uint32_t w4[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const int e = g4 * 16 + u * 4;
              const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(__uint_as_float(ov[e]) * inv, __uint_as_float(ov[e + 1]) * inv),
                                                           __NV_SATFINITE, __NV_E4M3);
              const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(__uint_as_float(ov[e + 2]) * inv, __uint_as_float(ov[e + 3]) * inv),
                                                           __NV_SATFINITE, __NV_E4M3);
              w4[u] = lo | (hi << 16);
            }
            st_shared_v4(stg_row + (uint32_t)(((c * 2 + g4) ^ sw) << 4), w4[0], w4[1], w4[2], w4[3]);
          }
          if (c == 3) send(head * DH);
        } else {                                          // 256 bf16 bytes per row: two buffers' worth, two stores
          if ((c & 1) == 0) acquire();
#pragma unroll
          for (int g4 = 0; g4 < 4; ++g4)
            st_shared_v4(stg_row + (uint32_t)((((c & 1) * 4 + g4) ^ sw) << 4),
                         pack_bf16(__uint_as_float(ov[g4 * 8]) * inv, __uint_as_float(ov[g4 * 8 + 1]) * inv),
                         pack_bf16(__uint_as_float(ov[g4 * 8 + 2]) * inv, __uint_as_float(ov[g4 * 8 + 3]) * inv),
                         pack_bf16(__uint_as_float(ov[g4 * 8 + 4]) * inv, __uint_as_float(ov[g4 * 8 + 5]) * inv),
                         pack_bf16(__uint_as_float(ov[g4 * 8 + 6]) * inv, __uint_as_float(ov[g4 * 8 + 7]) * inv));
          if (c & 1) send(head * DH + (c >> 1) * 64);
        }
      }
    }
    ptx::bulk_wait<0>();                                  // every store of this warp has completed before the CTA exits
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem_base, 512); }
}

}  // namespace

cudaError_t launch_attn_tcgen05_v3(const void* qkv, void* out, int B, int S, int H, int dh, int num_sms, cudaStream_t st,
                                   bool out_e4m3) {
  if (dh != DH) return cudaErrorInvalidValue;
  if (B <= 0) return cudaSuccess;
  CUtensorMap tm;
  memset(&tm, 0, sizeof(tm));
  const uint64_t dims[3] = {(uint64_t)3 * H * DH, (uint64_t)S, (uint64_t)B};
  const uint64_t strides[2] = {(uint64_t)3 * H * DH * 2, (uint64_t)S * 3 * H * DH * 2};
  const uint32_t box[3] = {64, 64, 1};
  SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm, qkv, 3, dims, strides, box));
  // output [B, S, H * d_h] as bf16 (box 64 columns x 32 rows) or E4M3 bytes (box 128 x 32): one warp's staging buffer
  CUtensorMap tmo;
  memset(&tmo, 0, sizeof(tmo));
  const uint64_t es = out_e4m3 ? 1 : 2;
  const uint64_t odims[3] = {(uint64_t)H * DH, (uint64_t)S, (uint64_t)B};
  const uint64_t ostrides[2] = {(uint64_t)H * DH * es, (uint64_t)S * H * DH * es};
  const uint32_t obox[3] = {out_e4m3 ? 128u : 64u, 32u, 1u};
  if (out_e4m3) SPOT_CUDA_TRY(spot_make_tmap_u8(&tmo, out, 3, odims, ostrides, obox));
  else SPOT_CUDA_TRY(spot_make_tmap_bf16(&tmo, out, 3, odims, ostrides, obox));
  static bool attr_set = false;
  if (!attr_set) {
    SPOT_CUDA_TRY(cudaFuncSetAttribute(attn_tcgen05_v3_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ATT_SMEM));
    SPOT_CUDA_TRY(cudaFuncSetAttribute(attn_tcgen05_v3_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ATT_SMEM));
    attr_set = true;
  }
  const long long items = (long long)((S + QT * BQ - 1) / (QT * BQ)) * H * B;
  if (items > 0x7fffffffLL / 128) return cudaErrorInvalidValue;
  // A/B only: SPOT_ATTN_L2_HINT = L2 policy of the K / V loads (tcgen05.cuh l2_policy).  Measured at config 3, two rounds:
  // 2477 / 2480 / 2475 ms for normal / evict_last / evict_first - no effect, so the default stays normal.
  static int kv_policy = -1;
  if (kv_policy < 0) { const char* e = getenv("SPOT_ATTN_L2_HINT"); kv_policy = e ? atoi(e) : 0; }
  const int grid = (int)(items < num_sms ? items : num_sms);       // persistent: one CTA per SM walks the item list
  const float scale_log2 = 1.4426950408889634f / sqrtf((float)DH);
  if (out_e4m3) attn_tcgen05_v3_kernel<true><<<grid, ATT_THREADS, ATT_SMEM, st>>>(tm, tmo, S, H, (int)items, scale_log2, kv_policy);
  else attn_tcgen05_v3_kernel<false><<<grid, ATT_THREADS, ATT_SMEM, st>>>(tm, tmo, S, H, (int)items, scale_log2, kv_policy);
  return cudaGetLastError();
}
