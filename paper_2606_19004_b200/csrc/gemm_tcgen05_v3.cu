// gemm_tcgen05_v3.cu - K2, CTA-pair GEMM with a TMA-store epilogue (the default since round 1b).
// Mainloop as gemm_tcgen05_2cta.cu: a cluster of two CTAs works on one 256 x 256 output tile with
// tcgen05.mma.cta_group::2 (M 256, N 256, K 16), a 6-stage TMA ring of 128-byte-swizzled K-major tiles and two
// 256-column TMEM accumulators, so the epilogue of tile i overlaps the mainloop of tile i + 1.
//
// What is new is the epilogue (warps 4-7 of each CTA, one TMEM lane quarter = 32 rows each; 8 warps, two per quarter, for
// the fused QKV epilogue on E4M3 operands - see epi_warps below):
//   * results leave the SM through shared memory and TMA instead of per-thread global accesses: each warp packs
//     32 rows x 128 bytes into its own swizzled staging buffer (two buffers per warp, so the TMA engine drains
//     one while the warp fills the other; the buffer is acquired as late as possible, behind the arithmetic) and one lane issues cp.async.bulk.tensor (store) - full 128-byte
//     lines, rows past the end of a sequence clipped by the tensor map;
//   * EPI_GATE_RES  h += gate * (y + bias): the tile of gate * (y + bias) is sent with cp.reduce.async.bulk.tensor
//     .add.f32, so the fp32 residual stream is never loaded by the SM (the add happens in the memory system; every
//     element belongs to exactly one tile, so the result does not depend on scheduling);
//   * EPI_BIAS_GELU uses tanh.approx.f32 (one MUFU op; abs. error < 2^-10, below the bf16 rounding of the output);
//   * EPI_QKV_ROPE  fuses K4 (north_star (c)) into the QKV projection: a 256-column tile is two whole heads and a
//     thread owns one token row of the accumulator, so the per-head RMS is thread-local: pass 1 over TMEM sums the
//     squares of (acc + bias), pass 2 scales by rsqrt(mean + eps) * gain, rotates pairs (2i, 2i+1) by the table
//     angle of the token's joint position and stores bf16.  v heads take the plain bias path.
#pragma nv_diag_suppress 128   // "loop is not reachable": the E4M3 QKV instantiation leaves the generic epilogue through `continue`
#include <cuda_fp8.h>
#include <stdlib.h>
#include <string.h>

#include "kernels.h"
#include "tcgen05.cuh"

namespace {

constexpr int BLOCK_M = 128 /*per CTA*/, PAIR_M = 256, BLOCK_N = 256, HALF_N = 128, BLOCK_K = 64, UMMA_K = 16;
constexpr int STAGES = 6;
constexpr uint32_t A_BYTES = BLOCK_M * BLOCK_K * 2, B_BYTES = HALF_N * BLOCK_K * 2, STAGE_BYTES = A_BYTES + B_BYTES;
constexpr uint32_t STG_BYTES = 32 * 128;                         // one staging buffer: 32 rows x 128 bytes
// Epilogue warps: 4 (one per TMEM lane quarter, two staging buffers each) or 8 (two per quarter: columns [0,128) and
// [128,256), one buffer each).  Measured: 8 warps only pay where the epilogue is the pace-maker, i.e. the fused
// QKV + RMSNorm + RoPE epilogue behind the half-as-long E4M3 mainloop (ncu 63 % tensor-pipe active with 4 warps; FP8
// rollout 1566 -> 1519 ms); every other instantiation is 1-5 % faster with 4 warps.
__host__ __device__ constexpr int epi_warps(int epi, bool fp8) { return (fp8 && epi == EPI_QKV_ROPE) ? 8 : 4; }
// Ring depth: the E4M3 QKV instantiation gives its sixth stage (32 KB) to the epilogue's per-warp column constants.
__host__ __device__ constexpr int ring_stages(int epi, bool fp8) { return (fp8 && epi == EPI_QKV_ROPE) ? STAGES - 1 : STAGES; }
constexpr uint32_t OFF_COLC = (STAGES - 1) * STAGE_BYTES;        // [8 warps][scale, bias, gain][128 columns] fp32 (that instantiation only)
constexpr int MAX_THREADS = 128 + 8 * 32;
constexpr uint32_t OFF_STG = STAGES * STAGE_BYTES;               // 8 staging buffers: 4 warps x 2 or 8 warps x 1
constexpr uint32_t OFF_BAR = OFF_STG + 8 * STG_BYTES;
constexpr uint32_t SMEM_BYTES = OFF_BAR + 256 /*barriers*/ + 1024 /*align slack*/;
static_assert(SMEM_BYTES <= 232448, "shared memory budget");

struct V3Problem {
  int m_tiles, n_tiles, tiles_per_seq, rps, N, k_blocks, tile_start;   // m_tiles counts 256-row pair tiles
  int group_m;              // rasterisation: tiles run n-major inside groups of group_m M-tiles (L2 residency)
  const bf16* bias;
  const float* gate;
  const float* w_scale;     // FP8 variant: per-output-channel dequantisation scale
  // EPI_QKV_ROPE
  const bf16* q_gain;
  const bf16* k_gain;
  const float* cos_t;
  const float* sin_t;
  int pos_off, hidden;
  float rms_eps;
};
struct V3Params {
  V3Problem p[2];
  int n_probs, total_tiles;
  int l2_a, l2_w, l2_o;     // L2 eviction priority of the A / W loads and of the output stores / reductions (tcgen05.cuh l2_policy: 0 normal, 1 evict_last, 2 evict_first)
};
struct TileCoord { int prob, mt, nt; };

__device__ __forceinline__ TileCoord decode_tile(const V3Params& P, int t) {
  TileCoord c;
  c.prob = (P.n_probs > 1 && t >= P.p[1].tile_start) ? 1 : 0;
  const V3Problem& q = P.p[c.prob];
  t -= q.tile_start;
  const int per_group = q.group_m * q.n_tiles;
  const int g = t / per_group, first_m = g * q.group_m;
  const int gm = min(q.group_m, q.m_tiles - first_m);
  const int r = t - g * per_group;
  c.mt = first_m + r % gm;
  c.nt = r / gm;
  return c;
}

__device__ __forceinline__ float tanh_approx(float x) {
  float y;
  asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float gelu_tanh_fast(float x) {
  const float k0 = 0.7978845608028654f, k1 = 0.7978845608028654f * 0.044715f;
  const float x2 = x * x;
  const float inner = x * fmaf(k1, x2, k0);
  const float hx = 0.5f * x;
  return fmaf(hx, tanh_approx(inner), hx);
}
__device__ __forceinline__ uint32_t pack2(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
// acc (fp32 bits from TMEM) + bias for 32 consecutive columns starting at bias pointer bp (16-byte aligned)
__device__ __forceinline__ void add_bias32(const uint32_t (&v)[32], const bf16* bp, float (&y)[32]) {
  const uint4* p4 = reinterpret_cast<const uint4*>(bp);
#pragma unroll
  for (int g = 0; g < 4; ++g) {
    uint4 braw = __ldg(p4 + g);
    const bf16* bb = reinterpret_cast<const bf16*>(&braw);
#pragma unroll
    for (int j = 0; j < 8; ++j) y[g * 8 + j] = __uint_as_float(v[g * 8 + j]) + __bfloat162float(bb[j]);
  }
}
// FP8 variant: y = acc * w_scale[n] + bias[n]  (per-output-channel dequantisation, DESIGN.md section 13 reading Q4)
__device__ __forceinline__ void scale_bias32(const uint32_t (&v)[32], const float* sp, const bf16* bp, float (&y)[32]) {
  const uint4* p4 = reinterpret_cast<const uint4*>(bp);
  const float4* s4 = reinterpret_cast<const float4*>(sp);
#pragma unroll
  for (int g = 0; g < 4; ++g) {
    uint4 braw = __ldg(p4 + g);
    const bf16* bb = reinterpret_cast<const bf16*>(&braw);
    const float4 sa = __ldg(s4 + 2 * g), sb = __ldg(s4 + 2 * g + 1);
    const float sc[8] = {sa.x, sa.y, sa.z, sa.w, sb.x, sb.y, sb.z, sb.w};
#pragma unroll
    for (int j = 0; j < 8; ++j) y[g * 8 + j] = fmaf(__uint_as_float(v[g * 8 + j]), sc[j], __bfloat162float(bb[j]));
  }
}
template <bool FP8>
__device__ __forceinline__ void acc_to_y(const uint32_t (&v)[32], const float* sp, const bf16* bp, float (&y)[32]) {
  if (FP8) scale_bias32(v, sp, bp, y);
  else add_bias32(v, bp, y);
}
__device__ __forceinline__ uint32_t pack4_e4m3(float a, float b, float c, float d) {
  const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3);
  const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(c, d), __NV_SATFINITE, __NV_E4M3);
  return lo | (hi << 16);
}
// 32 fp32 values -> 32 bytes of E4M3 = 16-byte chunks c0, c0+1 of this thread's 128-byte staging row
__device__ __forceinline__ void stage_e4m3_32(uint32_t row_addr, int sw, int c0, const float (&y)[32]) {
#pragma unroll
  for (int g = 0; g < 2; ++g)
    st_shared_v4(row_addr + (uint32_t)(((c0 + g) ^ sw) << 4), pack4_e4m3(y[16 * g], y[16 * g + 1], y[16 * g + 2], y[16 * g + 3]),
                 pack4_e4m3(y[16 * g + 4], y[16 * g + 5], y[16 * g + 6], y[16 * g + 7]),
                 pack4_e4m3(y[16 * g + 8], y[16 * g + 9], y[16 * g + 10], y[16 * g + 11]),
                 pack4_e4m3(y[16 * g + 12], y[16 * g + 13], y[16 * g + 14], y[16 * g + 15]));
}
// 32 fp32 values -> 64 bytes of bf16 = 16-byte chunks c0 .. c0+3 of this thread's 128-byte staging row
__device__ __forceinline__ void stage_bf16_32(uint32_t row_addr, int sw, int c0, const float (&y)[32]) {
#pragma unroll
  for (int g = 0; g < 4; ++g)
    st_shared_v4(row_addr + (uint32_t)(((c0 + g) ^ sw) << 4), pack2(y[8 * g], y[8 * g + 1]), pack2(y[8 * g + 2], y[8 * g + 3]),
                 pack2(y[8 * g + 4], y[8 * g + 5]), pack2(y[8 * g + 6], y[8 * g + 7]));
}

// Loads whose issue point is pinned (volatile asm keeps its program order): used to start a load long before its use.
__device__ __forceinline__ float4 ldg_nc_f4(const float* p) {
  float4 v;
  asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint2 ldg_nc_u2(const void* p) {
  uint2 v;
  asm volatile("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}
struct ColConst { float4 s; uint2 b, g; };                       // scale, bias, gain of 4 consecutive columns (bf16 pairs raw)
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// FP8 = true: A and W are E4M3 (kind::f8f6f4, K = 32 per MMA; a 128-byte swizzled row then holds 128 elements, so a
// stage is a 128-element K block and everything else - ring, descriptors, 32-byte advance per MMA - is unchanged);
// accumulators are dequantised per output channel; EPI_BIAS / EPI_BIAS_GELU then store E4M3 (the next Linear's operand).
template <int EPI, bool FP8>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(MAX_THREADS, 1)
gemm_tcgen05_v3_kernel(const __grid_constant__ CUtensorMap tmA0, const __grid_constant__ CUtensorMap tmW0,
                       const __grid_constant__ CUtensorMap tmO0, const __grid_constant__ CUtensorMap tmA1,
                       const __grid_constant__ CUtensorMap tmW1, const __grid_constant__ CUtensorMap tmO1,
                       const V3Params P) {
  extern __shared__ uint8_t smem_raw[];
  constexpr int NST = ring_stages(EPI, FP8);
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + OFF_BAR;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
  volatile uint32_t* tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

  const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;   // warp index uniform FOR THE COMPILER (tcgen05.cuh)
  const uint32_t rank = __shfl_sync(0xffffffffu, ptx::cluster_ctarank(), 0);   // 0 = leader of the pair (uniform for the compiler)
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmA0); ptx::prefetch_tmap(&tmW0); ptx::prefetch_tmap(&tmO0);
    if (P.n_probs > 1) { ptx::prefetch_tmap(&tmA1); ptx::prefetch_tmap(&tmW1); ptx::prefetch_tmap(&tmO1); }
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < NST; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), 2 * epi_warps(EPI, FP8)); }
    ptx::fence_barrier_init();
  }
  if (warp == 2) { ptx::tmem_alloc_2cta(tmem_slot, 512); ptx::tmem_relinquish_2cta(); }
  ptx::tc_fence_before();
  ptx::cluster_sync();                                      // barriers of both CTAs initialised, TMEM allocated
  ptx::tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot_ptr, 0);

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    // elect.sync (not `lane == 0`): the compiler then knows the region is single-threaded and issues UTMALDG /
    // UTCHMMA straight from uniform registers (see "single-thread issue paths" in tcgen05.cuh)
    if (ptx::elect_one()) {
      int stage = 0; uint32_t phase = 0;
      const uint64_t pol_a = ptx::l2_policy(P.l2_a), pol_w = ptx::l2_policy(P.l2_w);
      for (int t = pair; t < P.total_tiles; t += n_pairs) {
        const TileCoord c = decode_tile(P, t);
        const V3Problem& q = P.p[c.prob];
        const CUtensorMap* mA = c.prob ? &tmA1 : &tmA0;
        const CUtensorMap* mW = c.prob ? &tmW1 : &tmW0;
        const int seq = c.mt / q.tiles_per_seq;
        const int r0 = (c.mt - seq * q.tiles_per_seq) * PAIR_M + (int)rank * BLOCK_M;
        const int n0 = c.nt * BLOCK_N + (int)rank * HALF_N;
        for (int kb = 0; kb < q.k_blocks; ++kb) {
          ptx::mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t leader_full = ptx::map_to_cta(full_bar(stage), 0);
          const uint32_t sa = smem_base + stage * STAGE_BYTES;
          ptx::tma_load_3d_2cta_hint(sa, mA, leader_full, kb * (FP8 ? 2 * BLOCK_K : BLOCK_K), r0, seq, pol_a);
          ptx::tma_load_2d_2cta_hint(sa + A_BYTES, mW, leader_full, kb * (FP8 ? 2 * BLOCK_K : BLOCK_K), n0, pol_w);
          // only the leader CTA arms its barrier, for the bytes of BOTH CTAs (see gemm_tcgen05_2cta.cu)
          if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), 2 * STAGE_BYTES);
          if (++stage == NST) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only, one elected thread) =====================
    // (the non-leader CTA runs the same code over zero tiles: a branch on `rank` around the elected region makes the
    //  compiler fall back to per-lane ELECT / BRA.U.ANY loops around every UTCHMMA)
    if (ptx::elect_one()) {
      const int my_tiles = rank == 0 ? P.total_tiles : 0;
      constexpr uint32_t idesc = FP8 ? ptx::make_idesc_e4m3(PAIR_M, BLOCK_N) : ptx::make_idesc_bf16(PAIR_M, BLOCK_N, 0, 0);
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t acc_phase = 0;
      for (int t = pair; t < my_tiles; t += n_pairs) {
        const TileCoord c = decode_tile(P, t);
        const int k_blocks = P.p[c.prob].k_blocks;
        ptx::mbar_wait(tempty_bar(acc), acc_phase ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BLOCK_N;
        for (int kb = 0; kb < k_blocks; ++kb) {
          ptx::mbar_wait(full_bar(stage), phase);
          ptx::tc_fence_after();
          const uint32_t sa = smem_base + stage * STAGE_BYTES, sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BLOCK_K / UMMA_K; ++k) {
            const uint64_t da = ptx::make_smem_desc(sa + k * UMMA_K * 2, 16, 1024);
            const uint64_t db = ptx::make_smem_desc(sb + k * UMMA_K * 2, 16, 1024);
            if (FP8) ptx::mma_f8_ss_2cta(d_tmem, da, db, idesc, (kb | k) ? 1u : 0u);
            else ptx::mma_f16_ss_2cta(d_tmem, da, db, idesc, (kb | k) ? 1u : 0u);
          }
          ptx::mma_commit_2cta(empty_bar(stage));
          if (kb == k_blocks - 1) ptx::mma_commit_2cta(tfull_bar(acc));
          if (++stage == NST) { stage = 0; phase ^= 1; }
        }
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue (both CTAs, own 128 TMEM lanes) =====================
    constexpr int EW = epi_warps(EPI, FP8), NBUF = 8 / EW;
    const int q4 = warp & 3, half = (warp - 4) >> 2;       // EW == 8: warps 8-11 take columns [128,256) of the tile
    const int col_lo = EW == 8 ? half : 0, col_hi = EW == 8 ? half + 1 : 2;   // range of 128-column half tiles of this warp
    const uint32_t stg0 = smem_base + OFF_STG + (uint32_t)(warp - 4) * NBUF * STG_BYTES;
    int buf = 0;
    const uint32_t row_off = (uint32_t)lane * 128u;
    const int sw = lane & 7;
    int acc = 0; uint32_t acc_phase = 0;
    // E4M3 QKV instantiation: this warp's column constants [scale | bias | gain][128] fp32 in the unused sixth stage
    const uint32_t colc_addr = smem_base + OFF_COLC + (uint32_t)(warp - 4) * 1536u;
    const float4* colc = reinterpret_cast<const float4*>(smem_raw + (colc_addr - ptx::smem_u32(smem_raw)));
    auto load_colconst = [&](int t, ColConst& cc) {          // lane l: columns 4l .. 4l+3 of this warp's head in tile t
      const TileCoord c = decode_tile(P, t);
      const V3Problem& q = P.p[c.prob];
      const int hcol0 = c.nt * BLOCK_N + half * 128;
      cc.s = make_float4(0.f, 0.f, 0.f, 0.f);
      cc.b = make_uint2(0u, 0u);
      cc.g = make_uint2(0x3f803f80u, 0x3f803f80u);
      if (hcol0 < q.N) {
        cc.s = ldg_nc_f4(q.w_scale + hcol0 + lane * 4);
        cc.b = ldg_nc_u2(q.bias + hcol0 + lane * 4);
        const int which = hcol0 / q.hidden;
        if (which < 2) cc.g = ldg_nc_u2((which ? q.k_gain : q.q_gain) + lane * 4);
      }
    };
    auto store_colconst = [&](const ColConst& cc) {
      __syncwarp();
      st_shared_v4(colc_addr + lane * 16, __float_as_uint(cc.s.x), __float_as_uint(cc.s.y), __float_as_uint(cc.s.z), __float_as_uint(cc.s.w));
      st_shared_v4(colc_addr + 512 + lane * 16, __float_as_uint(bf16_lo(cc.b.x)), __float_as_uint(bf16_hi(cc.b.x)),
                   __float_as_uint(bf16_lo(cc.b.y)), __float_as_uint(bf16_hi(cc.b.y)));
      st_shared_v4(colc_addr + 1024 + lane * 16, __float_as_uint(bf16_lo(cc.g.x)), __float_as_uint(bf16_hi(cc.g.x)),
                   __float_as_uint(bf16_lo(cc.g.y)), __float_as_uint(bf16_hi(cc.g.y)));
      __syncwarp();
    };
    if constexpr (EPI == EPI_QKV_ROPE && FP8) {
      if (pair < P.total_tiles) { ColConst first; load_colconst(pair, first); store_colconst(first); }
    }
    const uint64_t pol_o = ptx::l2_policy(P.l2_o);
    for (int t = pair; t < P.total_tiles; t += n_pairs) {
      const TileCoord c = decode_tile(P, t);
      const V3Problem& q = P.p[c.prob];
      const CUtensorMap* mO = c.prob ? &tmO1 : &tmO0;
      const int seq = c.mt / q.tiles_per_seq;
      const int row0 = (c.mt - seq * q.tiles_per_seq) * PAIR_M + (int)rank * BLOCK_M + q4 * 32;   // first row of this warp
      const bool warp_ok = row0 < q.rps;                    // whole warp past the end of the sequence: nothing to store
      const uint32_t taddr0 = tmem_base + acc * BLOCK_N + ((uint32_t)(q4 * 32) << 16);
      const int ncol0 = c.nt * BLOCK_N;

      // hand a filled staging buffer to the TMA engine
      auto send = [&](int n0) {
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (ptx::elect_one()) {                           // deterministic: the same lane every time (it owns the bulk groups)
          if (warp_ok) {
            if (EPI == EPI_GATE_RES) ptx::tma_reduce_add_3d_hint(mO, stg0 + buf * STG_BYTES, n0, row0, seq, pol_o);
            else ptx::tma_store_3d_hint(mO, stg0 + buf * STG_BYTES, n0, row0, seq, pol_o);
          }
          ptx::bulk_commit();
        }
        if (NBUF == 2) buf ^= 1;
      };
      // wait until the TMA engine has read the warp's staging buffer (called after the chunk's TMEM load was issued
      // and right before the first shared-memory store, so the wait overlaps the load and the arithmetic)
      auto acquire = [&]() {
        ptx::bulk_wait_read<NBUF - 1>();                  // the elected lane waits for its groups; trivially true elsewhere
        __syncwarp();
        return stg0 + buf * STG_BYTES + row_off;
      };

      if constexpr (EPI == EPI_QKV_ROPE && FP8) {
        // Behind the half-as-long E4M3 mainloop this epilogue sets the pace, and what it waited for was global loads
        // (ncu: 61 % of its samples on the long scoreboard - L1 is ~27 KB next to the 225 KB of shared memory, so the
        // per-column vectors and the per-row rotation tables arrive from L2 at every 32-column chunk).  Here each warp
        // owns one head (128 columns) of the tile: the column constants (scale, bias, gain) sit in shared memory,
        // loaded one tile ahead; the rotation table is loaded two chunks ahead, the first two before the accumulator
        // is even waited for.
        const int hcol0 = ncol0 + half * 128;
        const bool head_ok = hcol0 < q.N;
        const int which = head_ok ? hcol0 / q.hidden : 2;       // 0 = q, 1 = k, 2 = v (warp-uniform)
        const bool rope = which < 2;
        ColConst nxt;
        const bool have_next = t + n_pairs < P.total_tiles;
        if (have_next) load_colconst(t + n_pairs, nxt);
        float4 cA[4], sA[4], cB[4], sB[4];
        const int row = row0 + lane;
        const long long pos = q.pos_off + (row < q.rps ? row : 0);
        const float* cs = q.cos_t + pos * 64;
        const float* sn = q.sin_t + pos * 64;
        if (rope) {
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            cA[g] = ldg_nc_f4(cs + 4 * g); sA[g] = ldg_nc_f4(sn + 4 * g);
            cB[g] = ldg_nc_f4(cs + 16 + 4 * g); sB[g] = ldg_nc_f4(sn + 16 + 4 * g);
          }
        }
        ptx::mbar_wait(tfull_bar(acc), acc_phase);
        ptx::tc_fence_after();
        if (head_ok) {
          float rinv = 0.f;
          if (rope) {                                          // pass 1: sum of squares of (scale * acc + bias) over the head
            float ss0 = 0.f, ss1 = 0.f;
#pragma unroll 1
            for (int c4 = 0; c4 < 4; ++c4) {
              uint32_t v[32];
              ptx::tmem_ld_32x32(taddr0 + half * 128 + c4 * 32, v);
              ptx::tmem_ld_wait();
#pragma unroll
              for (int g = 0; g < 8; ++g) {
                const float4 sc = colc[c4 * 8 + g], bi = colc[32 + c4 * 8 + g];
                const float y0 = fmaf(__uint_as_float(v[4 * g]), sc.x, bi.x), y1 = fmaf(__uint_as_float(v[4 * g + 1]), sc.y, bi.y);
                const float y2 = fmaf(__uint_as_float(v[4 * g + 2]), sc.z, bi.z), y3 = fmaf(__uint_as_float(v[4 * g + 3]), sc.w, bi.w);
                ss0 = fmaf(y0, y0, ss0); ss1 = fmaf(y1, y1, ss1);
                ss0 = fmaf(y2, y2, ss0); ss1 = fmaf(y3, y3, ss1);
              }
            }
            rinv = rsqrtf((ss0 + ss1) * (1.f / 128.f) + q.rms_eps);
          }
          uint32_t ra = 0;
#pragma unroll
          for (int k = 0; k < 4; ++k) {                         // pass 2, 32 columns at a time; two of them fill a staging row
            uint32_t v[32];
            ptx::tmem_ld_32x32(taddr0 + half * 128 + k * 32, v);
            ptx::tmem_ld_wait();
            float y[32];
#pragma unroll
            for (int g = 0; g < 8; ++g) {
              const float4 sc = colc[k * 8 + g], bi = colc[32 + k * 8 + g];
              y[4 * g] = fmaf(__uint_as_float(v[4 * g]), sc.x, bi.x);
              y[4 * g + 1] = fmaf(__uint_as_float(v[4 * g + 1]), sc.y, bi.y);
              y[4 * g + 2] = fmaf(__uint_as_float(v[4 * g + 2]), sc.z, bi.z);
              y[4 * g + 3] = fmaf(__uint_as_float(v[4 * g + 3]), sc.w, bi.w);
            }
            if (rope) {
              float4 (&cc)[4] = (k & 1) ? cB : cA;
              float4 (&sd)[4] = (k & 1) ? sB : sA;
#pragma unroll
              for (int g = 0; g < 8; ++g) {                     // 4 columns = 2 rotation pairs
                const float4 gn = colc[64 + k * 8 + g];
                const float a0 = y[4 * g] * rinv * gn.x, b0 = y[4 * g + 1] * rinv * gn.y;
                const float a1 = y[4 * g + 2] * rinv * gn.z, b1 = y[4 * g + 3] * rinv * gn.w;
                const float c0 = (g & 1) ? cc[g >> 1].z : cc[g >> 1].x, s0 = (g & 1) ? sd[g >> 1].z : sd[g >> 1].x;
                const float c1 = (g & 1) ? cc[g >> 1].w : cc[g >> 1].y, s1 = (g & 1) ? sd[g >> 1].w : sd[g >> 1].y;
                y[4 * g] = a0 * c0 - b0 * s0;
                y[4 * g + 1] = a0 * s0 + b0 * c0;
                y[4 * g + 2] = a1 * c1 - b1 * s1;
                y[4 * g + 3] = a1 * s1 + b1 * c1;
              }
              if (k < 2) {                                      // this buffer's next use is chunk k + 2
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                  cc[g] = ldg_nc_f4(cs + (k + 2) * 16 + 4 * g);
                  sd[g] = ldg_nc_f4(sn + (k + 2) * 16 + 4 * g);
                }
              }
            }
            if ((k & 1) == 0) ra = acquire();
            stage_bf16_32(ra, sw, (k & 1) * 4, y);
            if (k & 1) send(hcol0 + (k >> 1) * 64);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster(ptx::map_to_cta(tempty_bar(acc), 0));
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        if (have_next) store_colconst(nxt);                     // all lanes are past their reads of this tile's constants
        continue;
      }
      ptx::mbar_wait(tfull_bar(acc), acc_phase);
      ptx::tc_fence_after();
      if (EPI == EPI_GATE_RES) {
#pragma unroll 1
        for (int ch = col_lo * 4; ch < col_hi * 4; ++ch) {
          const int n0 = ncol0 + ch * 32;
          if (n0 >= q.N) break;
          uint32_t v[32];
          ptx::tmem_ld_32x32(taddr0 + ch * 32, v);
          ptx::tmem_ld_wait();
          float y[32];
          acc_to_y<FP8>(v, q.w_scale + n0, q.bias + n0, y);
          const float4* gp = reinterpret_cast<const float4*>(q.gate + n0);
          const uint32_t ra = acquire();
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            const float4 gt = __ldg(gp + g);
            st_shared_v4(ra + (uint32_t)((g ^ sw) << 4), __float_as_uint(gt.x * y[4 * g]), __float_as_uint(gt.y * y[4 * g + 1]),
                         __float_as_uint(gt.z * y[4 * g + 2]), __float_as_uint(gt.w * y[4 * g + 3]));
          }
          send(n0);
        }
      } else {
        const int row = row0 + lane;                          // row inside the sequence (may be past its end)
#pragma unroll 1
        for (int hh = col_lo; hh < col_hi; ++hh) {            // a 128-column half tile = one head of the QKV output
          const int hcol0 = ncol0 + hh * 128;
          if (hcol0 >= q.N) break;
          float rinv = 0.f;
          const bf16* gain = nullptr;
          const float* cs = nullptr;
          const float* sn = nullptr;
          if (EPI == EPI_QKV_ROPE) {
            const int which = hcol0 / q.hidden;               // 0 = q, 1 = k, 2 = v
            if (which < 2) {
              gain = which ? q.k_gain : q.q_gain;
              const long long pos = q.pos_off + (row < q.rps ? row : 0);
              cs = q.cos_t + pos * 64;
              sn = q.sin_t + pos * 64;
              float ss = 0.f;                                 // pass 1: sum of squares of (acc + bias) over the head
#pragma unroll 1
              for (int c4 = 0; c4 < 4; ++c4) {
                uint32_t v[32];
                ptx::tmem_ld_32x32(taddr0 + hh * 128 + c4 * 32, v);
                ptx::tmem_ld_wait();
                float y[32];
                acc_to_y<FP8>(v, q.w_scale + hcol0 + c4 * 32, q.bias + hcol0 + c4 * 32, y);
#pragma unroll
                for (int j = 0; j < 32; ++j) ss = fmaf(y[j], y[j], ss);
              }
              rinv = rsqrtf(ss * (1.f / 128.f) + q.rms_eps);
            }
          }
          if (FP8 && EPI != EPI_QKV_ROPE) {                  // E4M3 output: 128 columns = 128 bytes per row, one send per half tile
            uint32_t ra = 0;
#pragma unroll 1
            for (int c4 = 0; c4 < 4; ++c4) {
              const int n0 = hcol0 + c4 * 32;
              float y[32];
              if (n0 < q.N) {
                uint32_t v[32];
                ptx::tmem_ld_32x32(taddr0 + hh * 128 + c4 * 32, v);
                ptx::tmem_ld_wait();
                scale_bias32(v, q.w_scale + n0, q.bias + n0, y);
                if (EPI == EPI_BIAS_GELU) {
#pragma unroll
                  for (int j = 0; j < 32; ++j) y[j] = gelu_tanh_fast(y[j]);
                }
              } else {
#pragma unroll
                for (int j = 0; j < 32; ++j) y[j] = 0.f;
              }
              if (c4 == 0) ra = acquire();
              stage_e4m3_32(ra, sw, c4 * 2, y);
            }
            send(hcol0);
            continue;
          }
#pragma unroll 1
          for (int c2 = 0; c2 < 2; ++c2) {                    // 64 columns = 128 bytes of bf16 per row
            const int n0 = hcol0 + c2 * 64;
            if (n0 >= q.N) break;
            const bool second = n0 + 32 < q.N;
            uint32_t v0[32], v1[32];
            ptx::tmem_ld_32x32(taddr0 + hh * 128 + c2 * 64, v0);
            ptx::tmem_ld_32x32(taddr0 + hh * 128 + c2 * 64 + 32, v1);
            uint32_t ra = 0;
            ptx::tmem_ld_wait();
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
              float y[32];
              if (hf == 0) acc_to_y<FP8>(v0, q.w_scale + n0, q.bias + n0, y);
              else if (second) acc_to_y<FP8>(v1, q.w_scale + n0 + 32, q.bias + n0 + 32, y);
              else {
#pragma unroll
                for (int j = 0; j < 32; ++j) y[j] = 0.f;
              }
              if (EPI == EPI_BIAS_GELU) {
#pragma unroll
                for (int j = 0; j < 32; ++j) y[j] = gelu_tanh_fast(y[j]);
              }
              if (EPI == EPI_QKV_ROPE && gain != nullptr) {
                const int hc = c2 * 64 + hf * 32;             // first column of this group inside the head
                const uint4* g4 = reinterpret_cast<const uint4*>(gain + hc);
                const float4* c4p = reinterpret_cast<const float4*>(cs + hc / 2);
                const float4* s4p = reinterpret_cast<const float4*>(sn + hc / 2);
#pragma unroll
                for (int g = 0; g < 4; ++g) {                 // 8 columns = 4 rotation pairs
                  uint4 graw = __ldg(g4 + g);
                  const bf16* gg = reinterpret_cast<const bf16*>(&graw);
                  const float4 cv = __ldg(c4p + g), sv = __ldg(s4p + g);
                  const float cc[4] = {cv.x, cv.y, cv.z, cv.w}, sd[4] = {sv.x, sv.y, sv.z, sv.w};
#pragma unroll
                  for (int pr = 0; pr < 4; ++pr) {
                    const float a = y[8 * g + 2 * pr] * rinv * __bfloat162float(gg[2 * pr]);
                    const float b = y[8 * g + 2 * pr + 1] * rinv * __bfloat162float(gg[2 * pr + 1]);
                    y[8 * g + 2 * pr] = a * cc[pr] - b * sd[pr];
                    y[8 * g + 2 * pr + 1] = a * sd[pr] + b * cc[pr];
                  }
                }
              }
              if (hf == 0) ra = acquire();                    // as late as possible: the previous chunk's TMA read overlaps the math
              stage_bf16_32(ra, sw, hf * 4, y);
            }
            send(n0);
          }
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster(ptx::map_to_cta(tempty_bar(acc), 0));
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
    ptx::bulk_wait<0>();                                    // all stores of this warp have completed
  }

  ptx::tc_fence_before();
  ptx::cluster_sync();                                      // nobody of the pair still uses TMEM or remote barriers
  if (warp == 2) { ptx::tc_fence_after(); ptx::tmem_dealloc_2cta(tmem_base, 512); }
}

}  // namespace

bool tcgen05_v3_qkv_rope_supported(const GemmProblem& g) {
  return g.N % 3 == 0 && (g.N / 3) % 128 == 0 && g.q_gain && g.k_gain && g.cos_t && g.sin_t && g.pos_off >= 0 &&
         reinterpret_cast<uintptr_t>(g.q_gain) % 16 == 0 && reinterpret_cast<uintptr_t>(g.k_gain) % 16 == 0 &&
         reinterpret_cast<uintptr_t>(g.cos_t) % 16 == 0 && reinterpret_cast<uintptr_t>(g.sin_t) % 16 == 0;
}

cudaError_t launch_gemm_tcgen05_v3(Epilogue epi, const GemmProblem* probs, int n_probs, int num_sms, cudaStream_t st) {
  if (n_probs < 1 || n_probs > 2) return cudaErrorInvalidValue;
  V3Params P;
  memset(&P, 0, sizeof(P));
  {
    // L2 eviction priorities: both operands evict_last, outputs (stores and the residual reduce-add) evict_first.  A tile of
    // A is re-read by the other N tiles of its raster group and a tile of W by the other M tiles, while an output line is
    // never read again by this kernel; without the hints the 0.2-0.5 GB a launch writes push operand lines out.  Measured
    // at config 3, same box, back to back, two rounds: 2469.5 / 2473.9 ms (no hints) -> 2414.2 / 2416.5 ms; A evict_first
    // instead: 2651 ms and 2.2-4.1 GB of DRAM reads per launch (profiles/r2_gemm_l2.md).  SPOT_GEMM_L2_HINT =
    // 100 * output + 10 * A + W policy (0 normal, 1 evict_last, 2 evict_first) overrides, for A/B timing only.
    static int hint = -1;
    if (hint < 0) { const char* e = getenv("SPOT_GEMM_L2_HINT"); hint = e ? atoi(e) : 211; }
    P.l2_o = hint / 100; P.l2_a = hint / 10 % 10; P.l2_w = hint % 10;
  }
  CUtensorMap tm[6];
  memset(tm, 0, sizeof(tm));
  int tiles = 0, np = 0;
  bool fp8 = false;
  for (int i = 0; i < n_probs; ++i) {
    const GemmProblem& g = probs[i];
    if (g.M <= 0) continue;
    if (np > 0 && (g.fp8 != 0) != fp8) return cudaErrorInvalidValue;   // both problems of a launch share the operand type
    fp8 = g.fp8 != 0;
    const int es = fp8 ? 1 : 2;                     // bytes per operand element
    const int bk = fp8 ? 2 * BLOCK_K : BLOCK_K;     // operand elements per 128-byte K block
    const bool out8 = fp8 && (epi == EPI_BIAS || epi == EPI_BIAS_GELU);
    if (!tcgen05_gemm_supported(g)) return cudaErrorInvalidValue;
    if ((epi == EPI_GATE_RES) != (g.resid != nullptr)) return cudaErrorInvalidValue;
    if (epi != EPI_GATE_RES && !g.out) return cudaErrorInvalidValue;
    if (epi == EPI_QKV_ROPE && !tcgen05_v3_qkv_rope_supported(g)) return cudaErrorInvalidValue;
    V3Problem& q = P.p[np];
    const int rps = g.a_map.rows_per_seq, nseq = g.M / rps;
    q.rps = rps;
    q.tiles_per_seq = (rps + PAIR_M - 1) / PAIR_M;
    q.m_tiles = nseq * q.tiles_per_seq;
    q.n_tiles = (g.N + BLOCK_N - 1) / BLOCK_N;
    q.N = g.N;
    q.k_blocks = (g.K + bk - 1) / bk;
    q.tile_start = tiles;
    {
      // Rasterisation: tiles of one group sweep all N for group_m M-tiles, so a wave of 74 pair tiles touches
      // ~group_m A panels and 74 / group_m W panels.  Measured at config 3 (M = 20480; TFLOP/s alone, group 2 / 8 / 16):
      // QKV (N 9216, K 3072) 1594 / 1622 / 1658, fc1 (N 12288) 1506 / 1575 / 1627, out-proj (N 3072) 1627 / 1606 / 1585,
      // fc2 (N 3072, K 12288) 1521 / 1505 / 1493: wide outputs want tall groups (W is re-used from L2 across 16 M-tiles),
      // narrow outputs want short ones.  SPOT_GEMM_GROUP_M overrides (A/B timing only).
      static int forced = -1;
      if (forced < 0) { const char* e = getenv("SPOT_GEMM_GROUP_M"); forced = e ? atoi(e) : 0; }
      static int narrow = -1;                       // A/B only: group height of the narrow-output GEMMs (out-proj, fc2)
      if (narrow < 0) { const char* e = getenv("SPOT_GEMM_GROUP_M_NARROW"); narrow = e ? atoi(e) : 0; }
      int gm = narrow > 0 ? narrow : 2;
      if (q.n_tiles >= 24) {
        gm = (int)(25.0e6 / ((double)es * PAIR_M * (double)g.K));  // A panel of a group ~25 MB
        if (gm > 16) gm = 16;
        if (gm < 2) gm = 2;
      }
      q.group_m = forced > 0 ? forced : gm;
    }
    q.bias = (const bf16*)g.bias;
    q.gate = g.gate;
    q.w_scale = g.w_scale;
    q.q_gain = (const bf16*)g.q_gain; q.k_gain = (const bf16*)g.k_gain;
    q.cos_t = g.cos_t; q.sin_t = g.sin_t; q.pos_off = g.pos_off; q.hidden = g.N / 3; q.rms_eps = g.rms_eps;
    tiles += q.m_tiles * q.n_tiles;
    const uint64_t adims[3] = {(uint64_t)g.K, (uint64_t)rps, (uint64_t)nseq};
    const uint64_t astr[2] = {(uint64_t)g.a_map.ld * es,
                              (uint64_t)(nseq > 1 ? g.a_map.seq_stride : g.a_map.ld * (long long)rps) * es};
    const uint32_t abox[3] = {(uint32_t)bk, BLOCK_M, 1};
    const uint64_t wdims[2] = {(uint64_t)g.K, (uint64_t)g.N};
    const uint64_t wstr[1] = {(uint64_t)g.K * es};
    const uint32_t wbox[2] = {(uint32_t)bk, HALF_N};
    if (fp8) {
      SPOT_CUDA_TRY(spot_make_tmap_u8(&tm[3 * np], (const uint8_t*)g.A + g.a_map.offset, 3, adims, astr, abox));
      SPOT_CUDA_TRY(spot_make_tmap_u8(&tm[3 * np + 1], g.W, 2, wdims, wstr, wbox));
    } else {
      SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm[3 * np], (const bf16*)g.A + g.a_map.offset, 3, adims, astr, abox));
      SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm[3 * np + 1], g.W, 2, wdims, wstr, wbox));
    }
    const uint64_t odims[3] = {(uint64_t)g.N, (uint64_t)rps, (uint64_t)nseq};
    if (epi == EPI_GATE_RES) {
      const RowMap& m = g.resid_map;
      const uint64_t ostr[2] = {(uint64_t)m.ld * 4, (uint64_t)(nseq > 1 ? m.seq_stride : m.ld * (long long)rps) * 4};
      const uint32_t obox[3] = {32, 32, 1};
      SPOT_CUDA_TRY(spot_make_tmap_f32(&tm[3 * np + 2], g.resid + m.offset, 3, odims, ostr, obox));
    } else if (out8) {
      const RowMap& m = g.out_map;
      const uint64_t ostr[2] = {(uint64_t)m.ld, (uint64_t)(nseq > 1 ? m.seq_stride : m.ld * (long long)rps)};
      const uint32_t obox[3] = {128, 32, 1};
      SPOT_CUDA_TRY(spot_make_tmap_u8(&tm[3 * np + 2], (uint8_t*)g.out + m.offset, 3, odims, ostr, obox));
    } else {
      const RowMap& m = g.out_map;
      const uint64_t ostr[2] = {(uint64_t)m.ld * 2, (uint64_t)(nseq > 1 ? m.seq_stride : m.ld * (long long)rps) * 2};
      const uint32_t obox[3] = {64, 32, 1};
      SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm[3 * np + 2], (bf16*)g.out + m.offset, 3, odims, ostr, obox));
    }
    ++np;
  }
  if (np == 0) return cudaSuccess;
  if (np == 1) { tm[3] = tm[0]; tm[4] = tm[1]; tm[5] = tm[2]; }
  P.n_probs = np;
  P.total_tiles = tiles;
  int pairs = num_sms / 2;
  if (tiles < pairs) pairs = tiles;
  const int grid = 2 * pairs;
#define V3_LAUNCH(E, F)                                                                                              \
  do {                                                                                                               \
    static bool attr_set = false;                                                                                    \
    if (!attr_set) {                                                                                                 \
      SPOT_CUDA_TRY(cudaFuncSetAttribute(gemm_tcgen05_v3_kernel<E, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                         (int)SMEM_BYTES));                                                          \
      attr_set = true;                                                                                               \
    }                                                                                                                \
    gemm_tcgen05_v3_kernel<E, F><<<grid, 128 + epi_warps(E, F) * 32, SMEM_BYTES, st>>>(tm[0], tm[1], tm[2], tm[3], tm[4], tm[5], P); \
  } while (0)
#define V3_LAUNCH2(E)              \
  do {                             \
    if (fp8) V3_LAUNCH(E, true);   \
    else V3_LAUNCH(E, false);      \
  } while (0)
  switch (epi) {
    case EPI_BIAS: V3_LAUNCH2(EPI_BIAS); break;
    case EPI_BIAS_GELU: V3_LAUNCH2(EPI_BIAS_GELU); break;
    case EPI_GATE_RES: V3_LAUNCH2(EPI_GATE_RES); break;
    case EPI_QKV_ROPE: V3_LAUNCH2(EPI_QKV_ROPE); break;
  }
#undef V3_LAUNCH2
#undef V3_LAUNCH
  return cudaGetLastError();
}
