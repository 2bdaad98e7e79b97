// gemm_tcgen05.cu - K2: persistent, warp-specialised bf16 GEMM C = epi(A W^T + bias) on the 5th-gen
// tensor cores (north_star (b): "tcgen05/TMEM GEMMs fed by TMA ... with fused epilogues").
//
//   warp 0      TMA producer: A tile [128 x 64] (3-D map: K, row-in-sequence, sequence) and W tile
//               [256 x 64], both K-major with 128-byte swizzle, into a 4-stage shared-memory ring
//   warp 1      MMA issuer: one thread issues 4 x tcgen05.mma (M128 N256 K16) per stage into one of two
//               256-column TMEM accumulators, tcgen05.commit frees the stage / publishes the tile
//   warp 2      TMEM allocator (512 columns)
//   warps 4-7   epilogue: tcgen05.ld 32 lanes x 32 columns, + bias, then
//                 EPI_BIAS       -> bf16 store                       (QKV projection)
//                 EPI_BIAS_GELU  -> tanh-GELU -> bf16 store          (fc1)
//                 EPI_GATE_RES   -> h += gate * y on the fp32 residual stream (out-proj, fc2)
//               while the MMA warp already fills the other accumulator (epilogue/mainloop overlap).
// Grid = min(#SMs, #tiles), static round-robin over a GROUP_M-swizzled tile order so that one wave
// touches ~16 M-tiles x ~9 N-tiles (keeps A and W panels L2-resident).  Up to two problems (image
// and text streams, which have separate weights) are served by one launch.
#include "kernels.h"
#include "tcgen05.cuh"
#include <string.h>

namespace {

constexpr int BLOCK_M = 128, BLOCK_N = 256, BLOCK_K = 64, UMMA_K = 16, STAGES = 4, GROUP_M = 16;
constexpr uint32_t A_BYTES = BLOCK_M * BLOCK_K * 2, B_BYTES = BLOCK_N * BLOCK_K * 2, STAGE_BYTES = A_BYTES + B_BYTES;
constexpr uint32_t SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
constexpr int NUM_THREADS = 256;

struct TcProblem {
  int m_tiles, n_tiles, tiles_per_seq, rps, N, k_blocks, tile_start;
  const bf16* bias;
  bf16* out;
  long long o_seq, o_off, o_ld;
  const float* gate;
  float* resid;
  long long r_seq, r_off, r_ld;
};
struct TcParams {
  TcProblem p[2];
  int n_probs, total_tiles;
};

struct TileCoord { int prob, mt, nt; };

__device__ __forceinline__ TileCoord decode_tile(const TcParams& P, int t) {
  TileCoord c;
  c.prob = (P.n_probs > 1 && t >= P.p[1].tile_start) ? 1 : 0;
  const TcProblem& q = P.p[c.prob];
  t -= q.tile_start;
  const int per_group = GROUP_M * q.n_tiles;
  const int g = t / per_group, first_m = g * GROUP_M;
  const int gm = min(GROUP_M, q.m_tiles - first_m);
  const int r = t - g * per_group;
  c.mt = first_m + r % gm;
  c.nt = r / gm;
  return c;
}

template <int EPI>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ CUtensorMap tmA0, const __grid_constant__ CUtensorMap tmW0,
                    const __grid_constant__ CUtensorMap tmA1, const __grid_constant__ CUtensorMap tmW1,
                    const TcParams P) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
  volatile uint32_t* tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmA0); ptx::prefetch_tmap(&tmW0);
    if (P.n_probs > 1) { ptx::prefetch_tmap(&tmA1); ptx::prefetch_tmap(&tmW1); }
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), 4); }
    ptx::fence_barrier_init();
  }
  if (warp == 2) { ptx::tmem_alloc(tmem_slot, 512); ptx::tmem_relinquish(); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int t = blockIdx.x; t < P.total_tiles; t += gridDim.x) {
        const TileCoord c = decode_tile(P, t);
        const TcProblem& q = P.p[c.prob];
        const CUtensorMap* mA = c.prob ? &tmA1 : &tmA0;
        const CUtensorMap* mW = c.prob ? &tmW1 : &tmW0;
        const int seq = c.mt / q.tiles_per_seq, r0 = (c.mt - seq * q.tiles_per_seq) * BLOCK_M;
        for (int kb = 0; kb < q.k_blocks; ++kb) {
          ptx::mbar_wait(empty_bar(stage), phase ^ 1);
          ptx::mbar_arrive_expect_tx(full_bar(stage), STAGE_BYTES);
          const uint32_t sa = smem_base + stage * STAGE_BYTES;
          ptx::tma_load_3d(sa, mA, full_bar(stage), kb * BLOCK_K, r0, seq);
          ptx::tma_load_2d(sa + A_BYTES, mW, full_bar(stage), kb * BLOCK_K, c.nt * BLOCK_N);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_bf16(BLOCK_M, BLOCK_N, 0, 0);
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t acc_phase = 0;
      for (int t = blockIdx.x; t < P.total_tiles; t += gridDim.x) {
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
            ptx::mma_f16_ss(d_tmem, da, db, idesc, (kb | k) ? 1u : 0u);
          }
          ptx::mma_commit(empty_bar(stage));
          if (kb == k_blocks - 1) ptx::mma_commit(tfull_bar(acc));
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue =====================
    const int q4 = warp & 3;                      // TMEM lane quarter this warp may access
    int acc = 0; uint32_t acc_phase = 0;
    for (int t = blockIdx.x; t < P.total_tiles; t += gridDim.x) {
      const TileCoord c = decode_tile(P, t);
      const TcProblem& q = P.p[c.prob];
      const int seq = c.mt / q.tiles_per_seq, r = (c.mt - seq * q.tiles_per_seq) * BLOCK_M + q4 * 32 + lane;
      const bool row_ok = r < q.rps;
      ptx::mbar_wait(tfull_bar(acc), acc_phase);
      ptx::tc_fence_after();
      const uint32_t taddr0 = tmem_base + acc * BLOCK_N + ((uint32_t)(q4 * 32) << 16);
#pragma unroll 1
      for (int ch = 0; ch < BLOCK_N / 32; ++ch) {
        const int n0 = c.nt * BLOCK_N + ch * 32;
        if (n0 >= q.N) break;                      // warp-uniform
        uint32_t v[32];
        ptx::tmem_ld_32x32(taddr0 + ch * 32, v);
        ptx::tmem_ld_wait();
        float y[32];
        const uint4* bp = reinterpret_cast<const uint4*>(q.bias + n0);
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          uint4 braw = __ldg(bp + g);
          const bf16* bb = reinterpret_cast<const bf16*>(&braw);
#pragma unroll
          for (int j = 0; j < 8; ++j) y[g * 8 + j] = __uint_as_float(v[g * 8 + j]) + __bfloat162float(bb[j]);
        }
        if (EPI == EPI_BIAS_GELU) {
#pragma unroll
          for (int j = 0; j < 32; ++j) y[j] = gelu_tanh_f(y[j]);
        }
        if (EPI == EPI_GATE_RES) {
          if (row_ok) {
            float4* rp = reinterpret_cast<float4*>(q.resid + (long long)seq * q.r_seq + q.r_off + (long long)r * q.r_ld + n0);
            const float4* gp = reinterpret_cast<const float4*>(q.gate + n0);
#pragma unroll
            for (int g = 0; g < 8; ++g) {
              float4 h = rp[g];
              const float4 gt = __ldg(gp + g);
              h.x = fmaf(gt.x, y[4 * g], h.x); h.y = fmaf(gt.y, y[4 * g + 1], h.y);
              h.z = fmaf(gt.z, y[4 * g + 2], h.z); h.w = fmaf(gt.w, y[4 * g + 3], h.w);
              rp[g] = h;
            }
          }
        } else {
          if (row_ok) {
            uint4* op = reinterpret_cast<uint4*>(q.out + (long long)seq * q.o_seq + q.o_off + (long long)r * q.o_ld + n0);
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              uint4 pk;
              __nv_bfloat162 p0 = __floats2bfloat162_rn(y[8 * g], y[8 * g + 1]);
              __nv_bfloat162 p1 = __floats2bfloat162_rn(y[8 * g + 2], y[8 * g + 3]);
              __nv_bfloat162 p2 = __floats2bfloat162_rn(y[8 * g + 4], y[8 * g + 5]);
              __nv_bfloat162 p3 = __floats2bfloat162_rn(y[8 * g + 6], y[8 * g + 7]);
              pk.x = *reinterpret_cast<uint32_t*>(&p0); pk.y = *reinterpret_cast<uint32_t*>(&p1);
              pk.z = *reinterpret_cast<uint32_t*>(&p2); pk.w = *reinterpret_cast<uint32_t*>(&p3);
              op[g] = pk;
            }
          }
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(tempty_bar(acc));
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) { ptx::tc_fence_after(); ptx::tmem_dealloc(tmem_base, 512); }
}

}  // namespace

// ================================================================================================
// host side
spot_encode_tiled_fn spot_get_encode_tiled() {
  static spot_encode_tiled_fn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<spot_encode_tiled_fn>(p);
  }
  return fn;
}

static cudaError_t make_tmap(CUtensorMap* out, CUtensorMapDataType dt, const void* base, int rank, const uint64_t* dims,
                             const uint64_t* strides_bytes, const uint32_t* box, bool swizzle = true) {
  spot_encode_tiled_fn enc = spot_get_encode_tiled();
  if (!enc) return cudaErrorNotSupported;
  cuuint64_t gdim[5], gstr[5];
  cuuint32_t bx[5], es[5];
  for (int i = 0; i < rank; ++i) { gdim[i] = dims[i]; bx[i] = box[i]; es[i] = 1; }
  for (int i = 0; i + 1 < rank; ++i) gstr[i] = strides_bytes[i];
  CUresult r = enc(out, dt, (cuuint32_t)rank, const_cast<void*>(base), gdim, gstr, bx, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t spot_make_tmap_bf16(CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                                const uint64_t* strides_bytes, const uint32_t* box) {
  return make_tmap(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, base, rank, dims, strides_bytes, box);
}

cudaError_t spot_make_tmap_u8(CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                              const uint64_t* strides_bytes, const uint32_t* box) {
  return make_tmap(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, base, rank, dims, strides_bytes, box);
}

cudaError_t spot_make_tmap_u8_linear(CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                                     const uint64_t* strides_bytes, const uint32_t* box) {
  return make_tmap(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, base, rank, dims, strides_bytes, box, false);
}

cudaError_t spot_make_tmap_f32(CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                               const uint64_t* strides_bytes, const uint32_t* box) {
  return make_tmap(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, base, rank, dims, strides_bytes, box);
}

bool tcgen05_gemm_supported(const GemmProblem& p) {
  if (p.M <= 0 || p.N <= 0 || p.K <= 0) return false;
  const int es = p.fp8 ? 1 : 2;                     // bytes per operand element
  if ((p.K * es) % 16 || p.N % 32) return false;
  if (p.fp8 && (!p.w_scale || reinterpret_cast<uintptr_t>(p.w_scale) % 16)) return false;
  const RowMap& a = p.a_map;
  if (a.rows_per_seq <= 0 || p.M % a.rows_per_seq) return false;
  if ((a.ld * es) % 16 || (a.offset * es) % 16 || (a.seq_stride * es) % 16) return false;
  if (reinterpret_cast<uintptr_t>(p.A) % 16 || reinterpret_cast<uintptr_t>(p.W) % 16) return false;
  if (p.out && (p.out_map.rows_per_seq != a.rows_per_seq || p.out_map.ld % 16 || p.out_map.offset % 16 ||
                p.out_map.seq_stride % 16 || reinterpret_cast<uintptr_t>(p.out) % 16))
    return false;
  if (p.resid && (p.resid_map.rows_per_seq != a.rows_per_seq || p.resid_map.ld % 4 || p.resid_map.offset % 4 ||
                  p.resid_map.seq_stride % 4 || reinterpret_cast<uintptr_t>(p.resid) % 16))
    return false;
  if (!p.bias || reinterpret_cast<uintptr_t>(p.bias) % 16) return false;
  return spot_get_encode_tiled() != nullptr;
}

cudaError_t launch_gemm_tcgen05(Epilogue epi, const GemmProblem* probs, int n_probs, int num_sms, cudaStream_t st) {
  if (n_probs < 1 || n_probs > 2) return cudaErrorInvalidValue;
  TcParams P;
  memset(&P, 0, sizeof(P));
  CUtensorMap tm[4];
  memset(tm, 0, sizeof(tm));
  int tiles = 0, np = 0;
  for (int i = 0; i < n_probs; ++i) {
    const GemmProblem& g = probs[i];
    if (g.M <= 0) continue;
    if (!tcgen05_gemm_supported(g)) return cudaErrorInvalidValue;
    if ((epi == EPI_GATE_RES) != (g.resid != nullptr)) return cudaErrorInvalidValue;
    TcProblem& q = P.p[np];
    const int rps = g.a_map.rows_per_seq, nseq = g.M / rps;
    q.rps = rps;
    q.tiles_per_seq = (rps + BLOCK_M - 1) / BLOCK_M;
    q.m_tiles = nseq * q.tiles_per_seq;
    q.n_tiles = (g.N + BLOCK_N - 1) / BLOCK_N;
    q.N = g.N;
    q.k_blocks = (g.K + BLOCK_K - 1) / BLOCK_K;
    q.tile_start = tiles;
    q.bias = (const bf16*)g.bias;
    q.out = (bf16*)g.out;
    q.o_seq = g.out_map.seq_stride; q.o_off = g.out_map.offset; q.o_ld = g.out_map.ld;
    q.gate = g.gate;
    q.resid = g.resid;
    q.r_seq = g.resid_map.seq_stride; q.r_off = g.resid_map.offset; q.r_ld = g.resid_map.ld;
    tiles += q.m_tiles * q.n_tiles;
    const uint64_t adims[3] = {(uint64_t)g.K, (uint64_t)rps, (uint64_t)nseq};
    const uint64_t astr[2] = {(uint64_t)g.a_map.ld * 2,
                              (uint64_t)(nseq > 1 ? g.a_map.seq_stride : g.a_map.ld * (long long)rps) * 2};
    const uint32_t abox[3] = {BLOCK_K, BLOCK_M, 1};
    SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm[2 * np], (const bf16*)g.A + g.a_map.offset, 3, adims, astr, abox));
    const uint64_t wdims[2] = {(uint64_t)g.K, (uint64_t)g.N};
    const uint64_t wstr[1] = {(uint64_t)g.K * 2};
    const uint32_t wbox[2] = {BLOCK_K, BLOCK_N};
    SPOT_CUDA_TRY(spot_make_tmap_bf16(&tm[2 * np + 1], g.W, 2, wdims, wstr, wbox));
    ++np;
  }
  if (np == 0) return cudaSuccess;
  if (np == 1) { tm[2] = tm[0]; tm[3] = tm[1]; }
  P.n_probs = np;
  P.total_tiles = tiles;
  const int grid = tiles < num_sms ? tiles : num_sms;
#define TC_LAUNCH(E)                                                                                             \
  do {                                                                                                           \
    static bool attr_set = false;                                                                                \
    if (!attr_set) {                                                                                             \
      SPOT_CUDA_TRY(cudaFuncSetAttribute(gemm_tcgen05_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                                         (int)SMEM_BYTES));                                                      \
      attr_set = true;                                                                                           \
    }                                                                                                            \
    gemm_tcgen05_kernel<E><<<grid, NUM_THREADS, SMEM_BYTES, st>>>(tm[0], tm[1], tm[2], tm[3], P);                \
  } while (0)
  switch (epi) {
    case EPI_BIAS: TC_LAUNCH(EPI_BIAS); break;
    case EPI_BIAS_GELU: TC_LAUNCH(EPI_BIAS_GELU); break;
    case EPI_GATE_RES: TC_LAUNCH(EPI_GATE_RES); break;
  }
#undef TC_LAUNCH
  return cudaGetLastError();
}
