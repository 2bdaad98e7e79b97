// noise.cu - K1: seed -> Philox4x32-10 -> Box-Muller -> N(0,1) latents.
//
// PAPER.md:59 "starts from random Gaussian noise"; :61 "K distinct noise seeds"; :251 "we assign each
// sample a deterministic random seed".  Layout = DESIGN.md S1-S3: key = (lo32, hi32)(seed), counter =
// (lo32(j), hi32(j), stream_id, 0) for the 4-element block j; 24-bit uniforms u1 in (0,1], u2 in [0,1).
//
// One thread makes one Philox block = 4 normals = one 16-byte store; a warp writes 512 contiguous
// bytes.  Write-bandwidth bound (4 B/element algorithmic).
#include "kernels.h"
#include "philox.cuh"

namespace {

// grid.y = sequence (no 64-bit division per element), grid.x strides over the sequence's Philox blocks
template <bool WORDS>
__global__ void __launch_bounds__(256) noise_kernel(const uint64_t* __restrict__ seeds, long long blocks_per_seed,
                                                    uint32_t stream_id, float4* __restrict__ out, uint4* __restrict__ words) {
  const int b = blockIdx.y;
  const uint64_t seed = seeds[b];
  const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
  const long long base = (long long)b * blocks_per_seed;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < blocks_per_seed; j += stride) {
    const uint4 w = philox4x32_10(make_uint4((uint32_t)j, (uint32_t)((unsigned long long)j >> 32), stream_id, 0u), key);
    if (WORDS) {
      words[base + j] = w;
    } else {
      const float2 a = box_muller(w.x, w.y), c = box_muller(w.z, w.w);
      out[base + j] = make_float4(a.x, a.y, c.x, c.y);
    }
  }
}

}  // namespace

cudaError_t launch_noise(const uint64_t* d_seeds, int n_seeds, long long elems_per_seed, uint32_t stream_id,
                         float* d_normals, uint32_t* d_words, cudaStream_t st) {
  const long long bps = elems_per_seed / 4;
  if (bps == 0 || n_seeds <= 0) return cudaSuccess;
  if (n_seeds > 65535) return cudaErrorInvalidValue;
  long long want = (bps + 255) / 256;
  const long long cap = (148LL * 32 + n_seeds - 1) / n_seeds;      // ~32 blocks per SM over the whole grid
  if (want > cap) want = cap < 1 ? 1 : cap;
  const dim3 grid((unsigned)want, (unsigned)n_seeds);
  if (d_words)
    noise_kernel<true><<<grid, 256, 0, st>>>(d_seeds, bps, stream_id, nullptr, (uint4*)d_words);
  else
    noise_kernel<false><<<grid, 256, 0, st>>>(d_seeds, bps, stream_id, (float4*)d_normals, nullptr);
  return cudaGetLastError();
}
