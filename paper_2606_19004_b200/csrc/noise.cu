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

template <bool WORDS>
__global__ void __launch_bounds__(256) noise_kernel(const uint64_t* __restrict__ seeds, long long blocks_per_seed,
                                                    long long total_blocks, uint32_t stream_id,
                                                    float4* __restrict__ out, uint4* __restrict__ words) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < total_blocks; i += stride) {
    long long b = i / blocks_per_seed;
    unsigned long long j = (unsigned long long)(i - b * blocks_per_seed);
    uint64_t seed = seeds[b];
    uint4 w = philox4x32_10(make_uint4((uint32_t)j, (uint32_t)(j >> 32), stream_id, 0u),
                            make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
    if (WORDS) {
      words[i] = w;
    } else {
      float2 a = box_muller(w.x, w.y), c = box_muller(w.z, w.w);
      out[i] = make_float4(a.x, a.y, c.x, c.y);
    }
  }
}

}  // namespace

cudaError_t launch_noise(const uint64_t* d_seeds, int n_seeds, long long elems_per_seed, uint32_t stream_id,
                         float* d_normals, uint32_t* d_words, cudaStream_t st) {
  long long bps = elems_per_seed / 4, total = bps * n_seeds;
  if (total == 0) return cudaSuccess;
  long long want = (total + 255) / 256;
  int grid = (int)(want < 148LL * 32 ? want : 148LL * 32);   // grid-stride: a multiple of the SM count when large
  if (d_words)
    noise_kernel<true><<<grid, 256, 0, st>>>(d_seeds, bps, total, stream_id, nullptr, (uint4*)d_words);
  else
    noise_kernel<false><<<grid, 256, 0, st>>>(d_seeds, bps, total, stream_id, (float4*)d_normals, nullptr);
  return cudaGetLastError();
}
