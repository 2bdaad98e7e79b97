// euler_static.cu - spot_euler_update_static: the Euler update + probe reward (K6; S8-S9) for
// callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  The kernels are the ones spot_euler_update launches; only the scratch for the reward's partial sums differs:
// it is a file-scope __device__ array of SPOT_STATIC_PARTIALS_MAX floats (256 KiB), held by every GPU that loads this
// library until the process exits, instead of a buffer the caller passes.
//
// In host code the array's NAME is a host-side stand-in, not a device address, so the address the kernels get is taken
// with cudaGetSymbolAddress, once per device, with that device current (first call on the device = set-up; it must not
// happen under stream capture, every later call is capture-safe).  No cudaMalloc / cudaFree / allocating library routine.
// Every call on a device shares the array: calls that overlap on the GPU (different streams) race on it.  Nothing in it has
// to start at zero - each (sequence, chunk) slot is overwritten by the block that owns it before reward_finalize reads it.
#include <mutex>

#include "../../include/spot_kernels.h"
#include "kernels.h"

namespace {

constexpr int kMaxDevices = 64;
static __device__ __align__(256) float g_static_partials[SPOT_STATIC_PARTIALS_MAX];

// device address of g_static_partials on the CURRENT device; set up (and the device's architecture checked) on first use
spot_status static_partials(float** out) {
  static std::mutex mu;
  static float* addr[kMaxDevices] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return SPOT_ERR_ARCH; }
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) {
      cudaGetLastError();
      return SPOT_ERR_ARCH;
    }
    float* p = nullptr;
    if (cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_partials) != cudaSuccess || !p) {
      cudaGetLastError();
      return SPOT_ERR_CUDA;
    }
    addr[dev] = p;
  }
  *out = addr[dev];
  return SPOT_OK;
}

}  // namespace

extern "C" spot_status spot_euler_update_static(float* d_x, const float* d_v, float dt, int n_seqs, int64_t elems,
                                                const float* d_probe, float* d_rewards, void* cuda_stream) {
  if (n_seqs < 0 || n_seqs > 65535 || elems <= 0 || (elems & 3)) return SPOT_ERR_SHAPE;   // sequences ride on gridDim.y
  if (n_seqs == 0) return SPOT_OK;
  if (!d_x || !d_v || !d_probe || !d_rewards) return SPOT_ERR_NULL;
  if ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_v) | reinterpret_cast<uintptr_t>(d_probe)) & 15) return SPOT_ERR_ALIGN;
  const int64_t n_chunks = (elems + REWARD_CHUNK - 1) / REWARD_CHUNK;
  if (n_chunks * (int64_t)n_seqs > (int64_t)SPOT_STATIC_PARTIALS_MAX) return SPOT_ERR_WORKSPACE;   // beyond the static scratch
  float* partials = nullptr;
  const spot_status ss = static_partials(&partials);
  if (ss != SPOT_OK) return ss;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (launch_euler_update(d_x, d_v, dt, n_seqs, elems, d_probe, partials, st) != cudaSuccess) return SPOT_ERR_CUDA;
  if (launch_reward_finalize(partials, n_seqs, elems, d_rewards, st) != cudaSuccess) return SPOT_ERR_CUDA;
  return SPOT_OK;
}
