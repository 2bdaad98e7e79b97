// attn_simt.cu - K9: plain fp32 joint attention O = softmax(Q K^T / sqrt(d_h)) V, all S keys, no mask
// (S4 step 6, S6).  One warp per (sequence, head, query row); keys are streamed with an
// online softmax in fp32.  Used by the fp32 config and as the on-GPU cross-check of the tcgen05
// attention kernel; not a throughput path.
#include "kernels.h"

namespace {

template <typename T, int DH>
__global__ void __launch_bounds__(256) attn_simt_kernel(const T* __restrict__ qkv, T* __restrict__ out,
                                                        long long n_rows, int S, int H) {
  constexpr int EPL = DH / 32;
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= n_rows) return;
  const int lane = threadIdx.x & 31;
  // row index w = ((b * H) + h) * S + s : consecutive warps share (b, h) so K/V rows stay L1/L2 hot
  const int s = (int)(w % S);
  const long long bh = w / S;
  const int h = (int)(bh % H);
  const long long b = bh / H;
  const long long tok_stride = 3LL * H * DH;
  const T* base = qkv + b * S * tok_stride + (long long)h * DH + lane * EPL;
  float q[EPL], o[EPL];
  const float scale = rsqrtf((float)DH);
#pragma unroll
  for (int j = 0; j < EPL; ++j) { q[j] = to_f32(base[s * tok_stride + j]) * scale; o[j] = 0.f; }
  float m = -INFINITY, l = 0.f;
  for (int key = 0; key < S; ++key) {
    const T* kp = base + key * tok_stride + (long long)H * DH;
    const T* vp = kp + (long long)H * DH;
    float d = 0.f;
#pragma unroll
    for (int j = 0; j < EPL; ++j) d = fmaf(q[j], to_f32(kp[j]), d);
    d = warp_sum(d);
    const float m_new = fmaxf(m, d);
    const float alpha = expf(m - m_new), pexp = expf(d - m_new);
    l = l * alpha + pexp;
#pragma unroll
    for (int j = 0; j < EPL; ++j) o[j] = o[j] * alpha + pexp * to_f32(vp[j]);
    m = m_new;
  }
  T* op = out + (b * S + s) * (long long)(H * DH) + (long long)h * DH + lane * EPL;
  const float inv = 1.f / l;
#pragma unroll
  for (int j = 0; j < EPL; ++j) op[j] = from_f32<T>(o[j] * inv);
}

}  // namespace

cudaError_t launch_attn_simt(spot_dtype dt, const void* qkv, void* out, int B, int S, int H, int dh, cudaStream_t st) {
  const long long n = (long long)B * H * S;
  if (n <= 0) return cudaSuccess;
  const long long blocks = (n + 7) / 8;
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
#define ATT_CASE(T, DH) attn_simt_kernel<T, DH><<<(int)blocks, 256, 0, st>>>((const T*)qkv, (T*)out, n, S, H)
  if (dt == SPOT_F32 && dh == 64) ATT_CASE(float, 64);
  else if (dt == SPOT_F32 && dh == 128) ATT_CASE(float, 128);
  else if (dt == SPOT_BF16 && dh == 64) ATT_CASE(bf16, 64);
  else if (dt == SPOT_BF16 && dh == 128) ATT_CASE(bf16, 128);
  else return cudaErrorInvalidValue;
#undef ATT_CASE
  return cudaGetLastError();
}
