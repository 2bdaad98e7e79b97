// attn_tcgen05.cu - K5 placeholder until the tcgen05 flash attention lands: reports "unsupported" so
// every caller takes the SIMT attention kernel.
#include "kernels.h"
bool tcgen05_attn_supported(int, int, int) { return false; }
cudaError_t launch_attn_tcgen05(const void*, void*, int, int, int, int, int, cudaStream_t) { return cudaErrorNotSupported; }
