// smlm_debug_fill (include/smlm.h): a write-only bandwidth yardstick for bench.py.  K1 (stem.cu)
// is a write stream - 2 B/px in, 2C B/px out - so the roof it is held against is how fast this
// GPU takes plain 16-byte stores, measured in the same run: with cudaMemsetAsync and with a
// kernel of our own (one st.global.v4 per thread and step, grid-stride, 148 x 8 CTAs).
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/smlm.h"

namespace {

__global__ void __launch_bounds__(256) fill_v4_kernel(uint4* __restrict__ dst, size_t n16, uint4 v) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) dst[i] = v;
}

}  // namespace

extern "C" smlm_status smlm_debug_fill(void* dst, int64_t bytes, int32_t mode, void* cuda_stream) {
  if (!dst || bytes < 0 || (bytes & 15) || (reinterpret_cast<uintptr_t>(dst) & 15) || mode < 0 || mode > 1)
    return SMLM_ERR_INVALID_ARG;
  if (bytes == 0) return SMLM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (mode == 0) return cudaMemsetAsync(dst, 0x5a, (size_t)bytes, st) == cudaSuccess ? SMLM_OK : SMLM_ERR_CUDA;
  int dev = 0, n_sm = 148;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return SMLM_ERR_CUDA;
  const uint4 v = make_uint4(0x5a5a5a5au, 0x5a5a5a5au, 0x5a5a5a5au, 0x5a5a5a5au);
  fill_v4_kernel<<<n_sm * 8, 256, 0, st>>>(static_cast<uint4*>(dst), (size_t)bytes / 16, v);
  return cudaGetLastError() == cudaSuccess ? SMLM_OK : SMLM_ERR_CUDA;
}
