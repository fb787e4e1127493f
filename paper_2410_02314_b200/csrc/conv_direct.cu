// K2': one trunk layer on CUDA cores,  out = in + ReLU(conv3x3_dilated(in; W) + b)
// (smlm.h; zero padding = dilation at the window border).  fp32 math; storage float (the
// fp32 reference mode of BASELINE.json north_star (b)) or bf16 (cross-check of the tcgen05
// kernel with the same rounding points: bf16 inputs, bf16-valued weights, fp32 accumulate,
// one RNE rounding of the stored result).  A correctness mode, not the timed path.
//
// thread = (pixel, output chunk of 8 channels); the block walks ROWS rows of a 64-pixel
// strip with the whole layer's weights [9][C][C] resident in shared memory.
#include "chunk_io.cuh"
#include "smlm_internal.cuh"

namespace smlm {
namespace {

constexpr int PX = 64, ROWS = 16;

template <typename T, int C>
__global__ void __launch_bounds__(PX*(C / 8))
    conv_direct_kernel(const T* __restrict__ in, T* __restrict__ out, ActShape s, int dil,
                       const float* __restrict__ w /*[9][C][C] (tap, ci, co)*/,
                       const float* __restrict__ bias) {
  extern __shared__ __align__(16) float wsm[];  // [9][C][C]
  const int tid = threadIdx.y * PX + threadIdx.x, nthr = PX * (C / 8);
  for (int i = tid; i < 9 * C * C / 4; i += nthr)
    reinterpret_cast<float4*>(wsm)[i] = reinterpret_cast<const float4*>(w)[i];
  __syncthreads();

  const int b = blockIdx.z, kc = threadIdx.y;
  const int x = blockIdx.x * PX + threadIdx.x;
  if (x >= s.W) return;
  float bv[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) bv[c] = bias[kc * 8 + c];

  const int yend = min(s.H, (int)(blockIdx.y + 1) * ROWS);
  for (int y = blockIdx.y * ROWS; y < yend; ++y) {
    float acc[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] = bv[c];
    for (int ky = 0; ky < 3; ++ky) {
      const int yy = y + (ky - 1) * dil;
      if (yy < 0 || yy >= s.H) continue;
      for (int kx = 0; kx < 3; ++kx) {
        const int xx = x + (kx - 1) * dil;
        if (xx < 0 || xx >= s.W) continue;
        const float* wt = wsm + (ky * 3 + kx) * C * C + kc * 8;
#pragma unroll 2
        for (int ki = 0; ki < C / 8; ++ki) {
          float v[8];
          Chunk<T>::load(in, s.chunk_index(b, ki, yy, xx), v);
#pragma unroll
          for (int ci = 0; ci < 8; ++ci) {
            const float4 w0 = *reinterpret_cast<const float4*>(wt + (ki * 8 + ci) * C);
            const float4 w1 = *reinterpret_cast<const float4*>(wt + (ki * 8 + ci) * C + 4);
            acc[0] = fmaf(v[ci], w0.x, acc[0]);
            acc[1] = fmaf(v[ci], w0.y, acc[1]);
            acc[2] = fmaf(v[ci], w0.z, acc[2]);
            acc[3] = fmaf(v[ci], w0.w, acc[3]);
            acc[4] = fmaf(v[ci], w1.x, acc[4]);
            acc[5] = fmaf(v[ci], w1.y, acc[5]);
            acc[6] = fmaf(v[ci], w1.z, acc[6]);
            acc[7] = fmaf(v[ci], w1.w, acc[7]);
          }
        }
      }
    }
    float r[8];
    const size_t q = s.chunk_index(b, kc, y, x);
    Chunk<T>::load(in, q, r);
#pragma unroll
    for (int c = 0; c < 8; ++c) r[c] += fmaxf(acc[c], 0.0f);
    Chunk<T>::store(out, q, r);
  }
}

template <typename T, int C>
cudaError_t launch_tc(const void* in, void* out, ActShape s, int dil, const float* w,
                      const float* b, cudaStream_t st) {
  dim3 grid((s.W + PX - 1) / PX, (s.H + ROWS - 1) / ROWS, s.B), block(PX, C / 8);
  size_t smem = (size_t)9 * C * C * sizeof(float);
  conv_direct_kernel<T, C><<<grid, block, smem, st>>>((const T*)in, (T*)out, s, dil, w, b);
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_t(const void* in, void* out, ActShape s, int dil, const float* w,
                     const float* b, cudaStream_t st) {
  switch (s.C) {
    case 16: return launch_tc<T, 16>(in, out, s, dil, w, b, st);
    case 32: return launch_tc<T, 32>(in, out, s, dil, w, b, st);
    case 48: return launch_tc<T, 48>(in, out, s, dil, w, b, st);
    case 64: return launch_tc<T, 64>(in, out, s, dil, w, b, st);
    default: return cudaErrorInvalidValue;
  }
}

template <typename T, int C>
cudaError_t init_tc() {
  return cudaFuncSetAttribute(conv_direct_kernel<T, C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              9 * C * C * (int)sizeof(float));
}

}  // namespace

cudaError_t conv_direct_init(int C) {
  cudaError_t e;
  switch (C) {
#define INIT3(CC)                                                     \
  e = init_tc<float, CC>();                                           \
  if (e == cudaSuccess) e = init_tc<__nv_bfloat16, CC>();             \
  if (e == cudaSuccess) e = init_tc<__half, CC>();                    \
  break;
    case 16: INIT3(16)
    case 32: INIT3(32)
    case 48: INIT3(48)
    case 64: INIT3(64)
#undef INIT3
    default: e = cudaErrorInvalidValue;
  }
  return e;
}

cudaError_t launch_conv_direct(int dt, const void* in, void* out, ActShape s, int dil,
                               const float* w, const float* b, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  if (dt == ACT_BF16) return launch_t<__nv_bfloat16>(in, out, s, dil, w, b, st);
  if (dt == ACT_F16) return launch_t<__half>(in, out, s, dil, w, b, st);
  return launch_t<float>(in, out, s, dil, w, b, st);
}

}  // namespace smlm
