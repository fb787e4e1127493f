// K1: uint16 unpack + offset/gain normalisation + 3x3 stem convolution (1 -> C) (+ReLU),
// fused (BASELINE.json north_star (a); smlm.h: xhat = ((adu - offset)/gain)/norm_scale,
// a0 = act(conv3x3(xhat; W0) + b0), zero padding 1 at the FRAME border).
//
// HBM-bound: 2 B/px in, 2C B/px out (bf16).  One thread = one pixel, all C channels; a warp
// covers 32 consecutive pixels of a row, so each of its C/8 stores is one dense 512 B run
// in the chunk-planar layout.  The normalised (TY+2) x (TX+2) input patch is staged in
// shared memory once per block (the divisions happen once per pixel, not once per tap).
#include "chunk_io.cuh"
#include "smlm_internal.cuh"

namespace smlm {
namespace {

constexpr int TX = 64, TY = 4;

template <typename T, int C>
__global__ void __launch_bounds__(TX* TY)
    stem_kernel(const uint16_t* __restrict__ frames, int frame_base, ViewSet vs, ActShape s,
                NormParams np, const float* __restrict__ w /*[9][C]*/,
                const float* __restrict__ bias, int relu, T* __restrict__ act) {
  __shared__ float xs[TY + 2][TX + 2];
  __shared__ __align__(16) float ws[9][C];
  __shared__ __align__(16) float bs[C];

  const int b = blockIdx.z;
  const View v = view_of(vs, b, s.H, s.W);
  const int tid = threadIdx.y * TX + threadIdx.x;
  for (int i = tid; i < 9 * C; i += TX * TY) ws[i / C][i % C] = w[i];
  for (int i = tid; i < C; i += TX * TY) bs[i] = bias[i];

  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const uint16_t* frame = frames + (size_t)(v.frame - frame_base) * vs.Hf * vs.Wf;
  const float inv_scalar = 1.0f / (np.gain * np.norm_scale);
  for (int i = tid; i < (TY + 2) * (TX + 2); i += TX * TY) {
    int ly = i / (TX + 2), lx = i - ly * (TX + 2);
    int fy = v.wy0 + y0 + ly - 1, fx = v.wx0 + x0 + lx - 1;  // frame coordinates
    float xn = 0.0f;
    if (fy >= 0 && fy < vs.Hf && fx >= 0 && fx < vs.Wf) {
      size_t q = (size_t)fy * vs.Wf + fx;
      float adu = (float)frame[q];
      if (np.offset_map)
        xn = ((adu - np.offset_map[q]) / np.gain_map[q]) / np.norm_scale;
      else
        xn = (adu - np.offset) * inv_scalar;
    }
    xs[ly][lx] = xn;
  }
  __syncthreads();

  const int x = x0 + threadIdx.x, y = y0 + threadIdx.y;
  if (x >= s.W || y >= s.H) return;
  float xn[9];
#pragma unroll
  for (int ky = 0; ky < 3; ++ky)
#pragma unroll
    for (int kx = 0; kx < 3; ++kx) xn[ky * 3 + kx] = xs[threadIdx.y + ky][threadIdx.x + kx];

#pragma unroll
  for (int k = 0; k < C / 8; ++k) {
    float acc[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] = bs[k * 8 + c];
#pragma unroll
    for (int t = 0; t < 9; ++t)
#pragma unroll
      for (int c = 0; c < 8; ++c) acc[c] = fmaf(xn[t], ws[t][k * 8 + c], acc[c]);
    if (relu) {
#pragma unroll
      for (int c = 0; c < 8; ++c) acc[c] = fmaxf(acc[c], 0.0f);
    }
    Chunk<T>::store(act, s.chunk_index(b, k, y, x), acc);
  }
}

template <typename T>
cudaError_t launch_t(const uint16_t* frames, int frame_base, ViewSet vs, ActShape s, NormParams np,
                     const float* w, const float* b, int relu, void* act, cudaStream_t st) {
  dim3 grid((s.W + TX - 1) / TX, (s.H + TY - 1) / TY, s.B), block(TX, TY);
  switch (s.C) {
    case 16: stem_kernel<T, 16><<<grid, block, 0, st>>>(frames, frame_base, vs, s, np, w, b, relu, (T*)act); break;
    case 32: stem_kernel<T, 32><<<grid, block, 0, st>>>(frames, frame_base, vs, s, np, w, b, relu, (T*)act); break;
    case 48: stem_kernel<T, 48><<<grid, block, 0, st>>>(frames, frame_base, vs, s, np, w, b, relu, (T*)act); break;
    case 64: stem_kernel<T, 64><<<grid, block, 0, st>>>(frames, frame_base, vs, s, np, w, b, relu, (T*)act); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_stem(bool bf16, const uint16_t* frames, int frame_base, ViewSet vs, ActShape s,
                        NormParams np, const float* w_stem, const float* b_stem, int relu,
                        void* act, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  return bf16 ? launch_t<__nv_bfloat16>(frames, frame_base, vs, s, np, w_stem, b_stem, relu, act, st)
              : launch_t<float>(frames, frame_base, vs, s, np, w_stem, b_stem, relu, act, st);
}

}  // namespace smlm
