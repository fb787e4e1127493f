// Internal interface of the DilatedLoc (paper topology) path: dloc.cu (C ABI, dloc.h) drives
// the kernels of conv_gen.cu.  Nothing here is included by, or includes, anything under oracle/.
#pragma once
#include "smlm_internal.cuh"

namespace smlm {

// One convolution of the paper's net over a RANGE OF PLANES of chunk-planar buffers
// (act[b][plane][y][x][8]): the dense concatenation of a DCD block and the skip
// concatenations of the U-Net are ranges of planes of one buffer, so "reading several source
// maps" costs nothing - the K loop of the implicit GEMM just walks more planes.
//   out[co] = act(bias[co] + sum_{ci, ky, kx} w[co][ci][ky][kx] in[ci][y + (ky - r) d][x + (kx - r) d])
// k = 2r + 1 in {1, 3}, zero padding, stride 1.
struct ConvGen {
  const void* in;    // buffer base (bf16 / fp16 or fp32 elements)
  int in_planes;     // planes per view of the input buffer
  int ci_plane0;     // first input plane
  int CI;            // input channels, multiple of 16
  void* out;         // output buffer base (chunk-planar), unused when out_f32 != nullptr
  int out_planes;    // planes per view of the output buffer
  int co_plane0;     // first output plane
  int CO;            // output channels padded to a multiple of 16
  int B, H, W;
  int k, d, relu;
  float* out_f32;    // != nullptr: planar fp32 maps [B][n_valid][H][W] instead (the head maps)
  int n_valid;       // channels actually written when out_f32 != nullptr
};

// N tile of the tensor-core kernel for CO output channels (multiple of 16, <= 128, divides CO).
int conv_gen_ntile(int CO);
// bytes of the packed 16-bit weight image: [CO / NT][CI / 16][k * k][2][NT][8]
size_t conv_gen_packed_bytes(int CI, int CO, int k);
// w_oihw [CO_real][CI][k][k] fp32 -> packed image (RNE to bf16 / fp16); rows >= CO_real are zero
void conv_gen_pack_host(int CI, int CO, int CO_real, int k, const float* w_oihw, void* dst, bool f16);
// tcgen05 implicit GEMM (16-bit maps).  bias: device float [CO].
cudaError_t launch_conv_gen_umma(bool f16, const ConvGen& a, const void* wpack, const float* bias, int n_sm,
                                 cudaStream_t st);
// Row-chain kernel for the dense blocks (conv_chain.cu): the 3x3 dilated layers (C_out = 16 or 32) and
// the 1x1 transition (C_out <= 48); input planes [0, CI / 8) of a buffer, weights resident in shared
// memory, every input row fetched once.
bool conv_chain_supports(int CI, int CO, int k, int d);
size_t conv_chain_packed_bytes(int CI, int CO, int k);
void conv_chain_pack_host(int CI, int CO, int CO_real, int k, const float* w_oihw, void* dst, bool f16);
cudaError_t launch_conv_chain(bool f16, const ConvGen& a, const void* wpack, const LayerConst& lc, int n_sm,
                              cudaStream_t st);
// CUDA-core twin (fp32 math; maps float, bf16 or fp16).  w: device float [k * k][CI][CO].
cudaError_t launch_conv_gen_direct(int dt, const ConvGen& a, const float* w, const float* bias, cudaStream_t st);

// 2x2 max pooling, stride 2, floor (D4): planes [pi0, pi0 + np) of `in` (H x W) -> planes
// [po0, po0 + np) of `out` (H/2 x W/2).
cudaError_t launch_pool2(int dt, const void* in, int in_planes, int pi0, void* out, int out_planes, int po0, int np,
                         int B, int H, int W, cudaStream_t st);
// nearest-neighbour x2 to exactly Ho x Wo (D5): out[y][x] = in[min(y/2, H-1)][min(x/2, W-1)].
cudaError_t launch_up2(int dt, const void* in, int in_planes, int pi0, int H, int W, void* out, int out_planes,
                       int po0, int np, int B, int Ho, int Wo, cudaStream_t st);
// debug: planes [p0, p0 + np) -> float dst[b * view_stride + (c * H + y) * W + x]
cudaError_t launch_dump_planar(int dt, const void* in, int in_planes, int p0, int np, int B, int H, int W,
                               float* dst, size_t view_stride, cudaStream_t st);

struct DlocPostParams {
  HeadParams hp;      // n_h = 10; heads 0-5 decoded by the six-head rule of smlm.h
  float sigma_xy_px, sigma_z_nm, sigma_photons;
};
// detection + decode on fp32 maps [n][10][H][W]; frame index of view b = frame0 + b
cudaError_t launch_dloc_post(const float* maps, int n, int H, int W, int frame0, DlocPostParams pp, void* out48,
                             unsigned long long* counter, unsigned long long capacity, cudaStream_t st);

}  // namespace smlm
