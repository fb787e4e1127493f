// Internal declarations shared by the translation units of libsmlm_b200.
// Nothing here is included by, or includes, anything under oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/smlm.h"

namespace smlm {

// ---------------------------------------------------------------------------------------
// Activation layout in HBM ("chunk-planar NHWC8"):
//     act[b][k][y][x][8]      b < B views, k < C/8 channel chunks, y < H, x < Wp, 8 channels
// Wp = W rounded up to a multiple of 8; columns W..Wp-1 always hold zeros.
// Why: (1) a pixel's 8-channel chunk is one 16-byte (bf16) vector, and consecutive pixels of
// one chunk are consecutive in memory, so every warp-wide access is a dense 512 B run;
// (2) one chunk plane row IS the UMMA "K-major, no swizzle" core-matrix sequence
// (8 pixels x 16 B = one 128 B core matrix), so a TMA box lands in shared memory already in
// the layout tcgen05.mma reads, at any pixel shift (conv_umma.cu).
// ---------------------------------------------------------------------------------------
struct ActShape {
  int B, C, H, W, Wp;
  __host__ __device__ size_t elems() const { return (size_t)B * C * H * Wp; }
  __host__ __device__ size_t chunk_index(int b, int k, int y, int x) const {
    return ((((size_t)b * (C >> 3) + k) * H + y) * Wp + x);
  }
};

// One unit of a micro-batch: a window of a frame (whole frame, or one haloed tile).
struct View {
  int frame;           // frame index within the call
  int wy0, wx0;        // window origin inside the frame
  int cy0, cy1, cx0, cx1;  // owned ("core") rectangle in window coordinates, half-open
};

struct HeadParams {
  int n_h;
  float lthr;  // logit(threshold): -inf => all local maxima, +inf => none
  float xy_scale, z_scale_nm, photon_scale, bg_scale, pixel_size_nm;
};

struct NormParams {
  float offset, gain, norm_scale;
  const float* offset_map;  // device [Hf][Wf] or nullptr
  const float* gain_map;
};

// ----------------------------------------------------------------------------- launchers
// (each returns the cudaError_t of the launch; all are asynchronous on `st`)

// K1: uint16 unpack + normalise + 3x3 stem conv (+ReLU) -> act.  T = float | __nv_bfloat16.
cudaError_t launch_stem(bool bf16, const uint16_t* frames, int Hf, int Wf, const View* views,
                        ActShape s, NormParams np, const float* w_stem /*[9][C]*/,
                        const float* b_stem, int relu, void* act, cudaStream_t st);

// K2' reference trunk layer on CUDA cores (fp32 math; storage float or bf16).
// w: [9][C_in][C_out] float (already rounded to bf16 values in bf16 mode).
cudaError_t launch_conv_direct(bool bf16, const void* in, void* out, ActShape s, int dil,
                               const float* w, const float* b, cudaStream_t st);

// K2 trunk layer on tcgen05 tensor cores (bf16 storage, fp32 accumulate in TMEM).
struct UmmaLayerPlan;  // opaque, conv_umma.cu
UmmaLayerPlan* umma_plan_create(int C, int n_sm, char* err, size_t errlen);
void umma_plan_destroy(UmmaLayerPlan*);
// wpack: device, layout produced by umma_pack_weights_host; bias: device float [C].
size_t umma_packed_weight_bytes(int C);
void umma_pack_weights_host(int C, const float* w_oihw /*[C][C][3][3]*/, void* dst_bf16);
cudaError_t launch_conv_umma(UmmaLayerPlan* plan, const void* in, void* out, ActShape s, int dil,
                             const void* wpack, const float* bias, int band_rows,
                             cudaStream_t st, char* err, size_t errlen);

// K3: 1x1 heads + threshold + 3x3 NMS + decode + warp-aggregated compaction.
cudaError_t launch_head_post(bool bf16, const void* act, ActShape s, const View* views, int Wf,
                             const float* w_head /*[n_h][C]*/, const float* b_head, HeadParams hp,
                             smlm_emitter* out, unsigned long long* counter,
                             unsigned long long capacity, cudaStream_t st);

// debug: heads only -> fp32 maps [B][n_h][H][W] (pre-activation)
cudaError_t launch_head_maps(bool bf16, const void* act, ActShape s, const float* w_head,
                             const float* b_head, int n_h, float* maps, cudaStream_t st);
// debug: act -> float [B][slot of L1][H][W][C]
cudaError_t launch_dump_act(bool bf16, const void* act, ActShape s, float* dst, size_t view_stride,
                            cudaStream_t st);
// debug: detection + decode on caller maps [n][n_h][H][W]
cudaError_t launch_post_from_maps(const float* maps, int n, int H, int W, HeadParams hp,
                                  smlm_emitter* out, unsigned long long* counter,
                                  unsigned long long capacity, cudaStream_t st);

// copy records [done, min(counter, capacity)) from the device list to a mapped host list
cudaError_t launch_flush_emitters(const smlm_emitter* dev, smlm_emitter* host_mapped,
                                  const unsigned long long* counter, unsigned long long* flushed,
                                  unsigned long long capacity, cudaStream_t st);
// write min/actual count to a (mapped host or device) int64
cudaError_t launch_store_count(const unsigned long long* counter, long long* dst, cudaStream_t st);

}  // namespace smlm
