/*
 * dloc.h -- C ABI of the PAPER'S OWN network topology on one B200 (sm_100a): DilatedLoc
 * as arXiv 2410.02314 describes it, next to the residual stack of smlm.h that BASELINE.json
 * fixes.  Same library (libsmlm_b200.so), same camera struct, same
 * post-processing rule; only the network between the frames and the head maps differs.
 *
 * What the paper fixes (P:nn = /root/reference/PAPER.md line nn):
 *   P:57, P:67  Dense Connection Dilated blocks (DCD): "each layer [utilizes] outputs from all
 *               preceding layers" - layer i of a block is a dilated 3x3 convolution over the
 *               concatenation of the block input and the outputs of layers 0..i-1;
 *   P:59        one coarse-grained DCD (n = 1) followed by three multi-scale DCDs (n = 3);
 *   P:144       "dilation parameters ... (2, 4, 8, 16)";
 *   P:61, "fine-grained processing using a two-stage U-Net" with "two upsampling
 *               stages"; per pixel "the probability of a fluorescent molecule, along with the
 *               offset and uncertainty of the fluorescent molecule's position";
 *   P:53        optional three-frame temporal context.
 * What it does not fix (widths, growth rate, pooling, up-sampling, head activations) is a
 * READING, D1-D9 in DESIGN.md, a field or constant here and in oracle/dloc_oracle.c alike.
 *
 * Network (C0 = c0, G = growth, n = n_dil, CB = C0 + n G):
 *   xhat = ((adu - offset) / gain) / norm_scale                       (per frame; in_frames = 3:
 *          channels = frames f-1, f, f+1, indices clamped to the call)
 *   f    = act(conv3x3(xhat; in_frames -> C0))                        stem, zero padding 1
 *   n_blocks times:  for i < n:  g_i = ReLU(conv3x3 dilation d_i ([f | g_0 .. g_{i-1}]; -> G))
 *                    f = ReLU(conv1x1([f | g_0 .. g_{n-1}]; CB -> C0))  transition
 *   e0 = f;  e1 = ReLU(conv3x3(maxpool2(e0); C0 -> 2C0));  e2 = ReLU(conv3x3(maxpool2(e1); 2C0 -> 4C0))
 *   m1 = ReLU(conv3x3([up2(e2) | e1]; 6C0 -> 2C0));  m0 = ReLU(conv3x3([up2(m1) | e0]; 3C0 -> C0))
 *   o  = conv1x1(m0; C0 -> 10)       heads: p, dx, dy, z, N, bg, sigma_x, sigma_y, sigma_z, sigma_N
 * All convolutions are cross-correlations with zero ("same") padding; maxpool2 = 2x2 stride 2,
 * floor; up2 = nearest neighbour to exactly the finer map's size.
 * Detection and decode of heads 0-5: the rule of smlm.h (logit-domain threshold, 3x3 local
 * maximum with the lower-index tie rule, pixel-centre coordinates).  Uncertainties (D7):
 *   sigma_x_nm = sigma_xy_px sigmoid(o_6) pixel_size, sigma_y likewise (o_7),
 *   sigma_z_nm = sigma_z_nm sigmoid(o_8), sigma_photons = sigma_photons sigmoid(o_9).
 *
 * Precision: DLOC_FP32 = every kernel on CUDA cores in fp32 (reference mode, 1e-4 against the
 * fp64 oracle); DLOC_BF16 = 16-bit maps and weights, every convolution except the stem on the
 * tcgen05 tensor cores with fp32 accumulation (implicit GEMM over the concatenated source
 * planes: the chunk-planar layout makes a concatenation a range of planes), stem and
 * post-processing in fp32.
 *
 * Pointers: `frames_u16` device or PINNED host (double-buffered H2D on a copy stream);
 * `out_emitters` device or pinned host; maps of the debug call: device.  Errors as smlm.h.
 */
#ifndef DLOC_B200_H
#define DLOC_B200_H

#include "smlm.h"

#ifdef __cplusplus
extern "C" {
#endif

#define DLOC_ABI_VERSION 1
#define DLOC_HEADS 10
#define DLOC_MAX_DIL 8

typedef struct dloc_ctx dloc_ctx;

typedef struct {
  uint32_t struct_size; /* sizeof(dloc_net_desc) */
  uint32_t version;     /* DLOC_ABI_VERSION */
  int32_t c0;           /* base width, multiple of 16, 16..64 (D1) */
  int32_t growth;       /* channels each DCD layer adds, multiple of 16, 16..64 (D1) */
  int32_t n_blocks;     /* DCD blocks, 1..8 (1 + 3) */
  int32_t n_dil;        /* layers per block, 1..DLOC_MAX_DIL */
  int32_t dilations[DLOC_MAX_DIL]; /* 1..16 (2, 4, 8, 16) */
  int32_t in_frames;    /* 1 or 3 (D8) */
  int32_t stem_relu;
  int32_t precision;    /* SMLM_FP32 | SMLM_BF16 */
  float norm_scale, xy_scale, z_scale_nm, photon_scale, bg_scale;
  float sigma_xy_px, sigma_z_nm, sigma_photons; /* D7 */
  int32_t micro_batch;  /* frames per launch set; 0 = library default */
  int32_t conv_impl;    /* 16-bit precision only.  SMLM_CONV_AUTO: tcgen05, the dense-block layers through the
                           row-chain kernel (conv_chain.cu); TCGEN05: every convolution through the generic
                           tcgen05 kernel (the twin); DIRECT: CUDA cores */
} dloc_net_desc;

/* smlm_emitter plus the four uncertainties. */
typedef struct {
  int32_t frame, pix;
  float x_nm, y_nm, z_nm, photons, bg, p;
  float sx_nm, sy_nm, sz_nm, s_photons;
} dloc_emitter; /* 48 bytes */

/* weights: HOST pointer, one little-endian fp32 blob, OIHW, in this order:
 *   stem W[C0][in_frames][3][3] b[C0];  per block: per layer i W[G][C0+iG][3][3] b[G], then the
 *   transition W[C0][CB][1][1] b[C0];  enc1 W[2C0][C0][3][3] b;  enc2 W[4C0][2C0][3][3] b;
 *   dec1 W[2C0][6C0][3][3] b;  dec0 W[C0][3C0][3][3] b;  heads W[10][C0] b[10].
 * Synchronous.  INVALID_ARG, UNSUPPORTED_DEVICE, CUDA, OOM. */
smlm_status dloc_create(const dloc_net_desc* desc, const void* weights, dloc_ctx** out_ctx);

/* The whole path for n frames of H x W (H, W >= 4): stem, DCD blocks, U-Net, heads, detection,
 * decode, compaction.  *out_count in: capacity, out: emitters found; written from a host callback
 * ordered on the stream, so the int64 must stay allocated until the stream has finished the call.
 * Order of the list unspecified.
 * Asynchronous on `cuda_stream` when out_emitters is DEVICE memory.  With a PINNED HOST list the
 * call waits (cudaStreamSynchronize) for its own kernels before it returns: the list is compacted
 * on the device and copied out in one piece once the count is known, a copy that is not
 * overlapped with compute (smlm_localize's chunked write-back is not implemented for this net);
 * when the capacity grows it also reallocates the device list behind a device-wide sync. */
smlm_status dloc_localize(dloc_ctx* ctx, const uint16_t* frames_u16, int64_t n_frames, int32_t H, int32_t W,
                          const smlm_camera_params* camera_params, float threshold, dloc_emitter* out_emitters,
                          int64_t* out_count, void* cuda_stream);

/* Test export: pre-activation head maps [n][10][H][W] fp32 (device).  `dump` (device, may be
 * NULL) receives per frame, planar [c][h][w] fp32, in this order: stem (C0,H,W); each block's
 * transition output (C0,H,W); e1 (2C0,H/2,W/2); e2 (4C0,H/4,W/4); m1 (2C0,H/2,W/2); m0 (C0,H,W). */
smlm_status dloc_debug_forward_maps(dloc_ctx* ctx, const uint16_t* frames_u16, int64_t n_frames, int32_t H,
                                    int32_t W, const smlm_camera_params* camera_params, float* maps,
                                    float* dump, void* cuda_stream);

smlm_status dloc_check(dloc_ctx* ctx);            /* pending CUDA error / overflow of the last call */
const char* dloc_last_error(const dloc_ctx* ctx); /* NULL ctx: error of the last failed dloc_create */
int64_t dloc_launch_count(const dloc_ctx* ctx);   /* kernels launched so far */
/* CUDA-event timing of the convolution launches (the dominant kernel), as smlm_kernel_timing. */
smlm_status dloc_kernel_timing(dloc_ctx* ctx, int32_t enable);
smlm_status dloc_conv_time_ms(dloc_ctx* ctx, double* ms, int64_t* launches);
void dloc_destroy(dloc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
