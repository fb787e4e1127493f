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
//     act[b][k][y][x][8]      b < B views, k < C/8 channel chunks, y < H, x < W, 8 channels
// Why: (1) a pixel's 8-channel chunk is one 16-byte (bf16) vector, and consecutive pixels of
// one chunk are consecutive in memory, so every warp-wide access is a dense 512 B run;
// (2) one chunk-plane row IS the UMMA "K-major, no swizzle" core-matrix sequence
// (8 pixels x 16 B = one 128 B core matrix), so a TMA box lands in shared memory already in
// the layout tcgen05.mma reads, at ANY pixel shift (conv_umma.cu) - which is what a dilated
// convolution needs.
// ---------------------------------------------------------------------------------------
struct ActShape {
  int B, C, H, W;
  int CT = 0;  // channels per view of the buffer the map lives in (0: = C).  > C when the map is a
               // slice of a concatenation buffer (dloc.cu): the planes of a view stay contiguous
  __host__ __device__ size_t elems() const { return (size_t)B * C * H * W; }
  __host__ __device__ size_t chunk_index(int b, int k, int y, int x) const {
    return ((((size_t)b * ((CT > 0 ? CT : C) >> 3) + k) * H + y) * W + x);
  }
};

// One unit of a micro-batch is a VIEW: a window of a frame (the whole frame, or one tile plus
// halo clipped to the frame).  All views of a launch have the same window size (s.H x s.W).
// They are described parametrically (no table in memory): view v of the set is tile
// (ty0 + (v / nx) % ny, tx0 + v % nx) of frame frame0 + v / (ny * nx).
struct ViewSet {
  int frame0;        // first frame (index within the call)
  int Hf, Wf;        // frame size
  int tile;          // 0: whole frames
  int halo;          // tile mode: window = core +- halo, clipped to the frame
  int ty0, ny, tx0, nx;
  int tile_w;        // core width (0: = tile).  SMLM_TILE_MERGE_ROW sets it to the frame width: the
                     // tiles of one tile row share one window and their x halos are computed once
  int in_frames;     // 3: the stem reads frames f-1, f, f+1 (0 / 1: frame f only)
  int n_total;       // frames of the call: the clamp bound of the temporal context
};

// Storage type of the activation maps (smlm_net_desc.precision).
enum ActType { ACT_F32 = 0, ACT_BF16 = 1, ACT_F16 = 2 };

struct View {
  int frame;
  int wy0, wx0;            // window origin inside the frame
  int cy0, cy1, cx0, cx1;  // owned ("core") rectangle in window coordinates, half-open
};

__host__ __device__ inline View view_of(const ViewSet& vs, int v, int Hw, int Ww) {
  View r;
  if (vs.tile <= 0) {
    r.frame = vs.frame0 + v;
    r.wy0 = r.wx0 = 0;
    r.cy0 = r.cx0 = 0;
    r.cy1 = Hw;
    r.cx1 = Ww;
    return r;
  }
  int per = vs.ny * vs.nx;
  int f = v / per, t = v - f * per;
  int ty = vs.ty0 + t / vs.nx, tx = vs.tx0 + t % vs.nx;
  int tw = vs.tile_w > 0 ? vs.tile_w : vs.tile;
  int y0 = ty * vs.tile, x0 = tx * tw;
  int y1 = y0 + vs.tile < vs.Hf ? y0 + vs.tile : vs.Hf;
  int x1 = x0 + tw < vs.Wf ? x0 + tw : vs.Wf;
  r.frame = vs.frame0 + f;
  r.wy0 = y0 - vs.halo > 0 ? y0 - vs.halo : 0;
  r.wx0 = x0 - vs.halo > 0 ? x0 - vs.halo : 0;
  r.cy0 = y0 - r.wy0;
  r.cx0 = x0 - r.wx0;
  r.cy1 = y1 - r.wy0;
  r.cx1 = x1 - r.wx0;
  return r;
}

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

// K1: uint16 unpack + normalise + 3x3 stem conv (+ReLU) -> act.
// frames: device u16, frame f of the call at frames + (f - frame_base) * Hf * Wf.
cudaError_t launch_stem(int dt, const uint16_t* frames, int frame_base, ViewSet vs, ActShape s,
                        NormParams np, const float* w_stem /*[in_frames * 9][C]*/, const float* b_stem,
                        int relu, void* act, cudaStream_t st);

// K1 on the tensor cores (conv_chain.cu, STEM variant; 16-bit maps, in_frames = 1): the same
// function as launch_stem with fp32 accuracy from 16-bit operand pieces; HBM-write-bound.
struct LayerConst;
bool stem_umma_supports(int C, int in_frames);
size_t stem_umma_packed_bytes(int C);
void stem_umma_pack_host(int C, const float* w_stem /*[9][C]*/, const float* b_stem /*[C]*/, void* dst, bool f16);
cudaError_t launch_stem_umma(bool f16, const uint16_t* frames, int frame_base, ViewSet vs, ActShape s, NormParams np,
                             const void* wpack, const LayerConst& lc, int relu, void* act, int n_sm, cudaStream_t st);

// K2' reference trunk layer on CUDA cores (fp32 math; storage float, bf16 or fp16).
// w: [9][C_in][C_out] float (already rounded to the storage type's values in the 16-bit modes).
cudaError_t launch_conv_direct(int dt, const void* in, void* out, ActShape s, int dil,
                               const float* w, const float* b, cudaStream_t st);
cudaError_t conv_direct_init(int C);  // opt in to the shared memory the kernel needs

// K2 trunk layer on tcgen05 tensor cores (bf16 or fp16 storage, fp32 accumulate in TMEM).
size_t umma_packed_weight_bytes(int C);
// w_oihw [C][C][3][3] fp32 -> the kernel's shared-memory image (bf16 or fp16, RNE), host side.
void umma_pack_weights_host(int C, const float* w_oihw, void* dst, bool f16);
float round_to_act(float v, int dt);  // host: RNE to the storage type's value set
// STEM variant (first layer, K1 folded in): a_0 is computed in the kernel from the frames.
// The per-layer constants travel as kernel parameters: parameters live in constant memory,
// so a weight with a compile-time index is a free operand of the FMA that uses it (no
// shared-memory or register traffic - the shared-memory pipe belongs to the tensor core's
// operand fetch, profiles/).
struct LayerConst {
  float bias[64];
};
struct StemArgs {
  const uint16_t* frames;  // device; frame f of the call at frames + (f - frame_base) Hf Wf
  int frame_base;
  ViewSet vs;
  NormParams np;
  int relu;
  float w[9][64];  // [tap ky*3+kx][channel]
  float b[64];
};

// HEAD (K3 folded in): what the last layer's epilogue writes instead of the activation map.
struct HeadArgs {
  int n_h;
  float lthr;       // logit(threshold)
  float* logit;     // [B][H][W] detection logit of every pixel
  float* cand;      // [B][H][W][8]: heads 1 .. n_h-1 (pre-activation) of pixels with logit > lthr
  float w[64][8];   // [channel][head], zero beyond n_h
  float b[8];
};

bool conv_umma_supports(int C, int dil, bool stem);
// head != nullptr: last layer, HEAD variant (`out` is not written).  stem != nullptr: first
// layer, STEM variant (`in` is not read).
cudaError_t launch_conv_umma(bool f16, const void* in, void* out, ActShape s, int dil, const void* wpack,
                             const LayerConst& lc, const HeadArgs* head, const StemArgs* stem, int n_sm,
                             cudaStream_t st, char* err, size_t errlen);

// K2 pair (conv_pair.cu): layers l and l+1 with dilations (d, 2d) in one kernel; the map between
// them stays in shared memory.  Bit-identical to two launch_conv_umma calls.  head != nullptr:
// layer l+1 is the last one (HEAD variant: head->logit gets the detection logit of every pixel,
// `out` is written only where it exceeds head->lthr; head->cand is not used).  allow_cg2: rows with an even
// number of segments use tcgen05 cta_group::2 (one M = 256 MMA per CTA pair).
bool conv_pair_supports(int C, int dA, int dB, int W);
cudaError_t launch_conv_pair(bool f16, const void* in, void* out, ActShape s, int dA, const void* wpackA,
                             const void* wpackB, const LayerConst& lcA, const LayerConst& lcB, const HeadArgs* head,
                             bool allow_cg2, int n_sm, cudaStream_t st, char* err, size_t errlen);

// K3: 1x1 heads + threshold + 3x3 NMS + decode + warp-aggregated compaction.
cudaError_t launch_head_post(int dt, const void* act, ActShape s, ViewSet vs,
                             const float* w_head /*[n_h][C]*/, const float* b_head, HeadParams hp,
                             smlm_emitter* out, unsigned long long* counter,
                             unsigned long long capacity, cudaStream_t st);

// K3 after a HEAD conv layer: the detection logit comes from `logit` [B][H][W], the other
// heads of every pixel above the threshold from `cand` [B][H][W][8] (HeadArgs).
cudaError_t launch_post_logits(const float* logit, const float* cand, ActShape s, ViewSet vs,
                               HeadParams hp, smlm_emitter* out, unsigned long long* counter,
                               unsigned long long capacity, cudaStream_t st);

// K3 after the HEAD launch of conv_pair.cu: the detection logit from `logit`, the other heads
// evaluated here from `act` - the last map, which that launch stored for above-threshold pixels only.
cudaError_t launch_post_logits_act(int dt, const float* logit, const void* act, ActShape s, ViewSet vs,
                                   const float* w_head, const float* b_head, HeadParams hp, smlm_emitter* out,
                                   unsigned long long* counter, unsigned long long capacity, cudaStream_t st);

// debug: heads only -> fp32 maps [B][n_h][H][W] (pre-activation)
cudaError_t launch_head_maps(int dt, const void* act, ActShape s, const float* w_head,
                             const float* b_head, int n_h, float* maps, cudaStream_t st);
// debug: act -> float dst[b * view_stride + (y*W + x)*C + c]
cudaError_t launch_dump_act(int dt, const void* act, ActShape s, float* dst, size_t view_stride,
                            cudaStream_t st);
// debug: detection + decode on caller maps [n][n_h][H][W]
cudaError_t launch_post_from_maps(const float* maps, int n, int H, int W, HeadParams hp,
                                  smlm_emitter* out, unsigned long long* counter,
                                  unsigned long long capacity, cudaStream_t st);

// snap[0] = min(*counter, capacity)
cudaError_t launch_snapshot(const unsigned long long* counter, unsigned long long capacity,
                            unsigned long long* snap, cudaStream_t st);
// copy records [*lo, *hi) from the device list to a device-visible host list
cudaError_t launch_flush_emitters(const smlm_emitter* dev, smlm_emitter* host_mapped,
                                  const unsigned long long* lo, const unsigned long long* hi,
                                  cudaStream_t st);

}  // namespace smlm
