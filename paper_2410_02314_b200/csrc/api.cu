// C ABI of libsmlm_b200 (include/smlm.h) and the pipeline around the kernels:
// pinned host ring -> copy stream -> staging slots -> compute stream (K1, K2 x L, K3) ->
// write-back stream.  Enqueue only: no host synchronisation inside smlm_localize.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "ring.cuh"
#include "smlm_internal.cuh"

using namespace smlm;

namespace {

constexpr int kSlots = 3;  // staging slots of the preload ring (copy k+1, k+2 while k computes)
// Write-back (step W): flush k copies the records [snap[(k-1) % R], snap[k % R]) to the host
// list on the write-back stream.  The snapshots are written on the compute stream, so each
// flush owns one word of a ring; a word is rewritten only after the two flushes that read it
// (k - R as its upper end, k - R + 1 as its lower end) have finished (event wait below).
constexpr int kSnapRing = 4;
constexpr int kCounterWords = 2 + kSnapRing;

thread_local std::string g_create_error;

constexpr int kFirstParts = 4;

struct Layer {
  float* w_direct = nullptr;  // [9][C][C] (tap, ci, co)
  void* w_umma = nullptr;     // packed bf16 image for conv_umma
  float* bias = nullptr;
  LayerConst lc{};            // the bias again, as a kernel parameter of conv_umma
  int dil = 1;
};

}  // namespace

struct smlm_ctx {
  smlm_net_desc d{};
  bool bf16 = false;  // 16-bit storage (bf16 or fp16)
  int dt = ACT_F32;   // ActType of the maps
  int in_frames = 1;
  bool use_umma = false;
  int n_sm = 0;
  int radius = 0;  // receptive-field radius of the maps: 1 + sum(dilations)
  size_t l2_bytes = 0;

  float *w_stem = nullptr, *b_stem = nullptr, *w_head = nullptr, *b_head = nullptr;
  StemArgs stem_args{};  // host templates of conv_umma's parameter blocks (weights filled at create)
  HeadArgs head_args{};
  std::vector<Layer> layers;

  void* act[2] = {nullptr, nullptr};
  size_t act_bytes = 0;
  float* logit = nullptr;  // detection logit of every pixel, written by the last tcgen05 layer (HEAD)
  float* cand = nullptr;   // 32-byte candidate records (other heads) of above-threshold pixels
  bool fuse = true;        // desc.fusion != SMLM_FUSE_NONE: K3's heads in the last layer's epilogue
  bool fuse_stem = false;  // desc.fusion == SMLM_FUSE_ALL: K1 inside the first layer's kernel
  bool fuse_pairs = true;  // AUTO / ALL / PAIRS_1CTA: layers (d, 2d) as one kernel (conv_pair.cu)
  bool pair_cg2 = true;    // ... with tcgen05 cta_group::2 where a row has an even number of segments
  bool stem_tensor = false;  // K1 on the tensor cores (conv_chain.cu STEM variant)
  void* w_stem_umma = nullptr;
  LayerConst stem_lc{};

  uint16_t* slots = nullptr;  // kSlots x slot_elems
  size_t slot_elems = 0;
  bool slot_used[kSlots] = {false, false, false};
  cudaEvent_t ev_copied[kSlots]{}, ev_consumed[kSlots]{};
  cudaEvent_t ev_part[kFirstParts]{};  // the first chunk of a call arrives in parts: K1 starts on the first one
  cudaEvent_t ev_start = nullptr, ev_batch = nullptr;
  cudaEvent_t ev_wb[kSnapRing]{};  // flush k records ev_wb[k % kSnapRing] on the write-back stream
  cudaStream_t copy_stream = nullptr, wb_stream = nullptr;

  smlm_emitter* em_dev = nullptr;
  size_t em_cap = 0;
  unsigned long long* counters = nullptr;  // [0] count, [1] zero (lower end of flush 0), [2 ..) snapshot ring
  unsigned long long* h_count = nullptr;   // pinned, for smlm_check
  unsigned long long last_capacity = 0;

  float *cam_off = nullptr, *cam_gain = nullptr;
  size_t cam_elems = 0;

  int64_t launches = 0;
  bool timing = false;
  std::vector<cudaEvent_t> tev;  // pairs
  std::vector<int> tev_kind;     // one per pair
  size_t tev_used = 0;

  std::string err;
};

namespace {

smlm_status fail(smlm_ctx* c, smlm_status st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf;
  else g_create_error = buf;
  return st;
}

#define CK(c, call)                                                                          \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess)                                                                   \
      return fail(c, e_ == cudaErrorMemoryAllocation ? SMLM_ERR_OOM : SMLM_ERR_CUDA,          \
                  "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);      \
  } while (0)

// kernel timing (smlm_kernel_timing): bracket one launch with two events on its stream
smlm_status time_begin(smlm_ctx* c, int kind, cudaStream_t st, cudaEvent_t* e1) {
  *e1 = nullptr;
  if (!c->timing) return SMLM_OK;
  if (c->tev_used + 2 > c->tev.size()) {
    for (int i = 0; i < 2; ++i) {
      cudaEvent_t e;
      CK(c, cudaEventCreate(&e));
      c->tev.push_back(e);
    }
  }
  if (c->tev_kind.size() < c->tev.size() / 2) c->tev_kind.resize(c->tev.size() / 2);
  c->tev_kind[c->tev_used / 2] = kind;
  cudaEvent_t e0 = c->tev[c->tev_used++];
  *e1 = c->tev[c->tev_used++];
  CK(c, cudaEventRecord(e0, st));
  return SMLM_OK;
}
smlm_status time_end(smlm_ctx* c, cudaEvent_t e1, cudaStream_t st) {
  if (e1) CK(c, cudaEventRecord(e1, st));
  return SMLM_OK;
}

enum PtrKind { PTR_DEVICE, PTR_HOST_PINNED, PTR_OTHER };
PtrKind classify(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return PTR_OTHER;
  }
  if (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) return PTR_DEVICE;
  if (a.type == cudaMemoryTypeHost) return PTR_HOST_PINNED;
  return PTR_OTHER;
}

smlm_status ensure_act(smlm_ctx* c, size_t bytes) {
  if (bytes <= c->act_bytes) return SMLM_OK;
  for (int i = 0; i < 2; ++i) {
    if (c->act[i]) cudaFree(c->act[i]);
    c->act[i] = nullptr;
  }
  c->act_bytes = 0;
  for (int i = 0; i < 2; ++i) CK(c, cudaMalloc(&c->act[i], bytes));
  c->act_bytes = bytes;
  if (c->use_umma) {  // bytes / (C * 2) pixels: one fp32 logit and one 32-byte candidate record each
    if (c->logit) cudaFree(c->logit);
    if (c->cand) cudaFree(c->cand);
    c->logit = c->cand = nullptr;
    const size_t px = bytes / ((size_t)c->d.channels * 2);
    CK(c, cudaMalloc(&c->logit, px * sizeof(float)));
    CK(c, cudaMalloc(&c->cand, px * 8 * sizeof(float)));
  }
  return SMLM_OK;
}

// K1 -> K2 x L for one launch set; the result is in act[*result_buf] (or, when *have_logit
// comes back true, in c->logit / c->cand: the last layer ran as the HEAD variant).
// lthr: logit(threshold) for the HEAD variant (want_logit).
smlm_status run_trunk(smlm_ctx* c, const uint16_t* dev_frames, int frame_base, const ViewSet& vs,
                      ActShape s, const NormParams& np, cudaStream_t st, int* result_buf,
                      float* trunk_dump, size_t dump_view_stride, size_t dump_level_stride,
                      cudaEvent_t after_stem, bool want_logit, float lthr, bool* have_logit,
                      bool* heads_from_act = nullptr, int stem_parts = 1) {
  if (have_logit) *have_logit = false;
  if (heads_from_act) *heads_from_act = false;
  const size_t nl = c->layers.size();
  // layers l, l+1 run as one kernel (conv_pair.cu) when their dilations are (d, 2d); pairs are
  // formed greedily from the first layer on (the trunk dump wants every level: no pairs then)
  auto pair_at = [&](size_t l) {
    return c->use_umma && c->fuse_pairs && !trunk_dump && l + 1 < nl && c->layers[l + 1].dil == 2 * c->layers[l].dil &&
           conv_pair_supports(c->d.channels, c->layers[l].dil, c->layers[l + 1].dil, s.W);
  };
  // K1 folded into the first trunk layer (STEM variant) when the tcgen05 path runs it
  const bool fuse_stem = c->use_umma && c->fuse_stem && nl > 0 && c->dt == ACT_BF16 && c->in_frames == 1 &&
                         !pair_at(0) && conv_umma_supports(c->d.channels, c->layers[0].dil, true);
  cudaEvent_t te = nullptr;
  smlm_status tr = SMLM_OK;
  if (!fuse_stem || trunk_dump) {  // (the trunk dump wants a_0 itself)
    // stem_parts > 1 (first chunk of a call from host memory, whole frames): the frames arrive
    // in that many H2D copies (ev_part); K1 runs per part and starts as soon as the first one is
    // there, so only a quarter of the first copy is exposed
    for (int q = 0; q < stem_parts; ++q) {
      const int v0 = (int)((long long)s.B * q / stem_parts), v1 = (int)((long long)s.B * (q + 1) / stem_parts);
      if (v1 <= v0) continue;
      if (stem_parts > 1) CK(c, cudaStreamWaitEvent(st, c->ev_part[q], 0));
      ViewSet vq = vs;
      vq.frame0 = vs.frame0 + v0;
      ActShape sq = s;
      sq.B = v1 - v0;
      void* aq = static_cast<char*>(c->act[0]) + (size_t)v0 * s.C * s.H * s.W * (c->bf16 ? 2 : 4);
      if ((tr = time_begin(c, SMLM_KERNEL_STEM, st, &te)) != SMLM_OK) return tr;
      if (c->stem_tensor)
        CK(c, launch_stem_umma(c->dt == ACT_F16, dev_frames, frame_base, vq, sq, np, c->w_stem_umma, c->stem_lc,
                               c->d.stem_relu, aq, c->n_sm, st));
      else
        CK(c, launch_stem(c->dt, dev_frames, frame_base, vq, sq, np, c->w_stem, c->b_stem, c->d.stem_relu, aq, st));
      c->launches++;
      if ((tr = time_end(c, te, st)) != SMLM_OK) return tr;
    }
    if (trunk_dump) {
      CK(c, launch_dump_act(c->dt, c->act[0], s, trunk_dump, dump_view_stride, st));
      c->launches++;
    }
  }
  if (after_stem && !fuse_stem) CK(c, cudaEventRecord(after_stem, st));
  int cur = 0;
  for (size_t l = 0; l < nl; ++l) {
    const Layer& L = c->layers[l];
    cudaEvent_t e1 = nullptr;
    const bool pair = pair_at(l);
    if ((tr = time_begin(c, pair ? SMLM_KERNEL_CONV_PAIR : SMLM_KERNEL_CONV, st, &e1)) != SMLM_OK) return tr;
    if (pair) {
      char err[256] = {0};
      const bool head = want_logit && c->fuse && l + 2 == nl;
      if (head) {
        c->head_args.lthr = lthr;
        c->head_args.logit = c->logit;
        c->head_args.cand = c->cand;
      }
      const Layer& L2 = c->layers[l + 1];
      cudaError_t e = launch_conv_pair(c->dt == ACT_F16, c->act[cur], c->act[cur ^ 1], s, L.dil, L.w_umma, L2.w_umma,
                                       L.lc, L2.lc, head ? &c->head_args : nullptr, c->pair_cg2, c->n_sm, st, err, sizeof err);
      if (head && have_logit) *have_logit = true;
      if (head && heads_from_act) *heads_from_act = true;  // act[cur ^ 1] holds the last map at the candidates
      if (e != cudaSuccess) return fail(c, SMLM_ERR_CUDA, "conv_pair: %s %s", cudaGetErrorString(e), err);
      ++l;
    } else if (c->use_umma) {
      char err[256] = {0};
      const bool head = want_logit && c->fuse && l + 1 == nl;
      const bool stem = fuse_stem && l == 0;
      if (head) {
        c->head_args.lthr = lthr;
        c->head_args.logit = c->logit;
        c->head_args.cand = c->cand;
      }
      if (stem) {
        c->stem_args.frames = dev_frames;
        c->stem_args.frame_base = frame_base;
        c->stem_args.vs = vs;
        c->stem_args.np = np;
        c->stem_args.relu = c->d.stem_relu;
      }
      cudaError_t e = launch_conv_umma(c->dt == ACT_F16, c->act[cur], c->act[cur ^ 1], s, L.dil, L.w_umma, L.lc,
                                       head ? &c->head_args : nullptr, stem ? &c->stem_args : nullptr,
                                       c->n_sm, st, err, sizeof err);
      if (head && have_logit) *have_logit = true;
      if (e != cudaSuccess)
        return fail(c, SMLM_ERR_CUDA, "conv_umma: %s %s", cudaGetErrorString(e), err);
    } else {
      CK(c, launch_conv_direct(c->dt, c->act[cur], c->act[cur ^ 1], s, L.dil, L.w_direct, L.bias, st));
    }
    c->launches++;
    if ((tr = time_end(c, e1, st)) != SMLM_OK) return tr;
    // the frames of this launch set have been consumed once the first layer has run
    if (after_stem && fuse_stem && l == 0) CK(c, cudaEventRecord(after_stem, st));
    cur ^= 1;
    if (trunk_dump) {
      CK(c, launch_dump_act(c->dt, c->act[cur], s, trunk_dump + (l + 1) * dump_level_stride,
                            dump_view_stride, st));
      c->launches++;
    }
  }
  *result_buf = cur;
  return SMLM_OK;
}

smlm_status setup_camera(smlm_ctx* c, const smlm_camera_params* cam, int H, int W, cudaStream_t st,
                         NormParams* np) {
  np->offset = cam->offset;
  np->gain = cam->gain;
  np->norm_scale = c->d.norm_scale;
  np->offset_map = nullptr;
  np->gain_map = nullptr;
  if ((cam->offset_map == nullptr) != (cam->gain_map == nullptr))
    return fail(c, SMLM_ERR_INVALID_ARG, "offset_map and gain_map must both be given or both be NULL");
  if (!cam->offset_map) {
    if (!(cam->gain > 0.0f)) return fail(c, SMLM_ERR_INVALID_ARG, "camera gain must be > 0");
    return SMLM_OK;
  }
  size_t n = (size_t)H * W;
  const float* src[2] = {cam->offset_map, cam->gain_map};
  const float* dst[2] = {nullptr, nullptr};
  bool need_copy = classify(src[0]) != PTR_DEVICE || classify(src[1]) != PTR_DEVICE;
  if (need_copy) {
    if (n > c->cam_elems) {
      if (c->cam_off) cudaFree(c->cam_off);
      if (c->cam_gain) cudaFree(c->cam_gain);
      c->cam_off = c->cam_gain = nullptr;
      c->cam_elems = 0;
      CK(c, cudaMalloc(&c->cam_off, n * sizeof(float)));
      CK(c, cudaMalloc(&c->cam_gain, n * sizeof(float)));
      c->cam_elems = n;
    }
    CK(c, cudaMemcpyAsync(c->cam_off, src[0], n * sizeof(float), cudaMemcpyDefault, st));
    CK(c, cudaMemcpyAsync(c->cam_gain, src[1], n * sizeof(float), cudaMemcpyDefault, st));
    dst[0] = c->cam_off;
    dst[1] = c->cam_gain;
  } else {
    dst[0] = src[0];
    dst[1] = src[1];
  }
  np->offset_map = dst[0];
  np->gain_map = dst[1];
  return SMLM_OK;
}

HeadParams head_params(const smlm_ctx* c, const smlm_camera_params* cam, float threshold) {
  HeadParams hp;
  hp.n_h = c->d.head_channels;
  if (threshold <= 0.0f) hp.lthr = -INFINITY;
  else if (threshold >= 1.0f) hp.lthr = INFINITY;
  else hp.lthr = (float)std::log((double)threshold / (1.0 - (double)threshold));
  hp.xy_scale = c->d.xy_scale;
  hp.z_scale_nm = c->d.z_scale_nm;
  hp.photon_scale = c->d.photon_scale;
  hp.bg_scale = c->d.bg_scale;
  hp.pixel_size_nm = cam->pixel_size_nm;
  return hp;
}

// contiguous ranges of tile indices whose windows have the same extent
struct Range { int t0, n, ext; };
std::vector<Range> tile_classes(int F, int tile, int halo) {
  std::vector<Range> out;
  int T = (F + tile - 1) / tile;
  for (int t = 0; t < T; ++t) {
    int lo = std::max(0, t * tile - halo), hi = std::min(F, (t + 1) * tile + halo);
    int ext = hi - lo;
    if (!out.empty() && out.back().ext == ext) out.back().n++;
    else out.push_back({t, 1, ext});
  }
  return out;
}

size_t elt_size(const smlm_ctx* c) { return c->bf16 ? 2 : 4; }

// out_count may be pageable host memory: a D2H copy into it would block the host, so the
// count goes to the ctx's pinned word and a stream-ordered host function forwards it.
struct CountCopy { int64_t* dst; const unsigned long long* src; };
void CUDART_CB count_cb(void* p) {
  CountCopy* cc = static_cast<CountCopy*>(p);
  *cc->dst = (int64_t)*cc->src;
  delete cc;
}
smlm_status store_count(smlm_ctx* c, const unsigned long long* counter, int64_t* out_count,
                        cudaStream_t st) {
  CK(c, cudaMemcpyAsync(c->h_count, counter, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  CountCopy* cc = new (std::nothrow) CountCopy{out_count, c->h_count};
  if (!cc) return fail(c, SMLM_ERR_OOM, "host allocation failed");
  cudaError_t e = cudaLaunchHostFunc(st, count_cb, cc);
  if (e != cudaSuccess) {
    delete cc;
    return fail(c, SMLM_ERR_CUDA, "cudaLaunchHostFunc: %s", cudaGetErrorString(e));
  }
  return SMLM_OK;
}

int auto_micro_batch(const smlm_ctx* c, int Hw, int Ww) {
  if (c->d.micro_batch > 0) return c->d.micro_batch;
  // Measured on B200 (round-1 micro-batch sweep; profiles/bench_r2.md): keeping the two
  // ping-pong maps L2-resident (7 frames of 256x256x48) is SLOWER than streaming large
  // micro-batches from HBM - per-launch overheads (prologue, weight load, tail) and the halo
  // steps per work range weigh more than the DRAM traffic.  So: up to 128 views per launch
  // (round 2 sweep: 64 -> 128 views is +1.7 % on cfg 1, flat beyond), bounded by 1.5 GB per
  // activation buffer.
  size_t per_view = (size_t)Hw * Ww * c->d.channels * elt_size(c);
  size_t b = ((size_t)1536 << 20) / std::max<size_t>(per_view, 1);
  return (int)std::min<size_t>(std::max<size_t>(b, 1), 128);
}

}  // namespace

extern "C" {

smlm_status smlm_create(const smlm_net_desc* desc, const void* weights, smlm_ctx** out_ctx) {
  if (out_ctx) *out_ctx = nullptr;
  if (!desc || !weights || !out_ctx) return fail(nullptr, SMLM_ERR_INVALID_ARG, "NULL argument");
  if (desc->struct_size != sizeof(smlm_net_desc) || desc->version != SMLM_ABI_VERSION)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "smlm_net_desc size/version mismatch");
  const int C = desc->channels, L = desc->n_layers, nh = desc->head_channels;
  if (C < 16 || C > 64 || C % 16) return fail(nullptr, SMLM_ERR_INVALID_ARG, "channels must be 16, 32, 48 or 64");
  if (L < 0 || L > SMLM_MAX_LAYERS) return fail(nullptr, SMLM_ERR_INVALID_ARG, "n_layers out of range");
  if (nh != 5 && nh != 6) return fail(nullptr, SMLM_ERR_INVALID_ARG, "head_channels must be 5 or 6");
  if (desc->precision != SMLM_FP32 && desc->precision != SMLM_BF16 && desc->precision != SMLM_FP16)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "bad precision");
  if (desc->in_frames != 0 && desc->in_frames != 1 && desc->in_frames != 3)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "in_frames must be 1 or 3");
  if (desc->tile_merge != SMLM_TILE_MERGE_NONE && desc->tile_merge != SMLM_TILE_MERGE_ROW)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "bad tile_merge");
  if (desc->stem_impl < SMLM_STEM_AUTO || desc->stem_impl > SMLM_STEM_CUDA_CORES)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "bad stem_impl");
  if (desc->conv_impl < SMLM_CONV_AUTO || desc->conv_impl > SMLM_CONV_DIRECT)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "bad conv_impl");
  if (desc->precision == SMLM_FP32 && desc->conv_impl == SMLM_CONV_TCGEN05)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "the tcgen05 kernel needs a 16-bit precision");
  for (int l = 0; l < L; ++l)
    if (desc->dilations[l] < 1 || desc->dilations[l] > 16)
      return fail(nullptr, SMLM_ERR_INVALID_ARG, "dilations must be in 1..16");
  if (!(desc->norm_scale > 0.0f)) return fail(nullptr, SMLM_ERR_INVALID_ARG, "norm_scale must be > 0");
  if (desc->tile < 0 || desc->micro_batch < 0 || desc->writeback_frames < 0)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "negative tile / micro_batch / writeback_frames");
  if (desc->fusion < SMLM_FUSE_AUTO || desc->fusion > SMLM_FUSE_PAIRS_1CTA)
    return fail(nullptr, SMLM_ERR_INVALID_ARG, "bad fusion");

  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return fail(nullptr, SMLM_ERR_UNSUPPORTED_DEVICE, "no CUDA device");
  }
  if (prop.major != 10)
    return fail(nullptr, SMLM_ERR_UNSUPPORTED_DEVICE, "device %s is sm_%d%d; this library is sm_100a only",
                prop.name, prop.major, prop.minor);

  smlm_ctx* c = new (std::nothrow) smlm_ctx;
  if (!c) return fail(nullptr, SMLM_ERR_OOM, "host allocation failed");
  c->d = *desc;
  c->bf16 = desc->precision != SMLM_FP32;
  c->dt = desc->precision == SMLM_BF16 ? ACT_BF16 : (desc->precision == SMLM_FP16 ? ACT_F16 : ACT_F32);
  c->in_frames = desc->in_frames == 3 ? 3 : 1;
  c->use_umma = c->bf16 && desc->conv_impl != SMLM_CONV_DIRECT;
  c->fuse = desc->fusion != SMLM_FUSE_NONE;
  c->fuse_stem = desc->fusion == SMLM_FUSE_ALL;
  c->fuse_pairs = desc->fusion == SMLM_FUSE_AUTO || desc->fusion == SMLM_FUSE_ALL || desc->fusion == SMLM_FUSE_PAIRS_1CTA;
  c->pair_cg2 = desc->fusion != SMLM_FUSE_PAIRS_1CTA;
  c->n_sm = prop.multiProcessorCount;
  c->l2_bytes = (size_t)prop.l2CacheSize;
  c->radius = 1;
  for (int l = 0; l < L; ++l) c->radius += desc->dilations[l];

  smlm_status st = SMLM_OK;
  auto upload = [&](const std::vector<float>& h, float** d) -> smlm_status {
    CK(nullptr, cudaMalloc(d, h.size() * sizeof(float)));
    CK(nullptr, cudaMemcpy(*d, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice));
    return SMLM_OK;
  };
  auto body = [&]() -> smlm_status {
    const float* w = static_cast<const float*>(weights);
    const int IF = c->in_frames, T9 = 9 * IF;  // stem W[C][IF][3][3] -> [IF * 9][C] (channel, ky, kx) major
    std::vector<float> tmp((size_t)T9 * C);
    for (int co = 0; co < C; ++co)
      for (int t = 0; t < T9; ++t) tmp[(size_t)t * C + co] = w[(size_t)co * T9 + t];
    if ((st = upload(tmp, &c->w_stem)) != SMLM_OK) return st;
    if (IF == 1)
      for (int t = 0; t < 9; ++t)
        for (int co = 0; co < C; ++co) c->stem_args.w[t][co] = tmp[t * C + co];
    for (int co = 0; co < C; ++co) c->stem_args.b[co] = w[T9 * C + co];
    {
      const bool can = c->dt != ACT_F32 && c->in_frames == 1 && stem_umma_supports(C, 1);
      if (desc->stem_impl == SMLM_STEM_TENSOR && !can)
        return fail(nullptr, SMLM_ERR_INVALID_ARG, "SMLM_STEM_TENSOR needs 16-bit precision, in_frames = 1, channels 16/32/48/64");
      c->stem_tensor = can && desc->stem_impl == SMLM_STEM_TENSOR;
      if (c->stem_tensor) {
        std::vector<uint8_t> sp(stem_umma_packed_bytes(C));
        stem_umma_pack_host(C, tmp.data(), w + T9 * C, sp.data(), c->dt == ACT_F16);
        CK(nullptr, cudaMalloc(&c->w_stem_umma, sp.size()));
        CK(nullptr, cudaMemcpy(c->w_stem_umma, sp.data(), sp.size(), cudaMemcpyHostToDevice));
        for (int co = 0; co < C; ++co) c->stem_lc.bias[co] = w[T9 * C + co];
      }
    }
    if ((st = upload(std::vector<float>(w + T9 * C, w + (T9 + 1) * C), &c->b_stem)) != SMLM_OK) return st;
    w += (T9 + 1) * C;
    c->layers.resize(L);
    std::vector<float> wd((size_t)9 * C * C);
    std::vector<uint8_t> pack(c->use_umma ? umma_packed_weight_bytes(C) : 0);
    for (int l = 0; l < L; ++l) {
      Layer& Ly = c->layers[l];
      Ly.dil = desc->dilations[l];
      for (int co = 0; co < C; ++co)
        for (int ci = 0; ci < C; ++ci)
          for (int t = 0; t < 9; ++t) {
            float v = w[((size_t)co * C + ci) * 9 + t];
            wd[((size_t)t * C + ci) * C + co] = round_to_act(v, c->dt);
          }
      if ((st = upload(wd, &Ly.w_direct)) != SMLM_OK) return st;
      if ((st = upload(std::vector<float>(w + (size_t)9 * C * C, w + (size_t)9 * C * C + C), &Ly.bias)) != SMLM_OK)
        return st;
      for (int co = 0; co < C; ++co) Ly.lc.bias[co] = w[(size_t)9 * C * C + co];
      if (c->use_umma) {
        umma_pack_weights_host(C, w, pack.data(), c->dt == ACT_F16);
        CK(nullptr, cudaMalloc(&Ly.w_umma, pack.size()));
        CK(nullptr, cudaMemcpy(Ly.w_umma, pack.data(), pack.size(), cudaMemcpyHostToDevice));
      }
      w += (size_t)9 * C * C + C;
    }
    if ((st = upload(std::vector<float>(w, w + nh * C), &c->w_head)) != SMLM_OK) return st;
    for (int h = 0; h < nh; ++h) {
      for (int ci = 0; ci < C; ++ci) c->head_args.w[ci][h] = w[h * C + ci];
      c->head_args.b[h] = w[nh * C + h];
    }
    c->head_args.n_h = nh;
    if ((st = upload(std::vector<float>(w + nh * C, w + nh * C + nh), &c->b_head)) != SMLM_OK) return st;
    CK(nullptr, conv_direct_init(C));
    CK(nullptr, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    CK(nullptr, cudaStreamCreateWithFlags(&c->wb_stream, cudaStreamNonBlocking));
    for (int i = 0; i < kSlots; ++i) {
      CK(nullptr, cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming));
      CK(nullptr, cudaEventCreateWithFlags(&c->ev_consumed[i], cudaEventDisableTiming));
    }
    for (int i = 0; i < kFirstParts; ++i) {
      CK(nullptr, cudaEventCreateWithFlags(&c->ev_part[i], cudaEventDisableTiming));
    }
    CK(nullptr, cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
    CK(nullptr, cudaEventCreateWithFlags(&c->ev_batch, cudaEventDisableTiming));
    for (int i = 0; i < kSnapRing; ++i)
      CK(nullptr, cudaEventCreateWithFlags(&c->ev_wb[i], cudaEventDisableTiming));
    CK(nullptr, cudaMalloc(&c->counters, kCounterWords * sizeof(unsigned long long)));
    CK(nullptr, cudaMemset(c->counters, 0, kCounterWords * sizeof(unsigned long long)));
    CK(nullptr, cudaMallocHost(&c->h_count, sizeof(unsigned long long)));
    *c->h_count = 0;
    return SMLM_OK;
  };
  st = body();
  if (st != SMLM_OK) {
    smlm_destroy(c);
    return st;
  }
  *out_ctx = c;
  return SMLM_OK;
}

void smlm_destroy(smlm_ctx* c) {
  if (!c) return;
  cudaDeviceSynchronize();
  if (c->w_stem_umma) cudaFree(c->w_stem_umma);
  cudaFree(c->w_stem); cudaFree(c->b_stem); cudaFree(c->w_head); cudaFree(c->b_head);
  for (auto& L : c->layers) { cudaFree(L.w_direct); cudaFree(L.w_umma); cudaFree(L.bias); }
  cudaFree(c->act[0]); cudaFree(c->act[1]); cudaFree(c->logit); cudaFree(c->cand); cudaFree(c->slots);
  cudaFree(c->em_dev);
  cudaFree(c->counters); cudaFree(c->cam_off); cudaFree(c->cam_gain);
  if (c->h_count) cudaFreeHost(c->h_count);
  for (int i = 0; i < kSlots; ++i) {
    if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
    if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]);
  }
  for (int i = 0; i < kFirstParts; ++i) {
    if (c->ev_part[i]) cudaEventDestroy(c->ev_part[i]);
  }
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  if (c->ev_batch) cudaEventDestroy(c->ev_batch);
  for (int i = 0; i < kSnapRing; ++i)
    if (c->ev_wb[i]) cudaEventDestroy(c->ev_wb[i]);
  for (auto e : c->tev) cudaEventDestroy(e);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->wb_stream) cudaStreamDestroy(c->wb_stream);
  cudaGetLastError();
  delete c;
}

const char* smlm_last_error(const smlm_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int64_t smlm_launch_count(const smlm_ctx* c) { return c ? c->launches : 0; }

smlm_status smlm_kernel_timing(smlm_ctx* c, int32_t enable) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  c->timing = enable != 0;
  c->tev_used = 0;
  return SMLM_OK;
}

smlm_status smlm_kernel_time_ms(smlm_ctx* c, int32_t kind, double* total_ms, int64_t* launches) {
  if (!c || !total_ms || !launches || kind < SMLM_KERNEL_STEM || kind > SMLM_KERNEL_CONV_PAIR)
    return SMLM_ERR_INVALID_ARG;
  double tot = 0.0;
  int64_t n = 0;
  for (size_t i = 0; i + 1 < c->tev_used; i += 2) {
    if (c->tev_kind[i / 2] != kind) continue;
    CK(c, cudaEventSynchronize(c->tev[i + 1]));
    float ms = 0.f;
    CK(c, cudaEventElapsedTime(&ms, c->tev[i], c->tev[i + 1]));
    tot += ms;
    ++n;
  }
  *total_ms = tot;
  *launches = n;
  return SMLM_OK;
}

smlm_status smlm_check(smlm_ctx* c) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, SMLM_ERR_CUDA, "pending CUDA error: %s", cudaGetErrorString(e));
  if (*c->h_count > c->last_capacity)
    return fail(c, SMLM_ERR_OVERFLOW, "found %llu emitters, capacity %llu", *c->h_count, c->last_capacity);
  return SMLM_OK;
}

}  // extern "C"

namespace {

// One smlm_localize call, cut into begin / frames / end so that the frames may arrive in
// pieces (smlm_localize_ring feeds one ring chunk at a time; frame indices stay global).
struct Call {
  smlm_ctx* c = nullptr;
  cudaStream_t st = nullptr;
  int H = 0, W = 0, C = 0;
  int64_t n_total = 0;     // frames of the whole call
  NormParams np{};
  HeadParams hp{};
  bool tiled = false;
  int tile = 0, halo = 0, mb = 0, F = 1;
  int tile_w = 0;  // SMLM_TILE_MERGE_ROW: the frame width (one window per tile row), else 0
  std::vector<Range> ycls, xcls;
  smlm_emitter* out = nullptr;   // caller's list
  smlm_emitter* list = nullptr;  // where K3 appends (== out, or the ctx's device list)
  unsigned long long capacity = 0;
  bool host_out = false;
  int wbf = 256;
  int64_t n_flush = 0, chunk = 0;
};

smlm_status call_flush(Call& k) {
  smlm_ctx* c = k.c;
  unsigned long long* counter = c->counters;
  unsigned long long* snap_ring = c->counters + 2;
  const int64_t i = k.n_flush;
  // the word snap[i % R] was read by flushes i - R (upper end) and i - R + 1 (lower end)
  if (i >= kSnapRing) CK(c, cudaStreamWaitEvent(k.st, c->ev_wb[(i + 1) % kSnapRing], 0));
  // records below the snapshot are complete: every K3 that wrote them precedes it on `st`
  CK(c, launch_snapshot(counter, k.capacity, snap_ring + i % kSnapRing, k.st));
  CK(c, cudaEventRecord(c->ev_batch, k.st));
  CK(c, cudaStreamWaitEvent(c->wb_stream, c->ev_batch, 0));
  const unsigned long long* lo = i == 0 ? c->counters + 1 : snap_ring + (i - 1) % kSnapRing;
  CK(c, launch_flush_emitters(k.list, k.out, lo, snap_ring + i % kSnapRing, c->wb_stream));
  CK(c, cudaEventRecord(c->ev_wb[i % kSnapRing], c->wb_stream));
  c->launches += 2;
  ++k.n_flush;
  return SMLM_OK;
}

smlm_status call_begin(Call& k, smlm_ctx* c, int64_t n, int32_t H, int32_t W, const smlm_camera_params* cam,
                       float threshold, smlm_emitter* out, int64_t* out_count, bool host_frames,
                       int64_t max_piece, cudaStream_t st) {
  if (!cam || !out_count) return fail(c, SMLM_ERR_INVALID_ARG, "NULL camera / out_count");
  if (n < 0 || H < 1 || W < 1 || (int64_t)H * W > (int64_t)1 << 30 || n > INT32_MAX)
    return fail(c, SMLM_ERR_INVALID_ARG, "bad n_frames / H / W");
  if (*out_count < 0) return fail(c, SMLM_ERR_INVALID_ARG, "negative capacity");
  if (!(threshold == threshold)) return fail(c, SMLM_ERR_INVALID_ARG, "threshold is NaN");
  if (!(cam->pixel_size_nm > 0.0f)) return fail(c, SMLM_ERR_INVALID_ARG, "pixel_size_nm must be > 0");
  k.c = c;
  k.st = st;
  k.H = H;
  k.W = W;
  k.C = c->d.channels;
  k.n_total = n;
  k.capacity = (unsigned long long)*out_count;
  k.out = out;
  if (k.capacity > 0 && !out) return fail(c, SMLM_ERR_INVALID_ARG, "NULL out_emitters with capacity > 0");
  PtrKind ok = PTR_DEVICE;
  if (k.capacity > 0) {
    ok = classify(out);
    if (ok == PTR_OTHER)
      return fail(c, SMLM_ERR_INVALID_ARG, "out_emitters must be device or pinned host memory");
  }
  smlm_status r = setup_camera(c, cam, H, W, st, &k.np);
  if (r != SMLM_OK) return r;
  k.hp = head_params(c, cam, threshold);

  // ---- geometry: launch sets (all views of a set share one window size)
  k.tile = c->d.tile;
  k.tiled = k.tile > 0 && (k.tile < H || k.tile < W);
  k.halo = c->radius + 1;  // maps need `radius`; the 3x3 test reads one more pixel
  // SMLM_TILE_MERGE_ROW: the cores of one tile row share one window (core = tile rows x W)
  k.tile_w = (k.tiled && c->d.tile_merge == SMLM_TILE_MERGE_ROW && k.tile < H) ? W : 0;
  if (k.tiled && c->d.tile_merge == SMLM_TILE_MERGE_ROW && k.tile >= H) k.tiled = false;  // one row of tiles = the frame
  if (k.tiled) {
    k.ycls = tile_classes(H, k.tile, k.halo);
    if (k.tile_w) k.xcls.push_back({0, 1, W});
    else k.xcls = tile_classes(W, k.tile, k.halo);
  } else {
    k.ycls.push_back({0, 1, H});
    k.xcls.push_back({0, 1, W});
  }
  int maxHw = 0, maxWw = 0;
  for (auto& a : k.ycls) maxHw = std::max(maxHw, a.ext);
  for (auto& a : k.xcls) maxWw = std::max(maxWw, a.ext);
  k.mb = auto_micro_batch(c, maxHw, maxWw);  // views per launch
  // frames per chunk: whole frames -> one view each; tiles -> as many frames as keep the
  // largest launch set (all tiles of one window class, times the frames) within mb views
  int tiles_per_frame = 0;
  for (auto& a : k.ycls)
    for (auto& b : k.xcls) tiles_per_frame = std::max(tiles_per_frame, a.n * b.n);
  const int64_t piece = std::max<int64_t>(1, std::min<int64_t>(std::max<int64_t>(n, 1), max_piece));
  k.F = (int)std::max<int64_t>(1, std::min<int64_t>(k.tiled ? k.mb / std::max(tiles_per_frame, 1) : k.mb, piece));
  size_t need = 0;
  for (auto& a : k.ycls)
    for (auto& b : k.xcls) {
      int nv = k.tiled ? std::max(1, std::min(k.mb, k.F * a.n * b.n)) : k.F;
      need = std::max(need, (size_t)nv * a.ext * b.ext * k.C * elt_size(c));
    }
  if ((r = ensure_act(c, need)) != SMLM_OK) return r;

  const size_t frame_elems = (size_t)H * W;
  if (host_frames && n > 0) {
    size_t se = (size_t)(k.F + (c->in_frames == 3 ? 2 : 0)) * frame_elems;  // + frames f0-1 and f0+nf
    if (se > c->slot_elems) {
      CK(c, cudaDeviceSynchronize());  // a previous call may still read the old slots
      if (c->slots) cudaFree(c->slots);
      c->slots = nullptr;
      c->slot_elems = 0;
      CK(c, cudaMalloc(&c->slots, kSlots * se * sizeof(uint16_t)));
      c->slot_elems = se;
      for (int i = 0; i < kSlots; ++i) c->slot_used[i] = false;
    }
  }
  k.list = out;
  if (ok == PTR_HOST_PINNED && k.capacity > 0) {
    if (k.capacity > c->em_cap) {
      CK(c, cudaDeviceSynchronize());
      if (c->em_dev) cudaFree(c->em_dev);
      c->em_dev = nullptr;
      c->em_cap = 0;
      CK(c, cudaMalloc(&c->em_dev, k.capacity * sizeof(smlm_emitter)));
      c->em_cap = k.capacity;
    }
    k.list = c->em_dev;
  }
  CK(c, cudaMemsetAsync(c->counters, 0, kCounterWords * sizeof(unsigned long long), st));
  c->last_capacity = k.capacity;
  if (host_frames) {
    CK(c, cudaEventRecord(c->ev_start, st));
    CK(c, cudaStreamWaitEvent(c->copy_stream, c->ev_start, 0));
  }
  k.host_out = (ok == PTR_HOST_PINNED && k.capacity > 0);
  // 0 = library default: flush every 256 frames, so that only the last batch's D2H is exposed
  k.wbf = c->d.writeback_frames > 0 ? c->d.writeback_frames : 256;
  return SMLM_OK;
}

// frames [f_first, f_first + n) of the call, stored at `frames` (pinned host or device).
// *copied (may be NULL): an event of the copy stream to record once the last H2D copy of
// this piece has been enqueued (the ring loader releases its slot when it fires).
smlm_status call_frames(Call& k, const uint16_t* frames, int64_t f_first, int64_t n, bool host_frames) {
  smlm_ctx* c = k.c;
  cudaStream_t st = k.st;
  const int H = k.H, W = k.W, C = k.C, F = k.F;
  const size_t frame_elems = (size_t)H * W;
  unsigned long long* counter = c->counters;
  smlm_status r = SMLM_OK;
  for (int64_t f0 = f_first; f0 < f_first + n; f0 += F, ++k.chunk) {
    const int nf = (int)std::min<int64_t>(F, f_first + n - f0);
    const uint16_t* dev_frames = frames;
    int frame_base = (int)f_first;
    int slot = -1, parts = 1;
    if (host_frames) {
      // P1: the preload ring.  Copy chunk k into slot k % kSlots on the copy stream as soon
      // as the stem of chunk k - kSlots has consumed it; compute waits for the copy only.
      slot = (int)(k.chunk % kSlots);
      if (c->slot_used[slot]) CK(c, cudaStreamWaitEvent(c->copy_stream, c->ev_consumed[slot], 0));
      uint16_t* dst = c->slots + (size_t)slot * c->slot_elems;
      // temporal context: the chunk's neighbours f0-1 and f0+nf travel with it (the call's
      // frames are all in `frames`: smlm_localize_ring refuses in_frames = 3)
      int64_t c0 = f0, c1 = f0 + nf;
      if (c->in_frames == 3) {
        c0 = std::max<int64_t>(f0 - 1, f_first);
        c1 = std::min<int64_t>(f0 + nf + 1, f_first + n);
      }
      // the first chunk of a call has nothing to hide behind: it travels in kFirstParts copies and
      // K1 starts on the first (run_trunk, stem_parts)
      parts = (k.chunk == 0 && !k.tiled && c->in_frames == 1 && !c->fuse_stem && nf >= 16 * kFirstParts) ? kFirstParts : 1;
      for (int q = 0; q < parts; ++q) {
        const int64_t a = c0 + (c1 - c0) * q / parts, b = c0 + (c1 - c0) * (q + 1) / parts;
        CK(c, cudaMemcpyAsync(dst + (size_t)(a - c0) * frame_elems, frames + (size_t)(a - f_first) * frame_elems,
                              (size_t)(b - a) * frame_elems * 2, cudaMemcpyHostToDevice, c->copy_stream));
        if (parts > 1) CK(c, cudaEventRecord(c->ev_part[q], c->copy_stream));
      }
      CK(c, cudaEventRecord(c->ev_copied[slot], c->copy_stream));
      if (parts == 1) CK(c, cudaStreamWaitEvent(st, c->ev_copied[slot], 0));
      c->slot_used[slot] = true;
      dev_frames = dst;
      frame_base = (int)c0;
    }
    // launch sets of this chunk
    struct Set { ViewSet vs; ActShape s; };
    std::vector<Set> sets;
    if (!k.tiled) {
      ViewSet vs{(int)f0, H, W, 0, 0, 0, 1, 0, 1, 0, c->in_frames, (int)k.n_total};
      sets.push_back({vs, ActShape{nf, C, H, W}});
    } else {
      for (auto& a : k.ycls)
        for (auto& b : k.xcls) {
          // all tiles of the class for the nf frames of the chunk in one set if that is at
          // most mb views, else sub-blocks of tiles (times the frames) of at most mb views
          const int per_frame = std::max(1, k.mb / nf);
          int bx = std::min(b.n, per_frame), by = std::max(1, std::min(a.n, per_frame / bx));
          for (int ty = a.t0; ty < a.t0 + a.n; ty += by)
            for (int tx = b.t0; tx < b.t0 + b.n; tx += bx) {
              int ny = std::min(by, a.t0 + a.n - ty), nx = std::min(bx, b.t0 + b.n - tx);
              ViewSet vs{(int)f0, H, W, k.tile, k.halo, ty, ny, tx, nx, k.tile_w, c->in_frames, (int)k.n_total};
              sets.push_back({vs, ActShape{nf * ny * nx, C, a.ext, b.ext}});
            }
        }
    }
    for (size_t si = 0; si < sets.size(); ++si) {
      int res = 0;
      cudaEvent_t after_stem = (slot >= 0 && si + 1 == sets.size()) ? c->ev_consumed[slot] : nullptr;
      bool have_logit = false, from_act = false;
      r = run_trunk(c, dev_frames, frame_base, sets[si].vs, sets[si].s, k.np, st, &res, nullptr, 0, 0,
                    after_stem, true, k.hp.lthr, &have_logit, &from_act, parts);
      if (r != SMLM_OK) return r;
      cudaEvent_t te = nullptr;
      if ((r = time_begin(c, SMLM_KERNEL_POST, st, &te)) != SMLM_OK) return r;
      if (have_logit && from_act)
        CK(c, launch_post_logits_act(c->dt, c->logit, c->act[res], sets[si].s, sets[si].vs, c->w_head, c->b_head, k.hp,
                                     k.list, counter, k.capacity, st));
      else if (have_logit)
        CK(c, launch_post_logits(c->logit, c->cand, sets[si].s, sets[si].vs, k.hp, k.list, counter, k.capacity, st));
      else
        CK(c, launch_head_post(c->dt, c->act[res], sets[si].s, sets[si].vs, c->w_head, c->b_head, k.hp,
                               k.list, counter, k.capacity, st));
      c->launches++;
      if ((r = time_end(c, te, st)) != SMLM_OK) return r;
    }
    if (k.host_out && k.wbf > 0) {
      int64_t done = f0 + nf;
      if (done < k.n_total && done / k.wbf != f0 / k.wbf) {
        if ((r = call_flush(k)) != SMLM_OK) return r;
      }
    }
  }
  return SMLM_OK;
}

smlm_status call_end(Call& k, int64_t* out_count) {
  smlm_ctx* c = k.c;
  smlm_status r;
  if (k.host_out) {
    if ((r = call_flush(k)) != SMLM_OK) return r;
  }
  if (k.n_flush > 0) CK(c, cudaStreamWaitEvent(k.st, c->ev_wb[(k.n_flush - 1) % kSnapRing], 0));
  return store_count(c, c->counters, out_count, k.st);
}

}  // namespace

extern "C" {

smlm_status smlm_localize(smlm_ctx* c, const uint16_t* frames, int64_t n, int32_t H, int32_t W,
                          const smlm_camera_params* cam, float threshold, smlm_emitter* out,
                          int64_t* out_count, void* cuda_stream) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  PtrKind fk = PTR_DEVICE;
  if (n > 0) {
    if (!frames) return fail(c, SMLM_ERR_INVALID_ARG, "NULL frames");
    fk = classify(frames);
    if (fk == PTR_OTHER)
      return fail(c, SMLM_ERR_INVALID_ARG,
                  "frames_u16 must be pinned host memory (the preload ring) or device memory");
  }
  Call k;
  smlm_status r = call_begin(k, c, n, H, W, cam, threshold, out, out_count, fk == PTR_HOST_PINNED,
                             INT64_MAX, static_cast<cudaStream_t>(cuda_stream));
  if (r != SMLM_OK) return r;
  if ((r = call_frames(k, frames, 0, n, fk == PTR_HOST_PINNED)) != SMLM_OK) return r;
  return call_end(k, out_count);
}

namespace {
struct RingRelease { smlm_ring* r; int64_t k; };
void CUDART_CB ring_release_cb(void* p) {
  RingRelease* rr = static_cast<RingRelease*>(p);
  ring_release_chunk(rr->r, rr->k);
  delete rr;
}
}  // namespace

smlm_status smlm_localize_ring(smlm_ctx* c, smlm_ring* ring, const smlm_camera_params* cam, float threshold,
                               smlm_emitter* out, int64_t* out_count, void* cuda_stream) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  if (!ring) return fail(c, SMLM_ERR_INVALID_ARG, "NULL ring");
  if (!ring->pinned) return fail(c, SMLM_ERR_INVALID_ARG, "the ring is pageable (SMLM_RING_PAGEABLE is for tests)");
  if (c->in_frames == 3)
    return fail(c, SMLM_ERR_INVALID_ARG, "in_frames = 3 needs the whole stack (smlm_localize): ring chunks have no neighbours");
  {
    std::lock_guard<std::mutex> lk(ring->mu);
    if (ring->by_hand > 0)
      return fail(c, SMLM_ERR_INVALID_ARG, "chunks taken with smlm_ring_acquire have not been released");
  }
  ring_rewind(ring);  // waits for the previous pass's copies to have drained their slots
  Call k;
  smlm_status r = call_begin(k, c, ring->n_frames, ring->H, ring->W, cam, threshold, out, out_count, true,
                             ring->chunk_frames, static_cast<cudaStream_t>(cuda_stream));
  if (r != SMLM_OK) return r;
  for (int64_t ck = 0; ck < ring->n_chunks; ++ck) {
    const uint16_t* p = ring_wait_chunk(ring, ck);  // blocks on the disk only
    if (!p) return fail(c, SMLM_ERR_INVALID_ARG, "frame file: %s", ring->error.c_str());
    if ((r = call_frames(k, p, ck * ring->chunk_frames, ring->frames_of(ck), true)) != SMLM_OK) {
      cudaStreamSynchronize(c->copy_stream);  // a failed call must not leave a chunk handed out
      ring_release_chunk(ring, ck);
      return r;
    }
    // the slot goes back to the readers when the copy stream has drained this chunk's copies
    RingRelease* rr = new (std::nothrow) RingRelease{ring, ck};
    if (!rr) {
      cudaStreamSynchronize(c->copy_stream);
      ring_release_chunk(ring, ck);
      return fail(c, SMLM_ERR_OOM, "host allocation failed");
    }
    cudaError_t e = cudaLaunchHostFunc(c->copy_stream, ring_release_cb, rr);
    if (e != cudaSuccess) {
      delete rr;
      cudaStreamSynchronize(c->copy_stream);
      ring_release_chunk(ring, ck);
      return fail(c, SMLM_ERR_CUDA, "cudaLaunchHostFunc: %s", cudaGetErrorString(e));
    }
  }
  return call_end(k, out_count);
}

smlm_status smlm_debug_forward_maps(smlm_ctx* c, const uint16_t* frames, int64_t n, int32_t H,
                                    int32_t W, const smlm_camera_params* cam, float* maps,
                                    float* trunk, void* cuda_stream) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  if (!cam || !maps || (n > 0 && !frames) || n < 0 || H < 1 || W < 1 || n > INT32_MAX)
    return fail(c, SMLM_ERR_INVALID_ARG, "bad argument");
  if (classify(maps) != PTR_DEVICE || (trunk && classify(trunk) != PTR_DEVICE))
    return fail(c, SMLM_ERR_INVALID_ARG, "maps / trunk must be device memory");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  PtrKind fk = n > 0 ? classify(frames) : PTR_DEVICE;
  if (fk == PTR_OTHER) return fail(c, SMLM_ERR_INVALID_ARG, "frames must be pinned host or device memory");
  NormParams np;
  smlm_status r = setup_camera(c, cam, H, W, st, &np);
  if (r != SMLM_OK) return r;
  const int C = c->d.channels, L = c->d.n_layers, nh = c->d.head_channels;
  const int mb = auto_micro_batch(c, H, W);
  const size_t px = (size_t)H * W;
  if ((r = ensure_act(c, (size_t)std::min<int64_t>(mb, std::max<int64_t>(n, 1)) * px * C * elt_size(c))) != SMLM_OK)
    return r;
  uint16_t* tmp = nullptr;
  if (fk == PTR_HOST_PINNED && n > 0) {
    CK(c, cudaMalloc(&tmp, (size_t)n * px * 2));
    cudaError_t e = cudaMemcpyAsync(tmp, frames, (size_t)n * px * 2, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) {
      cudaFree(tmp);
      return fail(c, SMLM_ERR_CUDA, "cudaMemcpyAsync(frames): %s", cudaGetErrorString(e));
    }
    frames = tmp;
  }
  for (int64_t f0 = 0; f0 < n; f0 += mb) {
    int nf = (int)std::min<int64_t>(mb, n - f0);
    ViewSet vs{(int)f0, H, W, 0, 0, 0, 1, 0, 1, 0, c->in_frames, (int)n};
    ActShape s{nf, C, H, W};
    int res = 0;
    float* dump = trunk ? trunk + (size_t)f0 * (L + 1) * px * C : nullptr;
    r = run_trunk(c, frames, 0, vs, s, np, st, &res, dump, (size_t)(L + 1) * px * C, px * C, nullptr, false,
                  0.0f, nullptr);
    if (r != SMLM_OK) break;
    cudaError_t e = launch_head_maps(c->dt, c->act[res], s, c->w_head, c->b_head, nh,
                                     maps + (size_t)f0 * nh * px, st);
    c->launches++;
    if (e != cudaSuccess) {
      r = fail(c, SMLM_ERR_CUDA, "head_maps: %s", cudaGetErrorString(e));
      break;
    }
  }
  if (tmp) {
    cudaStreamSynchronize(st);
    cudaFree(tmp);
  }
  return r;
}

smlm_status smlm_debug_postprocess(smlm_ctx* c, const float* maps, int64_t n, int32_t H, int32_t W,
                                   const smlm_camera_params* cam, float threshold, smlm_emitter* out,
                                   int64_t* out_count, void* cuda_stream) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  if (!cam || !out_count || (n > 0 && !maps) || n < 0 || H < 1 || W < 1 || n > 65535 || *out_count < 0)
    return fail(c, SMLM_ERR_INVALID_ARG, "bad argument");
  const unsigned long long capacity = (unsigned long long)*out_count;
  if (capacity > 0 && (!out || classify(out) != PTR_DEVICE))
    return fail(c, SMLM_ERR_INVALID_ARG, "out_emitters must be device memory here");
  if (n > 0 && classify(maps) != PTR_DEVICE) return fail(c, SMLM_ERR_INVALID_ARG, "maps must be device memory");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const HeadParams hp = head_params(c, cam, threshold);
  CK(c, cudaMemsetAsync(c->counters, 0, kCounterWords * sizeof(unsigned long long), st));
  c->last_capacity = capacity;
  CK(c, launch_post_from_maps(maps, (int)n, H, W, hp, out, c->counters, capacity, st));
  c->launches++;
  return store_count(c, c->counters, out_count, st);
}

}  // extern "C"
