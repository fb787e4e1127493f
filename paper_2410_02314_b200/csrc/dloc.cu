// C ABI of the paper's own topology (include/dloc.h): DCD dense blocks of dilated
// convolutions, a two-stage U-Net and DECODE-style heads, driven layer
// by layer over chunk-planar concatenation buffers.  Every step runs in this library's CUDA
// kernels: stem.cu (K1), conv_gen.cu (every other convolution, pooling, up-sampling, detection
// and decode).  No CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/dloc.h"
#include "dloc_internal.cuh"

using namespace smlm;

namespace {

thread_local std::string g_dloc_create_error;

struct GLayer {
  int CI = 0, CO = 0, CO_real = 0, k = 3, d = 1, relu = 1;
  void* wpack = nullptr;     // tensor-core image (16-bit modes, tcgen05 path)
  float* w_direct = nullptr; // [k*k][CI][CO] fp32 (values rounded to the storage type in 16-bit modes)
  float* bias = nullptr;     // [CO]
  // conv_chain.cu (tcgen05 path): one pass per group of `chain_co` output channels - the dense
  // layers (growth 16: one pass), the transitions (one pass of C0), and dec0 (C0 / 16 passes of 16
  // channels: its whole weight image does not fit in shared memory, a 16-channel slice does)
  std::vector<void*> wchain;
  std::vector<LayerConst> lc;  // the bias slices, as kernel parameters
  int chain_co = 0;
};

struct Bufs {
  void *blk[2] = {nullptr, nullptr}, *cat0 = nullptr, *p1 = nullptr, *cat1 = nullptr, *p2 = nullptr, *e2 = nullptr,
       *m1 = nullptr, *m0 = nullptr;
  float* maps = nullptr;
  uint16_t* slots = nullptr;  // two staging slots of mb (+2) frames for pinned-host input
  size_t key_mb = 0, key_H = 0, key_W = 0;
};

}  // namespace

struct dloc_ctx {
  dloc_net_desc d{};
  int dt = ACT_F32;
  int in_frames = 1;
  bool use_umma = false;
  bool use_chain = true;  // dense-block layers through conv_chain.cu (SMLM_CONV_TCGEN05 keeps the generic kernel: the twin)
  int n_sm = 0;
  int CB = 0;
  float *w_stem = nullptr, *b_stem = nullptr;
  std::vector<GLayer> dcd;   // per block: n_dil dense layers + the transition
  GLayer enc1, enc2, dec1, dec0, heads;
  Bufs buf;
  float *cam_off = nullptr, *cam_gain = nullptr;
  size_t cam_elems = 0;
  unsigned long long* counter = nullptr;  // device
  unsigned long long* h_count = nullptr;  // pinned
  unsigned long long last_capacity = 0;
  dloc_emitter* em_dev = nullptr;
  size_t em_cap = 0;
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr}, ev_start = nullptr;
  bool slot_used[2] = {false, false};
  int64_t launches = 0;
  bool timing = false;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> tev;
  size_t tev_used = 0;
  double conv_ms = 0.0;
  int64_t conv_n = 0;
  std::string err;
};

namespace {

smlm_status dfail(dloc_ctx* c, smlm_status st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf;
  else g_dloc_create_error = buf;
  return st;
}

#define DCK(c, call)                                                                                  \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess)                                                                            \
      return dfail((c), e_ == cudaErrorMemoryAllocation ? SMLM_ERR_OOM : SMLM_ERR_CUDA, "%s: %s", #call, \
                   cudaGetErrorString(e_));                                                           \
  } while (0)

enum PKind { P_DEVICE, P_PINNED, P_OTHER };
PKind kind_of(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return P_OTHER;
  }
  if (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) return P_DEVICE;
  if (a.type == cudaMemoryTypeHost) return P_PINNED;
  return P_OTHER;
}

size_t esz(const dloc_ctx* c) { return c->dt == ACT_F32 ? 4 : 2; }

// one layer's weights: w OIHW [CO_real][CI][k][k], b [CO_real] at `w`; returns floats consumed
smlm_status make_layer(dloc_ctx* c, GLayer& L, int CI, int CO_real, int k, int d, int relu, const float* w,
                       size_t* used) {
  L.CI = CI;
  L.CO_real = CO_real;
  L.CO = (CO_real + 15) / 16 * 16;
  L.k = k;
  L.d = d;
  L.relu = relu;
  const int taps = k * k;
  std::vector<float> wd((size_t)taps * CI * L.CO, 0.0f);
  for (int co = 0; co < CO_real; ++co)
    for (int ci = 0; ci < CI; ++ci)
      for (int t = 0; t < taps; ++t)
        wd[((size_t)t * CI + ci) * L.CO + co] = round_to_act(w[((size_t)co * CI + ci) * taps + t], c->dt);
  DCK(nullptr, cudaMalloc(&L.w_direct, wd.size() * sizeof(float)));
  DCK(nullptr, cudaMemcpy(L.w_direct, wd.data(), wd.size() * sizeof(float), cudaMemcpyHostToDevice));
  std::vector<float> b(L.CO, 0.0f);
  std::memcpy(b.data(), w + (size_t)CO_real * CI * taps, sizeof(float) * CO_real);
  DCK(nullptr, cudaMalloc(&L.bias, b.size() * sizeof(float)));
  DCK(nullptr, cudaMemcpy(L.bias, b.data(), b.size() * sizeof(float), cudaMemcpyHostToDevice));
  if (c->use_umma) {
    std::vector<uint8_t> pack(conv_gen_packed_bytes(CI, L.CO, k));
    conv_gen_pack_host(CI, L.CO, CO_real, k, w, pack.data(), c->dt == ACT_F16);
    DCK(nullptr, cudaMalloc(&L.wpack, pack.size()));
    DCK(nullptr, cudaMemcpy(L.wpack, pack.data(), pack.size(), cudaMemcpyHostToDevice));
    // row-chain kernel: the whole layer in one pass if it fits, else (3x3 only) 16 output channels per pass
    L.chain_co = conv_chain_supports(CI, L.CO, k, d) ? L.CO : (k == 3 && conv_chain_supports(CI, 16, k, d) ? 16 : 0);
    for (int co0 = 0; L.chain_co && co0 < L.CO; co0 += L.chain_co) {
      const int n_real = std::max(0, std::min(L.chain_co, CO_real - co0));
      std::vector<uint8_t> cp(conv_chain_packed_bytes(CI, L.chain_co, k));
      conv_chain_pack_host(CI, L.chain_co, n_real, k, w + (size_t)co0 * CI * taps, cp.data(), c->dt == ACT_F16);
      void* dev = nullptr;
      DCK(nullptr, cudaMalloc(&dev, cp.size()));
      L.wchain.push_back(dev);
      DCK(nullptr, cudaMemcpy(dev, cp.data(), cp.size(), cudaMemcpyHostToDevice));
      LayerConst lc{};
      for (int i = 0; i < L.chain_co; ++i) lc.bias[i] = b[(size_t)co0 + i];
      L.lc.push_back(lc);
    }
  }
  *used = (size_t)CO_real * CI * taps + CO_real;
  return SMLM_OK;
}

void free_layer(GLayer& L) {
  if (L.wpack) cudaFree(L.wpack);
  for (void* p : L.wchain)
    if (p) cudaFree(p);
  L.wchain.clear();
  L.lc.clear();
  if (L.w_direct) cudaFree(L.w_direct);
  if (L.bias) cudaFree(L.bias);
  L.wpack = nullptr;
  L.w_direct = nullptr;
  L.bias = nullptr;
}

void free_bufs(dloc_ctx* c) {
  Bufs& b = c->buf;
  void* all[] = {b.blk[0], b.blk[1], b.cat0, b.p1, b.cat1, b.p2, b.e2, b.m1, b.m0, b.maps, b.slots};
  for (void* p : all)
    if (p) cudaFree(p);
  b = Bufs{};
}

int auto_mb(const dloc_ctx* c, int H, int W) {
  if (c->d.micro_batch > 0) return c->d.micro_batch;
  // ~ (2 CB + 4 C0 + quarter-resolution maps) channels per pixel; keep a launch set <= 8 GB.
  // Up to 64 views per launch: the dense-block launches are short (~50 us at 26 views), so
  // prologue and tail weigh (26 -> 64 views: 8.8 k -> see profiles/bench_r2.md frames/s).
  const double per_view = (double)H * W * esz(c) * (2.0 * c->CB + 5.0 * c->d.c0 + 3.0 * c->d.c0) + 40.0 * H * W;
  int mb = (int)((8192.0 * 1048576.0) / per_view);
  return std::max(1, std::min(mb, 64));
}

smlm_status ensure_bufs(dloc_ctx* c, int mb, int H, int W, bool host_frames) {
  Bufs& b = c->buf;
  if (b.key_mb >= (size_t)mb && b.key_H == (size_t)H && b.key_W == (size_t)W && (!host_frames || b.slots))
    return SMLM_OK;
  DCK(c, cudaDeviceSynchronize());
  free_bufs(c);
  const size_t e = esz(c), px = (size_t)H * W, px2 = (size_t)(H / 2) * (W / 2), px4 = (size_t)(H / 4) * (W / 4);
  const size_t C = c->d.c0;
  DCK(c, cudaMalloc(&b.blk[0], mb * px * c->CB * e));
  DCK(c, cudaMalloc(&b.blk[1], mb * px * c->CB * e));
  DCK(c, cudaMalloc(&b.cat0, mb * px * 3 * C * e));
  DCK(c, cudaMalloc(&b.p1, std::max<size_t>(mb * px2 * C * e, 16)));
  DCK(c, cudaMalloc(&b.cat1, std::max<size_t>(mb * px2 * 6 * C * e, 16)));
  DCK(c, cudaMalloc(&b.p2, std::max<size_t>(mb * px4 * 2 * C * e, 16)));
  DCK(c, cudaMalloc(&b.e2, std::max<size_t>(mb * px4 * 4 * C * e, 16)));
  DCK(c, cudaMalloc(&b.m1, std::max<size_t>(mb * px2 * 2 * C * e, 16)));
  DCK(c, cudaMalloc(&b.m0, mb * px * C * e));
  DCK(c, cudaMalloc(&b.maps, mb * px * DLOC_HEADS * sizeof(float)));
  if (host_frames) DCK(c, cudaMalloc(&b.slots, 2 * (size_t)(mb + 2) * px * sizeof(uint16_t)));
  b.key_mb = mb;
  b.key_H = H;
  b.key_W = W;
  c->slot_used[0] = c->slot_used[1] = false;
  return SMLM_OK;
}

smlm_status conv(dloc_ctx* c, const GLayer& L, const void* in, int in_ch, int ci0, void* out, int out_ch, int co0,
                 int B, int H, int W, float* out_f32, cudaStream_t st) {
  ConvGen a;
  a.in = in;
  a.in_planes = in_ch / 8;
  a.ci_plane0 = ci0 / 8;
  a.CI = L.CI;
  a.out = out;
  a.out_planes = out_ch / 8;
  a.co_plane0 = co0 / 8;
  a.CO = L.CO;
  a.B = B;
  a.H = H;
  a.W = W;
  a.k = L.k;
  a.d = L.d;
  a.relu = L.relu;
  a.out_f32 = out_f32;
  a.n_valid = L.CO_real;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing) {
    if (c->tev_used == c->tev.size()) {
      cudaEvent_t x, y;
      DCK(c, cudaEventCreate(&x));
      DCK(c, cudaEventCreate(&y));
      c->tev.push_back({x, y});
    }
    e0 = c->tev[c->tev_used].first;
    e1 = c->tev[c->tev_used].second;
    ++c->tev_used;
    DCK(c, cudaEventRecord(e0, st));
  }
  cudaError_t e = cudaSuccess;
  if (c->use_umma && !L.wchain.empty() && c->use_chain && a.ci_plane0 == 0 && (!out_f32 || L.wchain.size() == 1)) {
    ConvGen p = a;
    p.CO = L.chain_co;
    for (size_t i = 0; i < L.wchain.size() && e == cudaSuccess; ++i) {
      p.co_plane0 = a.co_plane0 + (int)i * L.chain_co / 8;
      e = launch_conv_chain(c->dt == ACT_F16, p, L.wchain[i], L.lc[i], c->n_sm, st);
    }
  } else
    e = c->use_umma ? launch_conv_gen_umma(c->dt == ACT_F16, a, L.wpack, L.bias, c->n_sm, st)
                    : launch_conv_gen_direct(c->dt, a, L.w_direct, L.bias, st);
  if (e != cudaSuccess) return dfail(c, SMLM_ERR_CUDA, "conv_gen: %s", cudaGetErrorString(e));
  if (c->timing) DCK(c, cudaEventRecord(e1, st));
  c->launches++;
  return SMLM_OK;
}

// forward pass of nf views (whole frames f0 .. f0+nf-1) into buf.maps; dump optional
smlm_status forward(dloc_ctx* c, const uint16_t* dev_frames, int frame_base, int f0, int nf, int n_total, int H,
                    int W, const NormParams& np, float* dump, size_t dump_stride, cudaStream_t st) {
  Bufs& b = c->buf;
  const int C = c->d.c0, G = c->d.growth, ND = c->d.n_dil, NB = c->d.n_blocks, CB = c->CB;
  const int H2 = H / 2, W2 = W / 2, H4 = H2 / 2, W4 = W2 / 2;
  const size_t px = (size_t)H * W;
  smlm_status r;
  size_t doff = 0;
  auto dump_planes = [&](const void* buf, int buf_ch, int ch0, int nch, int h, int w) -> smlm_status {
    if (!dump) return SMLM_OK;
    DCK(c, launch_dump_planar(c->dt, buf, buf_ch / 8, ch0 / 8, nch / 8, nf, h, w, dump + doff, dump_stride, st));
    c->launches++;
    doff += (size_t)nch * h * w;
    return SMLM_OK;
  };
  ViewSet vs{f0, H, W, 0, 0, 0, 1, 0, 1, 0, c->in_frames, n_total};
  DCK(c, launch_stem(c->dt, dev_frames, frame_base, vs, ActShape{nf, C, H, W, CB}, np, c->w_stem, c->b_stem,
                     c->d.stem_relu, b.blk[0], st));
  c->launches++;
  if ((r = dump_planes(b.blk[0], CB, 0, C, H, W)) != SMLM_OK) return r;
  int cur = 0;
  for (int blk = 0; blk < NB; ++blk) {
    for (int i = 0; i < ND; ++i) {  // dense layer i: planes [0, C + iG) -> planes [C + iG, C + (i+1)G) of the same buffer
      const GLayer& L = c->dcd[(size_t)blk * (ND + 1) + i];
      if ((r = conv(c, L, b.blk[cur], CB, 0, b.blk[cur], CB, C + i * G, nf, H, W, nullptr, st)) != SMLM_OK) return r;
    }
    const GLayer& T = c->dcd[(size_t)blk * (ND + 1) + ND];
    const bool last = blk + 1 == NB;
    // transition: all CB planes -> the next block's input planes, or (last block) e0 inside cat0 = [up(m1) | e0]
    if (last) r = conv(c, T, b.blk[cur], CB, 0, b.cat0, 3 * C, 2 * C, nf, H, W, nullptr, st);
    else r = conv(c, T, b.blk[cur], CB, 0, b.blk[cur ^ 1], CB, 0, nf, H, W, nullptr, st);
    if (r != SMLM_OK) return r;
    if (last) r = dump_planes(b.cat0, 3 * C, 2 * C, C, H, W);
    else r = dump_planes(b.blk[cur ^ 1], CB, 0, C, H, W);
    if (r != SMLM_OK) return r;
    cur ^= 1;
  }
  // two-stage U-Net
  DCK(c, launch_pool2(c->dt, b.cat0, 3 * C / 8, 2 * C / 8, b.p1, C / 8, 0, C / 8, nf, H, W, st));
  if ((r = conv(c, c->enc1, b.p1, C, 0, b.cat1, 6 * C, 4 * C, nf, H2, W2, nullptr, st)) != SMLM_OK) return r;
  if ((r = dump_planes(b.cat1, 6 * C, 4 * C, 2 * C, H2, W2)) != SMLM_OK) return r;
  DCK(c, launch_pool2(c->dt, b.cat1, 6 * C / 8, 4 * C / 8, b.p2, 2 * C / 8, 0, 2 * C / 8, nf, H2, W2, st));
  if ((r = conv(c, c->enc2, b.p2, 2 * C, 0, b.e2, 4 * C, 0, nf, H4, W4, nullptr, st)) != SMLM_OK) return r;
  if ((r = dump_planes(b.e2, 4 * C, 0, 4 * C, H4, W4)) != SMLM_OK) return r;
  DCK(c, launch_up2(c->dt, b.e2, 4 * C / 8, 0, H4, W4, b.cat1, 6 * C / 8, 0, 4 * C / 8, nf, H2, W2, st));
  if ((r = conv(c, c->dec1, b.cat1, 6 * C, 0, b.m1, 2 * C, 0, nf, H2, W2, nullptr, st)) != SMLM_OK) return r;
  if ((r = dump_planes(b.m1, 2 * C, 0, 2 * C, H2, W2)) != SMLM_OK) return r;
  DCK(c, launch_up2(c->dt, b.m1, 2 * C / 8, 0, H2, W2, b.cat0, 3 * C / 8, 0, 2 * C / 8, nf, H, W, st));
  if ((r = conv(c, c->dec0, b.cat0, 3 * C, 0, b.m0, C, 0, nf, H, W, nullptr, st)) != SMLM_OK) return r;
  if ((r = dump_planes(b.m0, C, 0, C, H, W)) != SMLM_OK) return r;
  c->launches += 4;
  // heads: 1x1, C0 -> 10 (padded to 16), fp32 planar maps
  if ((r = conv(c, c->heads, b.m0, C, 0, nullptr, 16, 0, nf, H, W, b.maps, st)) != SMLM_OK) return r;
  (void)px;
  return SMLM_OK;
}

smlm_status camera(dloc_ctx* c, const smlm_camera_params* cam, int H, int W, cudaStream_t st, NormParams* np) {
  np->offset = cam->offset;
  np->gain = cam->gain;
  np->norm_scale = c->d.norm_scale;
  np->offset_map = np->gain_map = nullptr;
  if ((cam->offset_map == nullptr) != (cam->gain_map == nullptr))
    return dfail(c, SMLM_ERR_INVALID_ARG, "offset_map and gain_map must both be given or both be NULL");
  if (!cam->offset_map) {
    if (!(cam->gain > 0.0f)) return dfail(c, SMLM_ERR_INVALID_ARG, "camera gain must be > 0");
    return SMLM_OK;
  }
  const size_t n = (size_t)H * W;
  if (kind_of(cam->offset_map) == P_DEVICE && kind_of(cam->gain_map) == P_DEVICE) {
    np->offset_map = cam->offset_map;
    np->gain_map = cam->gain_map;
    return SMLM_OK;
  }
  if (n > c->cam_elems) {
    if (c->cam_off) cudaFree(c->cam_off);
    if (c->cam_gain) cudaFree(c->cam_gain);
    c->cam_off = c->cam_gain = nullptr;
    c->cam_elems = 0;
    DCK(c, cudaMalloc(&c->cam_off, n * sizeof(float)));
    DCK(c, cudaMalloc(&c->cam_gain, n * sizeof(float)));
    c->cam_elems = n;
  }
  DCK(c, cudaMemcpyAsync(c->cam_off, cam->offset_map, n * sizeof(float), cudaMemcpyDefault, st));
  DCK(c, cudaMemcpyAsync(c->cam_gain, cam->gain_map, n * sizeof(float), cudaMemcpyDefault, st));
  np->offset_map = c->cam_off;
  np->gain_map = c->cam_gain;
  return SMLM_OK;
}

struct CountCopy2 { int64_t* dst; const unsigned long long* src; };
void CUDART_CB count_cb2(void* p) {
  CountCopy2* cc = static_cast<CountCopy2*>(p);
  *cc->dst = (int64_t)*cc->src;
  delete cc;
}

// frames [f0, f0 + nf) (+ context neighbours) onto the device: pinned host -> staging slot on the copy stream
smlm_status stage_frames(dloc_ctx* c, const uint16_t* frames, bool host, int64_t chunk, int64_t f0, int nf, int64_t n,
                         size_t px, cudaStream_t st, const uint16_t** dev, int* base, int* slot_out) {
  *slot_out = -1;
  if (!host) {
    *dev = frames;
    *base = 0;
    return SMLM_OK;
  }
  const int slot = (int)(chunk & 1);
  int64_t c0 = f0, c1 = f0 + nf;
  if (c->in_frames == 3) {
    c0 = std::max<int64_t>(f0 - 1, 0);
    c1 = std::min<int64_t>(f0 + nf + 1, n);
  }
  if (c->slot_used[slot]) DCK(c, cudaStreamWaitEvent(c->copy_stream, c->ev_consumed[slot], 0));
  uint16_t* dst = c->buf.slots + (size_t)slot * (c->buf.key_mb + 2) * px;
  DCK(c, cudaMemcpyAsync(dst, frames + (size_t)c0 * px, (size_t)(c1 - c0) * px * 2, cudaMemcpyHostToDevice,
                         c->copy_stream));
  DCK(c, cudaEventRecord(c->ev_copied[slot], c->copy_stream));
  DCK(c, cudaStreamWaitEvent(st, c->ev_copied[slot], 0));
  c->slot_used[slot] = true;
  *dev = dst;
  *base = (int)c0;
  *slot_out = slot;
  return SMLM_OK;
}

}  // namespace

extern "C" {

const char* dloc_last_error(const dloc_ctx* c) { return c ? c->err.c_str() : g_dloc_create_error.c_str(); }
int64_t dloc_launch_count(const dloc_ctx* c) { return c ? c->launches : 0; }

smlm_status dloc_create(const dloc_net_desc* desc, const void* weights, dloc_ctx** out) {
  if (out) *out = nullptr;
  if (!desc || !weights || !out) return dfail(nullptr, SMLM_ERR_INVALID_ARG, "NULL argument");
  if (desc->struct_size != sizeof(dloc_net_desc) || desc->version != DLOC_ABI_VERSION)
    return dfail(nullptr, SMLM_ERR_INVALID_ARG, "dloc_net_desc size / version mismatch");
  const int C = desc->c0, G = desc->growth, NB = desc->n_blocks, ND = desc->n_dil;
  if (C < 16 || C > 64 || C % 16) return dfail(nullptr, SMLM_ERR_INVALID_ARG, "c0 must be 16, 32, 48 or 64");
  if (G < 16 || G > 64 || G % 16) return dfail(nullptr, SMLM_ERR_INVALID_ARG, "growth must be 16, 32, 48 or 64");
  if (NB < 1 || NB > 8 || ND < 1 || ND > DLOC_MAX_DIL)
    return dfail(nullptr, SMLM_ERR_INVALID_ARG, "n_blocks must be 1..8, n_dil 1..8");
  for (int i = 0; i < ND; ++i)
    if (desc->dilations[i] < 1 || desc->dilations[i] > 16)
      return dfail(nullptr, SMLM_ERR_INVALID_ARG, "dilations must be in 1..16");
  if (desc->in_frames != 1 && desc->in_frames != 3) return dfail(nullptr, SMLM_ERR_INVALID_ARG, "in_frames must be 1 or 3");
  if (desc->precision != SMLM_FP32 && desc->precision != SMLM_BF16 && desc->precision != SMLM_FP16)
    return dfail(nullptr, SMLM_ERR_INVALID_ARG, "bad precision");
  if (desc->conv_impl < SMLM_CONV_AUTO || desc->conv_impl > SMLM_CONV_DIRECT)
    return dfail(nullptr, SMLM_ERR_INVALID_ARG, "bad conv_impl");
  if (desc->precision == SMLM_FP32 && desc->conv_impl == SMLM_CONV_TCGEN05)
    return dfail(nullptr, SMLM_ERR_INVALID_ARG, "the tcgen05 kernel needs a 16-bit precision");
  if (!(desc->norm_scale > 0.0f) || desc->micro_batch < 0)
    return dfail(nullptr, SMLM_ERR_INVALID_ARG, "norm_scale must be > 0, micro_batch >= 0");
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return dfail(nullptr, SMLM_ERR_UNSUPPORTED_DEVICE, "no CUDA device (this library has no CPU fallback)");
  }
  if (prop.major != 10) return dfail(nullptr, SMLM_ERR_UNSUPPORTED_DEVICE, "sm_100 (B200) required, found sm_%d%d",
                                     prop.major, prop.minor);
  dloc_ctx* c = new (std::nothrow) dloc_ctx;
  if (!c) return dfail(nullptr, SMLM_ERR_OOM, "host allocation failed");
  c->d = *desc;
  c->dt = desc->precision == SMLM_BF16 ? ACT_BF16 : (desc->precision == SMLM_FP16 ? ACT_F16 : ACT_F32);
  c->in_frames = desc->in_frames;
  c->use_umma = c->dt != ACT_F32 && desc->conv_impl != SMLM_CONV_DIRECT;
  c->use_chain = desc->conv_impl == SMLM_CONV_AUTO;
  c->n_sm = prop.multiProcessorCount;
  c->CB = C + ND * G;
  smlm_status st = SMLM_OK;
  auto body = [&]() -> smlm_status {
    const float* w = static_cast<const float*>(weights);
    const int IF = c->in_frames, T9 = 9 * IF;
    std::vector<float> tmp((size_t)T9 * C);
    for (int co = 0; co < C; ++co)
      for (int t = 0; t < T9; ++t) tmp[(size_t)t * C + co] = w[(size_t)co * T9 + t];
    DCK(nullptr, cudaMalloc(&c->w_stem, tmp.size() * sizeof(float)));
    DCK(nullptr, cudaMemcpy(c->w_stem, tmp.data(), tmp.size() * sizeof(float), cudaMemcpyHostToDevice));
    DCK(nullptr, cudaMalloc(&c->b_stem, C * sizeof(float)));
    DCK(nullptr, cudaMemcpy(c->b_stem, w + (size_t)T9 * C, C * sizeof(float), cudaMemcpyHostToDevice));
    w += (size_t)(T9 + 1) * C;
    size_t used = 0;
    c->dcd.resize((size_t)NB * (ND + 1));
    for (int b = 0; b < NB; ++b) {
      for (int i = 0; i < ND; ++i) {
        if ((st = make_layer(c, c->dcd[(size_t)b * (ND + 1) + i], C + i * G, G, 3, desc->dilations[i], 1, w, &used)) != SMLM_OK)
          return st;
        w += used;
      }
      if ((st = make_layer(c, c->dcd[(size_t)b * (ND + 1) + ND], c->CB, C, 1, 1, 1, w, &used)) != SMLM_OK) return st;
      w += used;
    }
    if ((st = make_layer(c, c->enc1, C, 2 * C, 3, 1, 1, w, &used)) != SMLM_OK) return st;
    w += used;
    if ((st = make_layer(c, c->enc2, 2 * C, 4 * C, 3, 1, 1, w, &used)) != SMLM_OK) return st;
    w += used;
    if ((st = make_layer(c, c->dec1, 6 * C, 2 * C, 3, 1, 1, w, &used)) != SMLM_OK) return st;
    w += used;
    if ((st = make_layer(c, c->dec0, 3 * C, C, 3, 1, 1, w, &used)) != SMLM_OK) return st;
    w += used;
    if ((st = make_layer(c, c->heads, C, DLOC_HEADS, 1, 1, 0, w, &used)) != SMLM_OK) return st;
    DCK(nullptr, cudaMalloc(&c->counter, sizeof(unsigned long long)));
    DCK(nullptr, cudaHostAlloc(&c->h_count, sizeof(unsigned long long), cudaHostAllocDefault));
    *c->h_count = 0;
    DCK(nullptr, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      DCK(nullptr, cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming));
      DCK(nullptr, cudaEventCreateWithFlags(&c->ev_consumed[i], cudaEventDisableTiming));
    }
    DCK(nullptr, cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
    return SMLM_OK;
  };
  st = body();
  if (st != SMLM_OK) {
    dloc_destroy(c);
    return st;
  }
  *out = c;
  return SMLM_OK;
}

void dloc_destroy(dloc_ctx* c) {
  if (!c) return;
  cudaDeviceSynchronize();
  free_bufs(c);
  for (auto& L : c->dcd) free_layer(L);
  free_layer(c->enc1);
  free_layer(c->enc2);
  free_layer(c->dec1);
  free_layer(c->dec0);
  free_layer(c->heads);
  if (c->w_stem) cudaFree(c->w_stem);
  if (c->b_stem) cudaFree(c->b_stem);
  if (c->cam_off) cudaFree(c->cam_off);
  if (c->cam_gain) cudaFree(c->cam_gain);
  if (c->counter) cudaFree(c->counter);
  if (c->h_count) cudaFreeHost(c->h_count);
  if (c->em_dev) cudaFree(c->em_dev);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  for (int i = 0; i < 2; ++i) {
    if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
    if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]);
  }
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  for (auto& p : c->tev) {
    cudaEventDestroy(p.first);
    cudaEventDestroy(p.second);
  }
  delete c;
}

smlm_status dloc_check(dloc_ctx* c) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return dfail(c, SMLM_ERR_CUDA, "pending CUDA error: %s", cudaGetErrorString(e));
  if (*c->h_count > c->last_capacity)
    return dfail(c, SMLM_ERR_OVERFLOW, "found %llu emitters, capacity %llu", *c->h_count, c->last_capacity);
  return SMLM_OK;
}

smlm_status dloc_kernel_timing(dloc_ctx* c, int32_t enable) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  c->timing = enable != 0;
  c->tev_used = 0;
  c->conv_ms = 0.0;
  c->conv_n = 0;
  return SMLM_OK;
}

smlm_status dloc_conv_time_ms(dloc_ctx* c, double* ms, int64_t* launches) {
  if (!c || !ms || !launches) return SMLM_ERR_INVALID_ARG;
  DCK(c, cudaDeviceSynchronize());
  double t = 0.0;
  for (size_t i = 0; i < c->tev_used; ++i) {
    float x = 0.0f;
    DCK(c, cudaEventElapsedTime(&x, c->tev[i].first, c->tev[i].second));
    t += x;
  }
  *ms = t;
  *launches = (int64_t)c->tev_used;
  return SMLM_OK;
}

smlm_status dloc_localize(dloc_ctx* c, const uint16_t* frames, int64_t n, int32_t H, int32_t W,
                          const smlm_camera_params* cam, float threshold, dloc_emitter* out, int64_t* out_count,
                          void* cuda_stream) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  if (!cam || !out_count) return dfail(c, SMLM_ERR_INVALID_ARG, "NULL camera / out_count");
  if (n < 0 || n > INT32_MAX || H < 4 || W < 4 || (int64_t)H * W > (int64_t)1 << 28)
    return dfail(c, SMLM_ERR_INVALID_ARG, "bad n_frames / H / W (H, W >= 4)");
  if (*out_count < 0) return dfail(c, SMLM_ERR_INVALID_ARG, "negative capacity");
  if (!(threshold == threshold)) return dfail(c, SMLM_ERR_INVALID_ARG, "threshold is NaN");
  if (!(cam->pixel_size_nm > 0.0f)) return dfail(c, SMLM_ERR_INVALID_ARG, "pixel_size_nm must be > 0");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const unsigned long long capacity = (unsigned long long)*out_count;
  PKind fk = P_DEVICE, ok = P_DEVICE;
  if (n > 0) {
    if (!frames) return dfail(c, SMLM_ERR_INVALID_ARG, "NULL frames");
    fk = kind_of(frames);
    if (fk == P_OTHER) return dfail(c, SMLM_ERR_INVALID_ARG, "frames_u16 must be pinned host or device memory");
  }
  if (capacity > 0) {
    if (!out) return dfail(c, SMLM_ERR_INVALID_ARG, "NULL out_emitters with capacity > 0");
    ok = kind_of(out);
    if (ok == P_OTHER) return dfail(c, SMLM_ERR_INVALID_ARG, "out_emitters must be device or pinned host memory");
  }
  NormParams np;
  smlm_status r = camera(c, cam, H, W, st, &np);
  if (r != SMLM_OK) return r;
  DlocPostParams pp;
  pp.hp.n_h = DLOC_HEADS;
  pp.hp.lthr = threshold <= 0.0f ? -INFINITY
                                 : (threshold >= 1.0f ? INFINITY
                                                      : (float)std::log((double)threshold / (1.0 - (double)threshold)));
  pp.hp.xy_scale = c->d.xy_scale;
  pp.hp.z_scale_nm = c->d.z_scale_nm;
  pp.hp.photon_scale = c->d.photon_scale;
  pp.hp.bg_scale = c->d.bg_scale;
  pp.hp.pixel_size_nm = cam->pixel_size_nm;
  pp.sigma_xy_px = c->d.sigma_xy_px;
  pp.sigma_z_nm = c->d.sigma_z_nm;
  pp.sigma_photons = c->d.sigma_photons;
  const int mb = (int)std::max<int64_t>(1, std::min<int64_t>(auto_mb(c, H, W), std::max<int64_t>(n, 1)));
  const bool host = fk == P_PINNED && n > 0;
  if ((r = ensure_bufs(c, mb, H, W, host)) != SMLM_OK) return r;
  dloc_emitter* list = out;
  if (ok == P_PINNED && capacity > 0) {
    if (capacity > c->em_cap) {
      DCK(c, cudaDeviceSynchronize());
      if (c->em_dev) cudaFree(c->em_dev);
      c->em_dev = nullptr;
      c->em_cap = 0;
      DCK(c, cudaMalloc(&c->em_dev, capacity * sizeof(dloc_emitter)));
      c->em_cap = capacity;
    }
    list = c->em_dev;
  }
  DCK(c, cudaMemsetAsync(c->counter, 0, sizeof(unsigned long long), st));
  c->last_capacity = capacity;
  if (host) {
    DCK(c, cudaEventRecord(c->ev_start, st));
    DCK(c, cudaStreamWaitEvent(c->copy_stream, c->ev_start, 0));
  }
  const size_t px = (size_t)H * W;
  int64_t chunk = 0;
  for (int64_t f0 = 0; f0 < n; f0 += mb, ++chunk) {
    const int nf = (int)std::min<int64_t>(mb, n - f0);
    const uint16_t* dev = nullptr;
    int base = 0, slot = -1;
    if ((r = stage_frames(c, frames, host, chunk, f0, nf, n, px, st, &dev, &base, &slot)) != SMLM_OK) return r;
    if ((r = forward(c, dev, base, (int)f0, nf, (int)n, H, W, np, nullptr, 0, st)) != SMLM_OK) return r;
    if (slot >= 0) DCK(c, cudaEventRecord(c->ev_consumed[slot], st));  // (recorded after the whole set: simple and safe)
    DCK(c, launch_dloc_post(c->buf.maps, nf, H, W, (int)f0, pp, list, c->counter, capacity, st));
    c->launches++;
  }
  DCK(c, cudaMemcpyAsync(c->h_count, c->counter, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  if (list != out) {
    // the list goes to the caller's pinned buffer once the count is known to the device: copy
    // min(count, capacity) records with a small kernel-free path - a full-capacity memcpy
    // would move megabytes of nothing, so read the count back first (one stream sync point)
    DCK(c, cudaStreamSynchronize(st));
    const unsigned long long cnt = std::min<unsigned long long>(*c->h_count, capacity);
    if (cnt) DCK(c, cudaMemcpyAsync(out, list, cnt * sizeof(dloc_emitter), cudaMemcpyDeviceToHost, st));
  }
  CountCopy2* cc = new (std::nothrow) CountCopy2{out_count, c->h_count};
  if (!cc) return dfail(c, SMLM_ERR_OOM, "host allocation failed");
  cudaError_t e = cudaLaunchHostFunc(st, count_cb2, cc);
  if (e != cudaSuccess) {
    delete cc;
    return dfail(c, SMLM_ERR_CUDA, "cudaLaunchHostFunc: %s", cudaGetErrorString(e));
  }
  return SMLM_OK;
}

smlm_status dloc_debug_forward_maps(dloc_ctx* c, const uint16_t* frames, int64_t n, int32_t H, int32_t W,
                                    const smlm_camera_params* cam, float* maps, float* dump, void* cuda_stream) {
  if (!c) return SMLM_ERR_INVALID_ARG;
  if (!cam || !maps || (n > 0 && !frames) || n < 0 || n > INT32_MAX || H < 4 || W < 4)
    return dfail(c, SMLM_ERR_INVALID_ARG, "bad argument");
  if (kind_of(maps) != P_DEVICE || (dump && kind_of(dump) != P_DEVICE) || (n > 0 && kind_of(frames) != P_DEVICE))
    return dfail(c, SMLM_ERR_INVALID_ARG, "frames / maps / dump must be device memory here");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  NormParams np;
  smlm_status r = camera(c, cam, H, W, st, &np);
  if (r != SMLM_OK) return r;
  const int mb = (int)std::max<int64_t>(1, std::min<int64_t>(auto_mb(c, H, W), std::max<int64_t>(n, 1)));
  if ((r = ensure_bufs(c, mb, H, W, false)) != SMLM_OK) return r;
  const size_t px = (size_t)H * W, C = c->d.c0;
  const size_t per = (size_t)(1 + c->d.n_blocks) * C * px + (size_t)4 * C * (H / 2) * (W / 2) +
                     (size_t)4 * C * (H / 4) * (W / 4) + C * px;
  for (int64_t f0 = 0; f0 < n; f0 += mb) {
    const int nf = (int)std::min<int64_t>(mb, n - f0);
    if ((r = forward(c, frames, 0, (int)f0, nf, (int)n, H, W, np, dump ? dump + (size_t)f0 * per : nullptr, per, st)) !=
        SMLM_OK)
      return r;
    DCK(c, cudaMemcpyAsync(maps + (size_t)f0 * DLOC_HEADS * px, c->buf.maps, (size_t)nf * DLOC_HEADS * px * sizeof(float),
                           cudaMemcpyDeviceToDevice, st));
  }
  return SMLM_OK;
}

}  // extern "C"
