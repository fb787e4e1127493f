// K3: 1x1 heads fused with the post-processing (BASELINE.json north_star (c); smlm.h):
//   o = Wh a_L + bh;  pixel q is an emitter iff sigmoid(o_p[q]) > thr (tested in the logit
//   domain: o_p > logit(thr)) and o_p[q] beats each in-frame 8-neighbour (greater, or equal
//   with the lower linear index);  x = (ix + xy_scale tanh(o_dx)) px, ... ; records are
//   appended to one list through a block-aggregated atomic counter.
// The output maps never reach HBM: the block computes the detection logit of a
// (TH+2) x (TW+2) patch into shared memory, runs the 3x3 test there, and evaluates the
// remaining heads (and every transcendental) for the survivors only.
//
// HBM/L2-read-bound: 2C B/px of activations (+ ~10 % halo re-read), 32 B per emitter out.
#include <math_constants.h>

#include "chunk_io.cuh"
#include "smlm_internal.cuh"

namespace smlm {
namespace {

constexpr int TW = 64, TH = 32, NT = 256;
constexpr int MAX_CAND = (TW / 2) * (TH / 2);  // no two detections are 8-adjacent

__device__ inline float sigmoid_f(float v) { return 1.0f / (1.0f + expf(-v)); }
__device__ inline float softplus_f(float v) { return fmaxf(v, 0.0f) + log1pf(expf(-fabsf(v))); }

// One head of one pixel from the activations.  Fixed summation order, shared with the HEAD
// epilogue of conv_umma.cu (whose two warps per pixel each own one channel half): two fmaf
// chains, channels [0, C/2) starting from the bias and [C/2, C) starting from zero, added at
// the end - so every kernel produces bit-identical values for the same pixel.
template <typename T, int C>
struct ActSource {
  const T* act;
  ActShape s;
  const float* wh;  // shared memory [n_h][C]
  const float* bh;  // shared memory [n_h]
  __device__ inline float head(int h, int b, int y, int x) const {
    float acc0 = bh[h], acc1 = 0.0f;
    const float* w = wh + h * C;
#pragma unroll
    for (int k = 0; k < C / 8; ++k) {
      float v[8];
      Chunk<T>::load(act, s.chunk_index(b, k, y, x), v);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        if (k < C / 16) acc0 = fmaf(v[c], w[k * 8 + c], acc0);
        else acc1 = fmaf(v[c], w[k * 8 + c], acc1);
      }
    }
    return acc0 + acc1;
  }
};

struct MapSource {
  const float* maps;  // [n][n_h][H][W]
  int n_h, H, W;
  __device__ inline float head(int h, int b, int y, int x) const {
    return maps[(((size_t)b * n_h + h) * H + y) * W + x];
  }
};

template <typename Src>
__device__ inline void detect_tile(const Src& src, int Hw, int Ww, const View& v, int b, int Wf,
                                   const HeadParams& hp, smlm_emitter* __restrict__ out,
                                   unsigned long long* __restrict__ counter,
                                   unsigned long long capacity) {
  __shared__ float lg[TH + 2][TW + 2];
  __shared__ int cand[MAX_CAND];
  __shared__ int ncand;
  __shared__ unsigned long long base;

  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
  if (tid == 0) ncand = 0;

  // phase 1: detection logit of the patch; outside the window (= outside the frame for
  // every pixel that neighbours an owned pixel) it is -inf: such neighbours never win.
  for (int i = tid; i < (TH + 2) * (TW + 2); i += NT) {
    int ly = i / (TW + 2), lx = i - ly * (TW + 2);
    int y = y0 + ly - 1, x = x0 + lx - 1;
    float o = -CUDART_INF_F;
    if (y >= 0 && y < Hw && x >= 0 && x < Ww) o = src.head(0, b, y, x);
    lg[ly][lx] = o;
  }
  __syncthreads();

  // phase 2: threshold + 3x3 local maximum with the index tie rule.  Neighbours with a
  // lower linear index (row above, left) must be strictly smaller; the others may be equal.
  for (int i = tid; i < TH * TW; i += NT) {
    int ly = i / TW, lx = i - ly * TW;
    int y = y0 + ly, x = x0 + lx;
    bool keep = (y >= v.cy0 && y < v.cy1 && x >= v.cx0 && x < v.cx1);
    if (keep) {
      float c = lg[ly + 1][lx + 1];
      keep = (c > hp.lthr) && c > lg[ly][lx] && c > lg[ly][lx + 1] && c > lg[ly][lx + 2] &&
             c > lg[ly + 1][lx] && c >= lg[ly + 1][lx + 2] && c >= lg[ly + 2][lx] &&
             c >= lg[ly + 2][lx + 1] && c >= lg[ly + 2][lx + 2];
    }
    unsigned m = __ballot_sync(0xffffffffu, keep);
    if (m) {
      int lane = tid & 31, leader = __ffs(m) - 1, slot = 0;
      if (lane == leader) slot = atomicAdd(&ncand, __popc(m));
      slot = __shfl_sync(0xffffffffu, slot, leader);
      if (keep) cand[slot + __popc(m & ((1u << lane) - 1u))] = i;
    }
  }
  __syncthreads();
  const int n = ncand;
  if (n == 0) return;
  if (tid == 0) base = atomicAdd(counter, (unsigned long long)n);
  __syncthreads();

  // phase 3: remaining heads + decode for the survivors only.
  for (int j = tid; j < n; j += NT) {
    unsigned long long slot = base + j;
    if (slot >= capacity) continue;  // counted, not stored (smlm_check reports overflow)
    int i = cand[j];
    int ly = i / TW, lx = i - ly * TW;
    int y = y0 + ly, x = x0 + lx;
    int fy = v.wy0 + y, fx = v.wx0 + x;
    const int hN = hp.n_h == 6 ? 4 : 3;
    float odx = src.head(1, b, y, x), ody = src.head(2, b, y, x);
    float oN = src.head(hN, b, y, x), obg = src.head(hN + 1, b, y, x);
    smlm_emitter e;
    e.frame = v.frame;
    e.pix = fy * Wf + fx;
    e.x_nm = ((float)fx + hp.xy_scale * tanhf(odx)) * hp.pixel_size_nm;
    e.y_nm = ((float)fy + hp.xy_scale * tanhf(ody)) * hp.pixel_size_nm;
    e.z_nm = hp.n_h == 6 ? hp.z_scale_nm * tanhf(src.head(3, b, y, x)) : 0.0f;
    e.photons = hp.photon_scale * softplus_f(oN);
    e.bg = hp.bg_scale * softplus_f(obg);
    e.p = sigmoid_f(lg[ly + 1][lx + 1]);
    uint4* dst = reinterpret_cast<uint4*>(out + slot);
    const uint4* srcv = reinterpret_cast<const uint4*>(&e);
    dst[0] = srcv[0];
    dst[1] = srcv[1];
  }
}

template <typename T, int C>
__global__ void __launch_bounds__(NT)
    head_post_kernel(const T* __restrict__ act, ActShape s, ViewSet vs,
                     const float* __restrict__ w_head, const float* __restrict__ b_head,
                     HeadParams hp, smlm_emitter* __restrict__ out,
                     unsigned long long* __restrict__ counter, unsigned long long capacity) {
  __shared__ float wh[6 * C];
  __shared__ float bh[8];
  for (int i = threadIdx.x; i < hp.n_h * C; i += NT) wh[i] = w_head[i];
  if (threadIdx.x < hp.n_h) bh[threadIdx.x] = b_head[threadIdx.x];
  __syncthreads();
  const int b = blockIdx.z;
  const View v = view_of(vs, b, s.H, s.W);
  ActSource<T, C> src{act, s, wh, bh};
  detect_tile(src, s.H, s.W, v, b, vs.Wf, hp, out, counter, capacity);
}

// K3 after a HEAD conv layer (conv_umma.cu): the detection logit is already an fp32 map and
// the other heads of every above-threshold pixel sit in 32-byte candidate records, so this
// kernel touches no activations.  One (LH+2) x (LW+2) logit patch per block goes to shared
// memory in one round trip (three independent loads per thread), the 3x3 test runs there,
// survivors are compacted through a warp-aggregated shared-memory counter, the block takes
// one contiguous range of the list with a single global atomicAdd (same-address atomics
// from every warp serialise in L2), and each survivor decodes its candidate record.
constexpr int LW = 64, LH = 16;  // NT = 256 threads, four pixels each
constexpr int LCAND = (LW / 2) * (LH / 2);  // no two detections are 8-adjacent

// Where a survivor's other heads (pre-activation) come from: the 32-byte candidate records of
// conv_umma.cu's HEAD epilogue, or (conv_pair.cu) the last activation map, which that kernel
// stores for above-threshold pixels only - evaluated here with the chains of ActSource.
struct CandHeads {
  const float* cand;
  __device__ inline void get(const ActShape& s, const HeadParams& hp, int b, int y, int x, float& odx, float& ody,
                             float& oz, float& oN, float& obg) const {
    const float4* cq = reinterpret_cast<const float4*>(cand) + (((size_t)b * s.H + y) * s.W + x) * 2;
    const float4 c0 = __ldg(cq), c1 = __ldg(cq + 1);
    const bool six = hp.n_h == 6;
    odx = c0.x;
    ody = c0.y;
    oz = c0.z;
    oN = six ? c0.w : c0.z;
    obg = six ? c1.x : c0.w;
  }
};
template <typename T, int C>
struct ActHeads {
  ActSource<T, C> src;
  __device__ inline void get(const ActShape&, const HeadParams& hp, int b, int y, int x, float& odx, float& ody,
                             float& oz, float& oN, float& obg) const {
    const int hN = hp.n_h == 6 ? 4 : 3;
    odx = src.head(1, b, y, x);
    ody = src.head(2, b, y, x);
    oz = hp.n_h == 6 ? src.head(3, b, y, x) : 0.0f;
    oN = src.head(hN, b, y, x);
    obg = src.head(hN + 1, b, y, x);
  }
};

template <typename Heads>
__device__ __forceinline__ void post_logits_body(const float* __restrict__ logit, const Heads& heads, ActShape s,
                                                 ViewSet vs, HeadParams hp, smlm_emitter* __restrict__ out,
                                                 unsigned long long* __restrict__ counter,
                                                 unsigned long long capacity) {
  __shared__ float lg[LH + 2][LW + 2];
  __shared__ int cnd[LCAND];
  __shared__ int ncand;
  __shared__ unsigned long long base;
  const int tid = threadIdx.x;
  const int b = blockIdx.z;
  const int x0 = blockIdx.x * LW, y0 = blockIdx.y * LH;
  const float* lmap = logit + (size_t)b * s.H * s.W;
  constexpr int PATCH = (LH + 2) * (LW + 2);
  float pv[(PATCH + NT - 1) / NT];
#pragma unroll
  for (int r = 0; r < (PATCH + NT - 1) / NT; ++r) {
    const int i = tid + r * NT;
    const int ly = i / (LW + 2), lx = i - ly * (LW + 2);
    const int y = y0 + ly - 1, x = x0 + lx - 1;
    pv[r] = (i < PATCH && y >= 0 && y < s.H && x >= 0 && x < s.W) ? __ldg(lmap + (size_t)y * s.W + x)
                                                                : -CUDART_INF_F;
  }
  if (tid == 0) ncand = 0;
#pragma unroll
  for (int r = 0; r < (PATCH + NT - 1) / NT; ++r) {
    const int i = tid + r * NT;
    if (i < PATCH) lg[i / (LW + 2)][i % (LW + 2)] = pv[r];
  }
  __syncthreads();

  const View v = view_of(vs, b, s.H, s.W);
#pragma unroll
  for (int r = 0; r < LW * LH / NT; ++r) {
    const int i = tid + r * NT;
    const int ly = i / LW, lx = i - ly * LW;
    const int y = y0 + ly, x = x0 + lx;
    bool keep = (y >= v.cy0 && y < v.cy1 && x >= v.cx0 && x < v.cx1);
    if (keep) {
      const float c = lg[ly + 1][lx + 1];
      keep = (c > hp.lthr) && c > lg[ly][lx] && c > lg[ly][lx + 1] && c > lg[ly][lx + 2] &&
             c > lg[ly + 1][lx] && c >= lg[ly + 1][lx + 2] && c >= lg[ly + 2][lx] &&
             c >= lg[ly + 2][lx + 1] && c >= lg[ly + 2][lx + 2];
    }
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    if (m) {
      const int lane = tid & 31, leader = __ffs(m) - 1;
      int slot = 0;
      if (lane == leader) slot = atomicAdd(&ncand, __popc(m));
      slot = __shfl_sync(0xffffffffu, slot, leader);
      if (keep) cnd[slot + __popc(m & ((1u << lane) - 1u))] = i;
    }
  }
  __syncthreads();
  const int n = ncand;
  if (n == 0) return;
  // the block's survivors take one contiguous range of the list: one global atomic per block
  if (tid == 0) base = atomicAdd(counter, (unsigned long long)n);
  __syncthreads();
  if (tid >= n) return;
  const unsigned long long slot = base + tid;
  if (slot >= capacity) return;  // counted, not stored (smlm_check reports overflow)
  const int i = cnd[tid];
  const int ly = i / LW, lx = i - ly * LW;
  const int y = y0 + ly, x = x0 + lx;
  const int fy = v.wy0 + y, fx = v.wx0 + x;
  // heads 1 .. n_h-1 (pre-activation) = (dx, dy, [z,] N, bg)
  const bool six = hp.n_h == 6;
  float odx, ody, oz, oN, obg;
  heads.get(s, hp, b, y, x, odx, ody, oz, oN, obg);
  smlm_emitter e;
  e.frame = v.frame;
  e.pix = fy * vs.Wf + fx;
  e.x_nm = ((float)fx + hp.xy_scale * tanhf(odx)) * hp.pixel_size_nm;
  e.y_nm = ((float)fy + hp.xy_scale * tanhf(ody)) * hp.pixel_size_nm;
  e.z_nm = six ? hp.z_scale_nm * tanhf(oz) : 0.0f;
  e.photons = hp.photon_scale * softplus_f(oN);
  e.bg = hp.bg_scale * softplus_f(obg);
  e.p = sigmoid_f(lg[ly + 1][lx + 1]);
  uint4* dst = reinterpret_cast<uint4*>(out + slot);
  const uint4* srcv = reinterpret_cast<const uint4*>(&e);
  dst[0] = srcv[0];
  dst[1] = srcv[1];
}

__global__ void __launch_bounds__(NT, 4)
    post_logits_kernel(const float* __restrict__ logit, const float* __restrict__ cand, ActShape s,
                       ViewSet vs, HeadParams hp, smlm_emitter* __restrict__ out,
                       unsigned long long* __restrict__ counter, unsigned long long capacity) {
  post_logits_body(logit, CandHeads{cand}, s, vs, hp, out, counter, capacity);
}

template <typename T, int C>
__global__ void __launch_bounds__(NT, 4)
    post_logits_act_kernel(const float* __restrict__ logit, const T* __restrict__ act, ActShape s, ViewSet vs,
                           const float* __restrict__ w_head, const float* __restrict__ b_head, HeadParams hp,
                           smlm_emitter* __restrict__ out, unsigned long long* __restrict__ counter,
                           unsigned long long capacity) {
  __shared__ float wh[6 * C];
  __shared__ float bh[8];
  for (int i = threadIdx.x; i < hp.n_h * C; i += NT) wh[i] = w_head[i];
  if (threadIdx.x < hp.n_h) bh[threadIdx.x] = b_head[threadIdx.x];
  __syncthreads();
  post_logits_body(logit, ActHeads<T, C>{ActSource<T, C>{act, s, wh, bh}}, s, vs, hp, out, counter, capacity);
}

__global__ void __launch_bounds__(NT)
    post_from_maps_kernel(const float* __restrict__ maps, int H, int W, HeadParams hp,
                          smlm_emitter* __restrict__ out, unsigned long long* __restrict__ counter,
                          unsigned long long capacity) {
  const int b = blockIdx.z;
  View v;
  v.frame = b;
  v.wy0 = v.wx0 = 0;
  v.cy0 = v.cx0 = 0;
  v.cy1 = H;
  v.cx1 = W;
  MapSource src{maps, hp.n_h, H, W};
  detect_tile(src, H, W, v, b, W, hp, out, counter, capacity);
}

template <typename T, int C>
__global__ void __launch_bounds__(NT)
    head_maps_kernel(const T* __restrict__ act, ActShape s, const float* __restrict__ w_head,
                     const float* __restrict__ b_head, int n_h, float* __restrict__ maps) {
  __shared__ float wh[6 * C];
  __shared__ float bh[8];
  for (int i = threadIdx.x; i < n_h * C; i += NT) wh[i] = w_head[i];
  if (threadIdx.x < n_h) bh[threadIdx.x] = b_head[threadIdx.x];
  __syncthreads();
  const int b = blockIdx.z, y = blockIdx.y;
  ActSource<T, C> src{act, s, wh, bh};
  for (int x = blockIdx.x * NT + threadIdx.x; x < s.W; x += gridDim.x * NT)
    for (int h = 0; h < n_h; ++h)
      maps[(((size_t)b * n_h + h) * s.H + y) * s.W + x] = src.head(h, b, y, x);
}

template <typename T>
__global__ void __launch_bounds__(NT)
    dump_act_kernel(const T* __restrict__ act, ActShape s, float* __restrict__ dst,
                    size_t view_stride) {
  const int b = blockIdx.z, y = blockIdx.y;
  for (int x = blockIdx.x * NT + threadIdx.x; x < s.W; x += gridDim.x * NT)
    for (int k = 0; k < s.C / 8; ++k) {
      float v[8];
      Chunk<T>::load(act, s.chunk_index(b, k, y, x), v);
      float* d = dst + (size_t)b * view_stride + ((size_t)y * s.W + x) * s.C + k * 8;
      for (int c = 0; c < 8; ++c) d[c] = v[c];
    }
}

__global__ void snapshot_kernel(const unsigned long long* counter, unsigned long long capacity,
                                unsigned long long* snap) {
  unsigned long long c = *counter;
  *snap = c < capacity ? c : capacity;
}

__global__ void __launch_bounds__(NT)
    flush_kernel(const smlm_emitter* __restrict__ dev, smlm_emitter* __restrict__ host,
                 const unsigned long long* __restrict__ lo_word,
                 const unsigned long long* __restrict__ hi_word) {
  // 16-byte units; grid-stride.  Both ends are snapshot words that nothing rewrites while
  // this launch runs (api.cu: ring of snapshots), so every block sees the same range.
  const unsigned long long lo = *lo_word * 2, hi = *hi_word * 2;
  const uint4* s = reinterpret_cast<const uint4*>(dev);
  uint4* d = reinterpret_cast<uint4*>(host);
  for (unsigned long long i = lo + (unsigned long long)blockIdx.x * NT + threadIdx.x; i < hi;
       i += (unsigned long long)gridDim.x * NT)
    d[i] = s[i];
}

template <typename T, int C>
cudaError_t head_post_tc(const void* act, ActShape s, ViewSet vs, const float* w, const float* b,
                         HeadParams hp, smlm_emitter* out, unsigned long long* counter,
                         unsigned long long cap, cudaStream_t st) {
  dim3 grid((s.W + TW - 1) / TW, (s.H + TH - 1) / TH, s.B);
  head_post_kernel<T, C><<<grid, NT, 0, st>>>((const T*)act, s, vs, w, b, hp, out, counter, cap);
  return cudaGetLastError();
}
template <typename T, int C>
cudaError_t head_maps_tc(const void* act, ActShape s, const float* w, const float* b, int n_h,
                         float* maps, cudaStream_t st) {
  dim3 grid((s.W + NT - 1) / NT, s.H, s.B);
  head_maps_kernel<T, C><<<grid, NT, 0, st>>>((const T*)act, s, w, b, n_h, maps);
  return cudaGetLastError();
}

#define SMLM_DISPATCH_C(T, FN, ...)                      \
  switch (s.C) {                                         \
    case 16: return FN<T, 16>(__VA_ARGS__);              \
    case 32: return FN<T, 32>(__VA_ARGS__);              \
    case 48: return FN<T, 48>(__VA_ARGS__);              \
    case 64: return FN<T, 64>(__VA_ARGS__);              \
    default: return cudaErrorInvalidValue;               \
  }

}  // namespace

cudaError_t launch_head_post(int dt, const void* act, ActShape s, ViewSet vs,
                             const float* w_head, const float* b_head, HeadParams hp,
                             smlm_emitter* out, unsigned long long* counter,
                             unsigned long long capacity, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  if (dt == ACT_BF16) {
    SMLM_DISPATCH_C(__nv_bfloat16, head_post_tc, act, s, vs, w_head, b_head, hp, out, counter, capacity, st)
  } else if (dt == ACT_F16) {
    SMLM_DISPATCH_C(__half, head_post_tc, act, s, vs, w_head, b_head, hp, out, counter, capacity, st)
  } else {
    SMLM_DISPATCH_C(float, head_post_tc, act, s, vs, w_head, b_head, hp, out, counter, capacity, st)
  }
}

cudaError_t launch_post_logits(const float* logit, const float* cand, ActShape s, ViewSet vs,
                               HeadParams hp, smlm_emitter* out, unsigned long long* counter,
                               unsigned long long capacity, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  dim3 grid((s.W + LW - 1) / LW, (s.H + LH - 1) / LH, s.B);
  post_logits_kernel<<<grid, NT, 0, st>>>(logit, cand, s, vs, hp, out, counter, capacity);
  return cudaGetLastError();
}

template <typename T, int C>
cudaError_t post_logits_act_tc(const float* logit, const void* act, ActShape s, ViewSet vs, const float* w,
                               const float* b, HeadParams hp, smlm_emitter* out, unsigned long long* counter,
                               unsigned long long capacity, cudaStream_t st) {
  dim3 grid((s.W + LW - 1) / LW, (s.H + LH - 1) / LH, s.B);
  post_logits_act_kernel<T, C><<<grid, NT, 0, st>>>(logit, static_cast<const T*>(act), s, vs, w, b, hp, out, counter,
                                                    capacity);
  return cudaGetLastError();
}

cudaError_t launch_post_logits_act(int dt, const float* logit, const void* act, ActShape s, ViewSet vs,
                                   const float* w_head, const float* b_head, HeadParams hp, smlm_emitter* out,
                                   unsigned long long* counter, unsigned long long capacity, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  if (dt == ACT_BF16) {
    SMLM_DISPATCH_C(__nv_bfloat16, post_logits_act_tc, logit, act, s, vs, w_head, b_head, hp, out, counter, capacity, st)
  } else if (dt == ACT_F16) {
    SMLM_DISPATCH_C(__half, post_logits_act_tc, logit, act, s, vs, w_head, b_head, hp, out, counter, capacity, st)
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_head_maps(int dt, const void* act, ActShape s, const float* w_head,
                             const float* b_head, int n_h, float* maps, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  if (dt == ACT_BF16) {
    SMLM_DISPATCH_C(__nv_bfloat16, head_maps_tc, act, s, w_head, b_head, n_h, maps, st)
  } else if (dt == ACT_F16) {
    SMLM_DISPATCH_C(__half, head_maps_tc, act, s, w_head, b_head, n_h, maps, st)
  } else {
    SMLM_DISPATCH_C(float, head_maps_tc, act, s, w_head, b_head, n_h, maps, st)
  }
}

cudaError_t launch_dump_act(int dt, const void* act, ActShape s, float* dst, size_t view_stride,
                            cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  dim3 grid((s.W + NT - 1) / NT, s.H, s.B);
  if (dt == ACT_BF16)
    dump_act_kernel<__nv_bfloat16><<<grid, NT, 0, st>>>((const __nv_bfloat16*)act, s, dst, view_stride);
  else if (dt == ACT_F16)
    dump_act_kernel<__half><<<grid, NT, 0, st>>>((const __half*)act, s, dst, view_stride);
  else
    dump_act_kernel<float><<<grid, NT, 0, st>>>((const float*)act, s, dst, view_stride);
  return cudaGetLastError();
}

cudaError_t launch_post_from_maps(const float* maps, int n, int H, int W, HeadParams hp,
                                  smlm_emitter* out, unsigned long long* counter,
                                  unsigned long long capacity, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  dim3 grid((W + TW - 1) / TW, (H + TH - 1) / TH, n);
  post_from_maps_kernel<<<grid, NT, 0, st>>>(maps, H, W, hp, out, counter, capacity);
  return cudaGetLastError();
}

cudaError_t launch_snapshot(const unsigned long long* counter, unsigned long long capacity,
                            unsigned long long* snap, cudaStream_t st) {
  snapshot_kernel<<<1, 1, 0, st>>>(counter, capacity, snap);
  return cudaGetLastError();
}

cudaError_t launch_flush_emitters(const smlm_emitter* dev, smlm_emitter* host_mapped,
                                  const unsigned long long* lo, const unsigned long long* hi,
                                  cudaStream_t st) {
  flush_kernel<<<64, NT, 0, st>>>(dev, host_mapped, lo, hi);
  return cudaGetLastError();
}

}  // namespace smlm
