// smlm_postprocess_static (include/smlm.h): the post-processing of head_post.cu's
// post_from_maps_kernel - threshold, 3x3 local-maximum test with the index tie rule, decode,
// compaction into one emitter list (BASELINE.json north_star (c); P:192 item 3) - for callers
// that must not allocate.
//
// Why it exists.  Every other entry point of the library lives on an smlm_ctx, and a ctx calls
// cudaMalloc: at smlm_create, and again inside smlm_localize whenever a shape or a capacity
// grows.  cudaMalloc and cudaFree take a device-wide lock and wait for the GPU to drain, and
// they can fail when another framework has reserved the card's memory for its own pool.  That
// rules them out for
//   - an acquisition loop that post-processes maps while the camera's next frames are being
//     copied in on another stream (a device-wide wait there drops frames),
//   - a plug-in that runs inside a host program (an inference server, another framework's custom
//     operator) which owns all device memory and hands the plug-in its buffers,
//   - code that runs after start-up in a process whose memory budget is fixed and audited.
// Such a caller passes the maps and the output list; the only other memory the method needs is
// the bookkeeping of the compaction, and here that lives in an array that is part of the
// library image itself (g_scratch below): it is there as soon as the library is loaded, on
// every GPU that loads it, until the process exits.
//
// What differs from the ctx path.  post_from_maps_kernel appends through one atomic counter, so
// its list order changes from run to run.  With a fixed scratch array an ordered compaction
// costs nothing extra to set up, so this variant is deterministic:
//   1. count_kernel   one block per 32 x 64 pixel tile: number of detections -> scratch word
//   2. scan_kernel    exclusive prefix sum of the words in place (one block), total -> *out_count
//   3. emit_kernel    the tile test again; detection j of tile t goes to list slot prefix[t] + j
// Records come out ordered by (frame, tile row, tile column, pixel within the tile).  Every
// scratch word a call reads was written earlier in the same call, so nothing has to be cleared
// between calls - but two calls whose kernels overlap on the GPU (different streams, or the same
// device from two threads) use the same words and corrupt each other.
//
// The arithmetic of a record is the same sequence of fp32 operations as detect_tile
// (head_post.cu), restated here so that no existing code path changes.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdarg.h>
#include <stdio.h>

#include <cmath>
#include <mutex>

#include "../../include/smlm.h"

namespace {

constexpr int TW = 64, TH = 32, NT = 256;  // pixels per tile, threads per block
constexpr int NWORDS = TW * TH / 32;       // one keep-bit per pixel
constexpr int HEADER_BYTES = 256;
constexpr long long MAX_TILES = SMLM_POST_STATIC_MAX_TILES;
static_assert(HEADER_BYTES + MAX_TILES * 4 == SMLM_POST_STATIC_SCRATCH_BYTES, "scratch layout");

// The scratch memory.  File scope, so the loader places it in device memory when the module is
// loaded on a GPU; no allocation call is ever made for it.  Layout: 256 reserved bytes, then one
// 32-bit word per tile.  In HOST code this name is only a handle for cudaGetSymbolAddress - its
// host address is not device memory - so the launches below never pass `g_scratch` itself.
static __device__ __align__(256) unsigned char g_scratch[SMLM_POST_STATIC_SCRATCH_BYTES];

struct PostParams {
  const float* maps;  // [n][n_h][H][W] pre-activation head outputs
  int n_h, H, W, tiles_x, tiles_y;
  float lthr;  // logit(threshold): -inf => every local maximum, +inf => none
  float xy_scale, z_scale_nm, photon_scale, bg_scale, pixel_size_nm;
};

__device__ inline float sigmoid_f(float v) { return 1.0f / (1.0f + expf(-v)); }
__device__ inline float softplus_f(float v) { return fmaxf(v, 0.0f) + log1pf(expf(-fabsf(v))); }

struct TileSmem {
  float lg[TH + 2][TW + 2];
  unsigned keep[NWORDS];
  unsigned before[NWORDS];  // detections of the tile in earlier words
};

// Detection logit patch of tile `t` -> sm.lg; keep-bit of every pixel -> sm.keep.
// Returns through b / y0 / x0 where the tile sits.  Ends with a __syncthreads.
__device__ inline void tile_test(const PostParams& p, unsigned t, TileSmem& sm, int& b, int& y0, int& x0) {
  const int tid = threadIdx.x;
  const unsigned per_frame = (unsigned)(p.tiles_x * p.tiles_y);
  b = (int)(t / per_frame);
  const unsigned r = t - (unsigned)b * per_frame;
  y0 = (int)(r / p.tiles_x) * TH;
  x0 = (int)(r % p.tiles_x) * TW;
  const float* lmap = p.maps + (size_t)b * p.n_h * p.H * p.W;  // head 0 = detection logit
  // outside the frame the logit is -inf: such a neighbour never wins
  for (int i = tid; i < (TH + 2) * (TW + 2); i += NT) {
    const int ly = i / (TW + 2), lx = i - ly * (TW + 2);
    const int y = y0 + ly - 1, x = x0 + lx - 1;
    sm.lg[ly][lx] = (y >= 0 && y < p.H && x >= 0 && x < p.W) ? lmap[(size_t)y * p.W + x] : -CUDART_INF_F;
  }
  __syncthreads();
  // neighbours with a lower linear index (row above, left) must be strictly smaller, the others
  // may be equal.  i = tid + k * NT: the 32 lanes of a warp hold the 32 pixels of word i / 32.
  for (int i = tid; i < TH * TW; i += NT) {
    const int ly = i / TW, lx = i - ly * TW;
    bool keep = (y0 + ly < p.H) && (x0 + lx < p.W);
    if (keep) {
      const float c = sm.lg[ly + 1][lx + 1];
      keep = (c > p.lthr) && c > sm.lg[ly][lx] && c > sm.lg[ly][lx + 1] && c > sm.lg[ly][lx + 2] &&
             c > sm.lg[ly + 1][lx] && c >= sm.lg[ly + 1][lx + 2] && c >= sm.lg[ly + 2][lx] &&
             c >= sm.lg[ly + 2][lx + 1] && c >= sm.lg[ly + 2][lx + 2];
    }
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    if ((tid & 31) == 0) sm.keep[i >> 5] = m;
  }
  __syncthreads();
}

__global__ void __launch_bounds__(NT) count_kernel(PostParams p, unsigned* __restrict__ tile_words) {
  __shared__ TileSmem sm;
  int b, y0, x0;
  tile_test(p, blockIdx.x, sm, b, y0, x0);
  if (threadIdx.x < 32) {
    unsigned c = __popc(sm.keep[threadIdx.x]) + __popc(sm.keep[threadIdx.x + 32]);
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (threadIdx.x == 0) tile_words[blockIdx.x] = c;
  }
}

// In-place exclusive prefix sum of words[0, n) by ONE block of 1024 threads, 1024 words per
// round with a running carry.  A tile holds at most 512 detections and n <= MAX_TILES, so the
// total stays below 2^27.
__global__ void __launch_bounds__(1024) scan_kernel(unsigned* __restrict__ words, unsigned n,
                                                    long long* __restrict__ out_count) {
  __shared__ unsigned warp_sum[32];
  __shared__ unsigned carry_s;
  const unsigned tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) carry_s = 0;
  __syncthreads();
  for (unsigned base = 0; base < n; base += 1024) {
    const unsigned i = base + tid;
    const unsigned v = i < n ? words[i] : 0u;
    unsigned inc = v;
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (unsigned)o) inc += u;
    }
    if (lane == 31) warp_sum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      unsigned s = warp_sum[lane];
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned u = __shfl_up_sync(0xffffffffu, s, o);
        if (lane >= (unsigned)o) s += u;
      }
      warp_sum[lane] = s;  // inclusive over warps
    }
    __syncthreads();
    const unsigned carry = carry_s;
    const unsigned excl = carry + (wid ? warp_sum[wid - 1] : 0u) + inc - v;
    if (i < n) words[i] = excl;
    __syncthreads();
    if (tid == 1023) carry_s = excl + v;
    __syncthreads();
  }
  if (tid == 0) *out_count = (long long)carry_s;
}

__global__ void __launch_bounds__(NT) emit_kernel(PostParams p, const unsigned* __restrict__ tile_words,
                                                  smlm_emitter* __restrict__ out, unsigned long long capacity) {
  __shared__ TileSmem sm;
  int b, y0, x0;
  tile_test(p, blockIdx.x, sm, b, y0, x0);
  const int tid = threadIdx.x;
  if (tid < NWORDS) {
    unsigned s = 0;
    for (int k = 0; k < tid; ++k) s += __popc(sm.keep[k]);
    sm.before[tid] = s;
  }
  __syncthreads();
  const unsigned long long first = tile_words[blockIdx.x];
  const float* fm = p.maps + (size_t)b * p.n_h * p.H * p.W;
  const size_t plane = (size_t)p.H * p.W;
  for (int i = tid; i < TH * TW; i += NT) {
    const unsigned m = sm.keep[i >> 5];
    if (!((m >> (i & 31)) & 1u)) continue;
    const unsigned long long slot = first + sm.before[i >> 5] + __popc(m & ((1u << (i & 31)) - 1u));
    if (slot >= capacity) continue;  // counted in *out_count, not stored
    const int ly = i / TW, lx = i - ly * TW;
    const int y = y0 + ly, x = x0 + lx;
    const size_t q = (size_t)y * p.W + x;
    const bool six = p.n_h == 6;
    const int hN = six ? 4 : 3;
    smlm_emitter e;
    e.frame = b;
    e.pix = y * p.W + x;
    e.x_nm = ((float)x + p.xy_scale * tanhf(fm[1 * plane + q])) * p.pixel_size_nm;
    e.y_nm = ((float)y + p.xy_scale * tanhf(fm[2 * plane + q])) * p.pixel_size_nm;
    e.z_nm = six ? p.z_scale_nm * tanhf(fm[3 * plane + q]) : 0.0f;
    e.photons = p.photon_scale * softplus_f(fm[hN * plane + q]);
    e.bg = p.bg_scale * softplus_f(fm[(hN + 1) * plane + q]);
    e.p = sigmoid_f(sm.lg[ly + 1][lx + 1]);
    uint4* dst = reinterpret_cast<uint4*>(out + slot);
    const uint4* src = reinterpret_cast<const uint4*>(&e);
    dst[0] = src[0];
    dst[1] = src[1];
  }
}

// ---- host side
thread_local char t_error[512] = "";

smlm_status fail(smlm_status st, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(t_error, sizeof t_error, fmt, ap);
  va_end(ap);
  return st;
}

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_dev[kMaxDevices];  // device address of g_scratch on each GPU, once known

// Device address of the scratch array on the CURRENT device.  The first call on a device asks
// the runtime for it (cudaGetSymbolAddress loads this library's device code on that GPU if it
// is not there yet - module loading, not an allocation); later calls read the cached pointer.
smlm_status scratch_address(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(SMLM_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(SMLM_ERR_INVALID_ARG, "device ordinal %d not supported (max %d)", dev, kMaxDevices - 1);
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_dev[dev]) {
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail(SMLM_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
    if (major != 10)
      return fail(SMLM_ERR_UNSUPPORTED_DEVICE, "device %d is sm_%dx; this library holds sm_100a code only", dev, major);
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_scratch);
    if (e != cudaSuccess || !ptr) {
      cudaGetLastError();
      return fail(SMLM_ERR_CUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
    }
    g_scratch_dev[dev] = static_cast<unsigned char*>(ptr);
  }
  *out = g_scratch_dev[dev];
  return SMLM_OK;
}

}  // namespace

extern "C" {

smlm_status smlm_postprocess_static(const float* maps, int64_t n_frames, int32_t H, int32_t W,
                                    const smlm_post_params* params, float threshold,
                                    smlm_emitter* out_emitters, int64_t capacity, int64_t* out_count,
                                    void* cuda_stream) {
  if (!params || !out_count) return fail(SMLM_ERR_INVALID_ARG, "params / out_count is NULL");
  if (n_frames < 0 || H < 1 || W < 1 || capacity < 0) return fail(SMLM_ERR_INVALID_ARG, "negative or zero size");
  if (params->head_channels != 5 && params->head_channels != 6)
    return fail(SMLM_ERR_INVALID_ARG, "head_channels must be 5 or 6");
  if (n_frames > 0 && !maps) return fail(SMLM_ERR_INVALID_ARG, "maps is NULL");
  if (capacity > 0 && (!out_emitters || (reinterpret_cast<uintptr_t>(out_emitters) & 15)))
    return fail(SMLM_ERR_INVALID_ARG, "out_emitters is NULL or not 16-byte aligned");
  if ((int64_t)H * W > INT32_MAX) return fail(SMLM_ERR_INVALID_ARG, "H * W exceeds the range of smlm_emitter.pix");
  const long long tx = (W + TW - 1) / TW, ty = (H + TH - 1) / TH;
  const long long tiles = tx * ty * (long long)n_frames;
  if (n_frames > INT32_MAX || tiles > MAX_TILES)
    return fail(SMLM_ERR_INVALID_ARG,
                "%lld frames of %d x %d are %lld tiles of %d x %d pixels; the static scratch array holds "
                "SMLM_POST_STATIC_MAX_TILES = %lld (at most %lld frames of this size per call): split the call",
                (long long)n_frames, H, W, tiles, TH, TW, MAX_TILES, MAX_TILES / (tx * ty));
  unsigned char* scratch = nullptr;
  smlm_status r = scratch_address(&scratch);
  if (r != SMLM_OK) return r;
  unsigned* tile_words = reinterpret_cast<unsigned*>(scratch + HEADER_BYTES);

  PostParams p;
  p.maps = maps;
  p.n_h = params->head_channels;
  p.H = H;
  p.W = W;
  p.tiles_x = (int)tx;
  p.tiles_y = (int)ty;
  if (threshold <= 0.0f) p.lthr = -INFINITY;
  else if (threshold >= 1.0f) p.lthr = INFINITY;
  else p.lthr = (float)std::log((double)threshold / (1.0 - (double)threshold));
  p.xy_scale = params->xy_scale;
  p.z_scale_nm = params->z_scale_nm;
  p.photon_scale = params->photon_scale;
  p.bg_scale = params->bg_scale;
  p.pixel_size_nm = params->pixel_size_nm;

  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaSuccess;
  if (tiles > 0) {
    count_kernel<<<(unsigned)tiles, NT, 0, st>>>(p, tile_words);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(SMLM_ERR_CUDA, "count_kernel: %s", cudaGetErrorString(e));
  }
  scan_kernel<<<1, 1024, 0, st>>>(tile_words, (unsigned)tiles, reinterpret_cast<long long*>(out_count));
  if ((e = cudaGetLastError()) != cudaSuccess) return fail(SMLM_ERR_CUDA, "scan_kernel: %s", cudaGetErrorString(e));
  if (tiles > 0 && capacity > 0) {
    emit_kernel<<<(unsigned)tiles, NT, 0, st>>>(p, tile_words, out_emitters, (unsigned long long)capacity);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(SMLM_ERR_CUDA, "emit_kernel: %s", cudaGetErrorString(e));
  }
  return SMLM_OK;
}

const char* smlm_postprocess_static_error(void) { return t_error; }

}  // extern "C"
