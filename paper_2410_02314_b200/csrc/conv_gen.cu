// Convolutions of the paper's own topology (dloc.h): 3x3 (any dilation)
// or 1x1, C_in != C_out, over a range of planes of a concatenation buffer, bias + optional
// ReLU in the epilogue.  Two kernels with the same interface (dloc_internal.cuh, ConvGen):
//
//  * conv_gen_umma_kernel: implicit GEMM on tcgen05 / TMEM / TMA (sm_100a).  One work item =
//    (output-channel group of NT <= 128 channels, view, image row, 128-pixel segment):
//    D[128 px x NT] = sum over K-steps of 16 input channels and k x k taps of
//    A[128 x 16] B[16 x NT].  Per K-step one shared-memory stage holds the k input rows of
//    the two channel-chunk planes (each a 1-D bulk copy of (128 + 2 pad) pixels x 16 B: in the
//    chunk-planar layout that IS the K-major no-swizzle operand, and a horizontal tap is a
//    16-byte shift of the descriptor address, at any dilation) and the k x k weight tiles of
//    that K-step (pre-packed, one bulk copy).  Rows outside the image are skipped (their taps
//    contribute zero), columns outside are bulk-copied zeros.  Warp roles: 0 = TMA producer,
//    1 = MMA issuer (one elected thread), 2-5 = epilogue (one TMEM lane quadrant each).  The
//    accumulator is double-buffered in TMEM, so the epilogue of tile t overlaps the MMAs of
//    tile t + 1; persistent CTAs stride over the tiles.
//    Unlike conv_umma.cu (C_in = C_out <= 64, weights resident, N = 3C row-chain walk) the
//    weights are streamed with the activations: with C_in up to 6 C0 and C_out up to 4 C0 they
//    do not fit next to the stages.  They stay L2-resident (<= 1 MB per layer).
//  * conv_gen_direct_kernel: the CUDA-core twin, fp32 math - the reference mode (SMLM_FP32,
//    1e-4 against the oracle) and the cross-check of the tensor-core kernel in 16-bit mode.
//
// Plus the small data-movement kernels of the U-Net (2x2 max pooling, nearest up-sampling),
// the planar debug dump, and detection + decode on the ten head maps.
#include <math_constants.h>

#include <cstring>

#include "chunk_io.cuh"
#include "dloc_internal.cuh"
#include "umma_ptx.cuh"
#include "../../include/dloc.h"

namespace smlm {
namespace {

using namespace ptx;

constexpr int kGThreads = 192;
constexpr int kGTileM = 128;
constexpr int kGMaxStages = 8;
constexpr int kGTmemCols = 256;  // two accumulator buffers of NT <= 128 columns
constexpr uint32_t kGSmemBudget = 200u * 1024u;

__device__ __align__(16) uint4 g_gen_zeros[160];  // (127 + 16) pixels x 16 B of zero padding

struct GenGeo {
  int NT, ngroups, nseg, ksteps, pad, PW;
  uint32_t a_row_bytes;  // one input row of one plane in a stage: PW x 16
  uint32_t a_bytes;      // k rows x 2 planes
  uint32_t b_bytes;      // k x k taps x 2 chunks x NT rows x 16 B
  uint32_t stage_bytes;
  int nstage;
  long long total;
};

__host__ __device__ inline void tile_of(const GenGeo& g, const ConvGen& a, long long t, int& grp, int& x0, int& y,
                                         int& b) {
  grp = (int)(t % g.ngroups);
  long long r = t / g.ngroups;
  x0 = (int)(r % g.nseg) * kGTileM;
  r /= g.nseg;
  y = (int)(r % a.H);
  b = (int)(r / a.H);
}

template <bool F16>
__global__ void __launch_bounds__(kGThreads, 1)
    conv_gen_umma_kernel(const __grid_constant__ ConvGen a, const __grid_constant__ GenGeo g,
                         const uint8_t* __restrict__ wpack, const float* __restrict__ bias) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 127u) & ~127u;
  uint8_t* smem = smem_raw + (sbase - sraw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t bar0 = sbase + (uint32_t)g.nstage * g.stage_bytes;
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (kGMaxStages + s); };
  auto acc_full = [&](int i) { return bar0 + 8u * (2 * kGMaxStages + i); };
  auto acc_empty = [&](int i) { return bar0 + 8u * (2 * kGMaxStages + 2 + i); };
  const uint32_t tmem_word = bar0 + 8u * (2 * kGMaxStages + 4);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + (tmem_word - sbase));

  if (threadIdx.x == 0) {
    for (int s = 0; s < kGMaxStages; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(acc_full(i), 1);
      mbar_init(acc_empty(i), 4);  // one arrival per epilogue warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_word), "n"(kGTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int r = a.k / 2;

  if (warp == 0) {
    // =========================== TMA producer
    const uint8_t* in_b = reinterpret_cast<const uint8_t*>(a.in);
    uint32_t st = 0, par = 1;
    for (long long t = blockIdx.x; t < g.total; t += gridDim.x) {
      int grp, x0, y, b;
      tile_of(g, a, t, grp, x0, y, b);
      const int xl = x0 - g.pad, xr = x0 + kGTileM + g.pad;
      const int lo = xl > 0 ? xl : 0, hi = xr < a.W ? xr : a.W;
      const uint32_t pre = (uint32_t)(lo - xl) * 16u, mid = (uint32_t)(hi - lo) * 16u, post = (uint32_t)(xr - hi) * 16u;
      int nrows = 0;
      for (int ky = 0; ky < a.k; ++ky) {
        const int row = y + (ky - r) * a.d;
        nrows += (row >= 0 && row < a.H) ? 1 : 0;
      }
      const uint32_t tx = (uint32_t)nrows * 2u * g.a_row_bytes + g.b_bytes;
      for (int ks = 0; ks < g.ksteps; ++ks) {
        mbar_wait(empty_bar(st), par);
        if (elect_one()) {
          const uint32_t dst = sbase + st * g.stage_bytes;
          const uint32_t bar = full_bar(st);
          mbar_expect_tx(bar, tx);
          for (int ky = 0; ky < a.k; ++ky) {
            const int row = y + (ky - r) * a.d;
            if (row < 0 || row >= a.H) continue;
            for (int pl = 0; pl < 2; ++pl) {
              const size_t plane = (size_t)b * a.in_planes + a.ci_plane0 + 2 * ks + pl;
              const uint8_t* src = in_b + ((plane * a.H + row) * a.W + lo) * 16u;
              const uint32_t d0 = dst + (uint32_t)(ky * 2 + pl) * g.a_row_bytes;
              bulk_load(d0 + pre, src, mid, bar);
              if (pre) bulk_load(d0, g_gen_zeros, pre, bar);
              if (post) bulk_load(d0 + pre + mid, g_gen_zeros, post, bar);
            }
          }
          const uint8_t* wsrc = wpack + ((size_t)grp * g.ksteps + ks) * g.b_bytes;
          for (uint32_t off = 0; off < g.b_bytes; off += 16384u) {
            const uint32_t n = g.b_bytes - off < 16384u ? g.b_bytes - off : 16384u;
            bulk_load(dst + g.a_bytes + off, wsrc + off, n, bar);
          }
        }
        __syncwarp();
        if (++st == (uint32_t)g.nstage) {
          st = 0;
          par ^= 1u;
        }
      }
    }
  } else if (warp == 1) {
    // =========================== MMA issuer
    const uint32_t idesc = umma_idesc(kGTileM, g.NT, F16);
    uint32_t st = 0, par = 0;
    uint32_t it = 0;
    for (long long t = blockIdx.x; t < g.total; t += gridDim.x, ++it) {
      int grp, x0, y, b;
      tile_of(g, a, t, grp, x0, y, b);
      const uint32_t buf = it & 1u;
      mbar_wait(acc_empty(buf), ((it >> 1) & 1u) ^ 1u);  // the epilogue has drained this buffer
      tc_fence_after();
      const uint32_t dcol = tmem_base + buf * (uint32_t)g.NT;
      uint32_t acc = 0;
      for (int ks = 0; ks < g.ksteps; ++ks) {
        mbar_wait(full_bar(st), par);
        tc_fence_after();
        const uint32_t sa = sbase + st * g.stage_bytes;
        if (elect_one()) {
          uint32_t accl = acc;
          for (int ky = 0; ky < a.k; ++ky) {
            const int row = y + (ky - r) * a.d;
            if (row < 0 || row >= a.H) continue;
            for (int kx = 0; kx < a.k; ++kx) {
              const uint32_t aaddr = sa + (uint32_t)(ky * 2) * g.a_row_bytes + (uint32_t)(kx * a.d) * 16u;
              const uint32_t baddr = sa + g.a_bytes + (uint32_t)(ky * a.k + kx) * 2u * (uint32_t)g.NT * 16u;
              tc_mma(dcol, umma_desc(aaddr, g.a_row_bytes, 128u), umma_desc(baddr, (uint32_t)g.NT * 16u, 128u), idesc,
                     accl);
              accl = 1u;
            }
          }
          tc_commit(empty_bar(st));
          if (ks + 1 == g.ksteps) tc_commit(acc_full(buf));
        }
        __syncwarp();
        acc = 1u;  // the centre row is always inside the image: every K-step issues at least one MMA
        if (++st == (uint32_t)g.nstage) {
          st = 0;
          par ^= 1u;
        }
      }
    }
  } else {
    // =========================== epilogue: warps 2..5, TMEM lane quadrant = warp % 4
    const int q = warp & 3;
    const int px = q * 32 + lane;
    uint32_t it = 0;
    const size_t plane_px = (size_t)a.H * a.W;
    for (long long t = blockIdx.x; t < g.total; t += gridDim.x, ++it) {
      int grp, x0, y, b;
      tile_of(g, a, t, grp, x0, y, b);
      const uint32_t buf = it & 1u;
      mbar_wait(acc_full(buf), (it >> 1) & 1u);
      tc_fence_after();
      const int x = x0 + px;
      const uint32_t tl = tmem_base + ((uint32_t)(q * 32) << 16) + buf * (uint32_t)g.NT;
      for (int c16 = 0; c16 < g.NT; c16 += 16) {
        uint32_t v[16];
        tc_ld16(tl + (uint32_t)c16, v);
        tc_wait_ld();
        const int ch0 = grp * g.NT + c16;
        float f[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          f[i] = __uint_as_float(v[i]) + __ldg(bias + ch0 + i);
          if (a.relu) f[i] = fmaxf(f[i], 0.0f);
        }
        if (x < a.W) {
          if (a.out_f32) {
#pragma unroll
            for (int i = 0; i < 16; ++i)
              if (ch0 + i < a.n_valid) a.out_f32[((size_t)b * a.n_valid + ch0 + i) * plane_px + (size_t)y * a.W + x] = f[i];
          } else {
            uint4* o = reinterpret_cast<uint4*>(a.out) +
                       (((size_t)b * a.out_planes + a.co_plane0 + (ch0 >> 3)) * a.H + y) * a.W + x;
            o[0] = make_uint4(pack2<F16>(f[0], f[1]), pack2<F16>(f[2], f[3]), pack2<F16>(f[4], f[5]),
                              pack2<F16>(f[6], f[7]));
            o[plane_px] = make_uint4(pack2<F16>(f[8], f[9]), pack2<F16>(f[10], f[11]), pack2<F16>(f[12], f[13]),
                                     pack2<F16>(f[14], f[15]));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(acc_empty(buf));
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kGTmemCols) : "memory");
  }
}

// ------------------------------------------------------------------------------ CUDA-core twin
// One block = 128 pixels of one row x 16 output channels; one thread per pixel.  The weights
// of one tap ([CI][16]) are staged in shared memory; fixed summation order (tap, ci).
template <typename T>
__global__ void __launch_bounds__(128)
    conv_gen_direct_kernel(const ConvGen a, const float* __restrict__ w /*[k*k][CI][CO]*/,
                           const float* __restrict__ bias) {
  extern __shared__ float ws[];  // [CI][16]
  // grid.x runs over (view, row): B * H may exceed the 65535 limit of grid.y / grid.z
  const int x = blockIdx.y * 128 + threadIdx.x;
  const int y = blockIdx.x % a.H, b = blockIdx.x / a.H;
  const int co0 = blockIdx.z * 16;
  const int r = a.k / 2;
  float acc[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) acc[i] = bias[co0 + i];
  ActShape si{a.B, a.CI, a.H, a.W, a.in_planes * 8};
  for (int tap = 0; tap < a.k * a.k; ++tap) {
    __syncthreads();
    for (int i = threadIdx.x; i < a.CI * 16; i += 128)
      ws[i] = w[((size_t)tap * a.CI + i / 16) * a.CO + co0 + i % 16];
    __syncthreads();
    const int yy = y + (tap / a.k - r) * a.d, xx = x + (tap % a.k - r) * a.d;
    if (x >= a.W || yy < 0 || yy >= a.H || xx < 0 || xx >= a.W) continue;
    for (int kc = 0; kc < a.CI / 8; ++kc) {
      float v[8];
      Chunk<T>::load(a.in, si.chunk_index(b, a.ci_plane0 + kc, yy, xx), v);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const float* wr = ws + (kc * 8 + j) * 16;
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = fmaf(v[j], wr[i], acc[i]);
      }
    }
  }
  if (x >= a.W) return;
  if (a.relu) {
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = fmaxf(acc[i], 0.0f);
  }
  if (a.out_f32) {
    for (int i = 0; i < 16; ++i)
      if (co0 + i < a.n_valid)
        a.out_f32[(((size_t)b * a.n_valid + co0 + i) * a.H + y) * a.W + x] = acc[i];
  } else {
    ActShape so{a.B, a.CO, a.H, a.W, a.out_planes * 8};
    Chunk<T>::store(a.out, so.chunk_index(b, a.co_plane0 + (co0 >> 3), y, x), acc);
    Chunk<T>::store(a.out, so.chunk_index(b, a.co_plane0 + (co0 >> 3) + 1, y, x), acc + 8);
  }
}

// ------------------------------------------------------------------------------ U-Net data movement
template <typename T>
__global__ void pool2_kernel(const T* __restrict__ in, int in_planes, int pi0, T* __restrict__ out, int out_planes,
                             int po0, int np, int B, int H, int W) {
  const int Ho = H / 2, Wo = W / 2;
  const size_t n = (size_t)B * np * Ho * Wo;
  ActShape si{B, np * 8, H, W, in_planes * 8}, so{B, np * 8, Ho, Wo, out_planes * 8};
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int x = (int)(i % Wo);
    size_t t = i / Wo;
    const int y = (int)(t % Ho);
    t /= Ho;
    const int p = (int)(t % np), b = (int)(t / np);
    float m[8], v[8];
    Chunk<T>::load(in, si.chunk_index(b, pi0 + p, 2 * y, 2 * x), m);
#pragma unroll
    for (int q = 1; q < 4; ++q) {
      Chunk<T>::load(in, si.chunk_index(b, pi0 + p, 2 * y + (q >> 1), 2 * x + (q & 1)), v);
#pragma unroll
      for (int c = 0; c < 8; ++c) m[c] = fmaxf(m[c], v[c]);
    }
    Chunk<T>::store(out, so.chunk_index(b, po0 + p, y, x), m);
  }
}

template <typename T>
__global__ void up2_kernel(const T* __restrict__ in, int in_planes, int pi0, int H, int W, T* __restrict__ out,
                           int out_planes, int po0, int np, int B, int Ho, int Wo) {
  const size_t n = (size_t)B * np * Ho * Wo;
  ActShape si{B, np * 8, H, W, in_planes * 8}, so{B, np * 8, Ho, Wo, out_planes * 8};
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int x = (int)(i % Wo);
    size_t t = i / Wo;
    const int y = (int)(t % Ho);
    t /= Ho;
    const int p = (int)(t % np), b = (int)(t / np);
    const int ys = y / 2 < H - 1 ? y / 2 : H - 1, xs = x / 2 < W - 1 ? x / 2 : W - 1;
    float v[8];
    Chunk<T>::load(in, si.chunk_index(b, pi0 + p, ys, xs), v);
    Chunk<T>::store(out, so.chunk_index(b, po0 + p, y, x), v);
  }
}

template <typename T>
__global__ void dump_planar_kernel(const T* __restrict__ in, int in_planes, int p0, int np, int B, int H, int W,
                                   float* __restrict__ dst, size_t view_stride) {
  const size_t n = (size_t)B * np * H * W;
  ActShape si{B, np * 8, H, W, in_planes * 8};
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int x = (int)(i % W);
    size_t t = i / W;
    const int y = (int)(t % H);
    t /= H;
    const int p = (int)(t % np), b = (int)(t / np);
    float v[8];
    Chunk<T>::load(in, si.chunk_index(b, p0 + p, y, x), v);
    for (int c = 0; c < 8; ++c) dst[(size_t)b * view_stride + ((size_t)(p * 8 + c) * H + y) * W + x] = v[c];
  }
}

// ------------------------------------------------------------------------------ detection + decode, ten heads
// The rule of smlm.h (head_post.cu) on fp32 maps [n][10][H][W]: logit-domain threshold, 3x3
// local maximum with the lower-index tie rule, six-head decode, plus the uncertainty heads.
constexpr int PW_ = 64, PH_ = 16, PNT = 256;
constexpr int PCAND = (PW_ / 2) * (PH_ / 2);
__device__ inline float sigmoid_g(float v) { return 1.0f / (1.0f + expf(-v)); }
__device__ inline float softplus_g(float v) { return fmaxf(v, 0.0f) + log1pf(expf(-fabsf(v))); }

__global__ void __launch_bounds__(PNT)
    dloc_post_kernel(const float* __restrict__ maps, int H, int W, int frame0, DlocPostParams pp,
                     dloc_emitter* __restrict__ out, unsigned long long* __restrict__ counter,
                     unsigned long long capacity) {
  __shared__ float lg[PH_ + 2][PW_ + 2];
  __shared__ int cnd[PCAND];
  __shared__ int ncand;
  __shared__ unsigned long long base;
  const int tid = threadIdx.x, b = blockIdx.z;
  const int x0 = blockIdx.x * PW_, y0 = blockIdx.y * PH_;
  const size_t px = (size_t)H * W;
  const float* m = maps + (size_t)b * DLOC_HEADS * px;
  if (tid == 0) ncand = 0;
  for (int i = tid; i < (PH_ + 2) * (PW_ + 2); i += PNT) {
    const int ly = i / (PW_ + 2), lx = i - ly * (PW_ + 2);
    const int y = y0 + ly - 1, x = x0 + lx - 1;
    lg[ly][lx] = (y >= 0 && y < H && x >= 0 && x < W) ? __ldg(m + (size_t)y * W + x) : -CUDART_INF_F;
  }
  __syncthreads();
  for (int i = tid; i < PH_ * PW_; i += PNT) {
    const int ly = i / PW_, lx = i - ly * PW_;
    const int y = y0 + ly, x = x0 + lx;
    bool keep = y < H && x < W;
    if (keep) {
      const float c = lg[ly + 1][lx + 1];
      keep = (c > pp.hp.lthr) && c > lg[ly][lx] && c > lg[ly][lx + 1] && c > lg[ly][lx + 2] && c > lg[ly + 1][lx] &&
             c >= lg[ly + 1][lx + 2] && c >= lg[ly + 2][lx] && c >= lg[ly + 2][lx + 1] && c >= lg[ly + 2][lx + 2];
    }
    const unsigned mk = __ballot_sync(0xffffffffu, keep);
    if (mk) {
      const int lane = tid & 31, leader = __ffs(mk) - 1;
      int slot = 0;
      if (lane == leader) slot = atomicAdd(&ncand, __popc(mk));
      slot = __shfl_sync(0xffffffffu, slot, leader);
      if (keep) cnd[slot + __popc(mk & ((1u << lane) - 1u))] = i;
    }
  }
  __syncthreads();
  const int n = ncand;
  if (n == 0) return;
  if (tid == 0) base = atomicAdd(counter, (unsigned long long)n);
  __syncthreads();
  if (tid >= n) return;
  const unsigned long long slot = base + tid;
  if (slot >= capacity) return;
  const int i = cnd[tid];
  const int ly = i / PW_, lx = i - ly * PW_;
  const int y = y0 + ly, x = x0 + lx;
  const size_t q = (size_t)y * W + x;
  const HeadParams& hp = pp.hp;
  dloc_emitter e;
  e.frame = frame0 + b;
  e.pix = y * W + x;
  e.x_nm = ((float)x + hp.xy_scale * tanhf(m[1 * px + q])) * hp.pixel_size_nm;
  e.y_nm = ((float)y + hp.xy_scale * tanhf(m[2 * px + q])) * hp.pixel_size_nm;
  e.z_nm = hp.z_scale_nm * tanhf(m[3 * px + q]);
  e.photons = hp.photon_scale * softplus_g(m[4 * px + q]);
  e.bg = hp.bg_scale * softplus_g(m[5 * px + q]);
  e.p = sigmoid_g(lg[ly + 1][lx + 1]);
  e.sx_nm = pp.sigma_xy_px * sigmoid_g(m[6 * px + q]) * hp.pixel_size_nm;
  e.sy_nm = pp.sigma_xy_px * sigmoid_g(m[7 * px + q]) * hp.pixel_size_nm;
  e.sz_nm = pp.sigma_z_nm * sigmoid_g(m[8 * px + q]);
  e.s_photons = pp.sigma_photons * sigmoid_g(m[9 * px + q]);
  uint4* dst = reinterpret_cast<uint4*>(out + slot);
  const uint4* sv = reinterpret_cast<const uint4*>(&e);
  dst[0] = sv[0];
  dst[1] = sv[1];
  dst[2] = sv[2];
}

uint16_t bits16(float f, bool f16) {
  if (f16) {
    const __half h = __float2half_rn(f);
    uint16_t u;
    std::memcpy(&u, &h, 2);
    return u;
  }
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

GenGeo make_geo(const ConvGen& a) {
  GenGeo g;
  g.NT = conv_gen_ntile(a.CO);
  g.ngroups = a.CO / g.NT;
  g.nseg = (a.W + kGTileM - 1) / kGTileM;
  g.ksteps = a.CI / 16;
  g.pad = a.k == 3 ? a.d : 0;
  g.PW = kGTileM + 2 * g.pad;
  g.a_row_bytes = (uint32_t)g.PW * 16u;
  g.a_bytes = (uint32_t)a.k * 2u * g.a_row_bytes;
  g.b_bytes = (uint32_t)(a.k * a.k) * 2u * (uint32_t)g.NT * 16u;
  g.stage_bytes = (g.a_bytes + g.b_bytes + 127u) & ~127u;
  int ns = (int)(kGSmemBudget / g.stage_bytes);
  g.nstage = ns > kGMaxStages ? kGMaxStages : ns;
  g.total = (long long)g.ngroups * a.B * a.H * g.nseg;
  return g;
}

inline int grid_for(size_t n, int block) {
  size_t gsz = (n + block - 1) / block;
  return (int)(gsz > 148 * 16 ? 148 * 16 : (gsz < 1 ? 1 : gsz));
}

}  // namespace

int conv_gen_ntile(int CO) {
  if (CO <= 128) return CO;
  for (int nt = 128; nt >= 16; nt -= 16)
    if (CO % nt == 0) return nt;
  return 16;
}

size_t conv_gen_packed_bytes(int CI, int CO, int k) { return (size_t)CO * CI * k * k * 2; }

void conv_gen_pack_host(int CI, int CO, int CO_real, int k, const float* w, void* dst, bool f16) {
  const int NT = conv_gen_ntile(CO), ng = CO / NT, KS = CI / 16, taps = k * k;
  uint16_t* o = static_cast<uint16_t*>(dst);
  for (int gi = 0; gi < ng; ++gi)
    for (int ks = 0; ks < KS; ++ks)
      for (int tap = 0; tap < taps; ++tap)
        for (int kc = 0; kc < 2; ++kc)
          for (int n = 0; n < NT; ++n)
            for (int j = 0; j < 8; ++j) {
              const int co = gi * NT + n, ci = ks * 16 + kc * 8 + j;
              const float v = co < CO_real ? w[((size_t)co * CI + ci) * taps + tap] : 0.0f;
              o[(((((size_t)gi * KS + ks) * taps + tap) * 2 + kc) * NT + n) * 8 + j] = bits16(v, f16);
            }
}

cudaError_t launch_conv_gen_umma(bool f16, const ConvGen& a, const void* wpack, const float* bias, int n_sm,
                                 cudaStream_t st) {
  if (a.B <= 0) return cudaSuccess;
  if (a.CI % 16 || a.CO % 16 || a.CI < 16 || a.CO < 16 || (a.k != 1 && a.k != 3) || a.d < 1 || a.d > 16)
    return cudaErrorInvalidValue;
  const GenGeo g = make_geo(a);
  if (g.nstage < 2) return cudaErrorInvalidValue;
  const size_t smem = (size_t)g.nstage * g.stage_bytes + 8u * (2 * kGMaxStages + 4) + 16u + 128u;
  static bool attr_done[2][64] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  if (!attr_done[f16][dev]) {
    cudaError_t e = f16 ? cudaFuncSetAttribute(conv_gen_umma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               227 * 1024)
                        : cudaFuncSetAttribute(conv_gen_umma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               227 * 1024);
    if (e != cudaSuccess) return e;
    attr_done[f16][dev] = true;
  }
  const int grid = (int)(g.total < n_sm ? g.total : n_sm);
  if (f16)
    conv_gen_umma_kernel<true><<<grid, kGThreads, smem, st>>>(a, g, (const uint8_t*)wpack, bias);
  else
    conv_gen_umma_kernel<false><<<grid, kGThreads, smem, st>>>(a, g, (const uint8_t*)wpack, bias);
  return cudaGetLastError();
}

cudaError_t launch_conv_gen_direct(int dt, const ConvGen& a, const float* w, const float* bias, cudaStream_t st) {
  if (a.B <= 0) return cudaSuccess;
  dim3 grid(a.B * a.H, (a.W + 127) / 128, a.CO / 16);
  const size_t smem = (size_t)a.CI * 16 * sizeof(float);
  if (dt == ACT_BF16) conv_gen_direct_kernel<__nv_bfloat16><<<grid, 128, smem, st>>>(a, w, bias);
  else if (dt == ACT_F16) conv_gen_direct_kernel<__half><<<grid, 128, smem, st>>>(a, w, bias);
  else conv_gen_direct_kernel<float><<<grid, 128, smem, st>>>(a, w, bias);
  return cudaGetLastError();
}

#define DLOC_BY_TYPE(KERNEL, GRID, ...)                                                   \
  if (dt == ACT_BF16) KERNEL<__nv_bfloat16><<<GRID, 256, 0, st>>>((const __nv_bfloat16*)in, __VA_ARGS__); \
  else if (dt == ACT_F16) KERNEL<__half><<<GRID, 256, 0, st>>>((const __half*)in, __VA_ARGS__);          \
  else KERNEL<float><<<GRID, 256, 0, st>>>((const float*)in, __VA_ARGS__);

cudaError_t launch_pool2(int dt, const void* in, int in_planes, int pi0, void* out, int out_planes, int po0, int np,
                         int B, int H, int W, cudaStream_t st) {
  const size_t n = (size_t)B * np * (H / 2) * (W / 2);
  if (n == 0) return cudaSuccess;
  const int grid = grid_for(n, 256);
  if (dt == ACT_BF16)
    pool2_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>((const __nv_bfloat16*)in, in_planes, pi0, (__nv_bfloat16*)out,
                                                      out_planes, po0, np, B, H, W);
  else if (dt == ACT_F16)
    pool2_kernel<__half><<<grid, 256, 0, st>>>((const __half*)in, in_planes, pi0, (__half*)out, out_planes, po0, np, B,
                                               H, W);
  else
    pool2_kernel<float><<<grid, 256, 0, st>>>((const float*)in, in_planes, pi0, (float*)out, out_planes, po0, np, B, H,
                                              W);
  return cudaGetLastError();
}

cudaError_t launch_up2(int dt, const void* in, int in_planes, int pi0, int H, int W, void* out, int out_planes,
                       int po0, int np, int B, int Ho, int Wo, cudaStream_t st) {
  const size_t n = (size_t)B * np * Ho * Wo;
  if (n == 0) return cudaSuccess;
  const int grid = grid_for(n, 256);
  if (dt == ACT_BF16)
    up2_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>((const __nv_bfloat16*)in, in_planes, pi0, H, W, (__nv_bfloat16*)out,
                                                    out_planes, po0, np, B, Ho, Wo);
  else if (dt == ACT_F16)
    up2_kernel<__half><<<grid, 256, 0, st>>>((const __half*)in, in_planes, pi0, H, W, (__half*)out, out_planes, po0, np,
                                             B, Ho, Wo);
  else
    up2_kernel<float><<<grid, 256, 0, st>>>((const float*)in, in_planes, pi0, H, W, (float*)out, out_planes, po0, np, B,
                                            Ho, Wo);
  return cudaGetLastError();
}

cudaError_t launch_dump_planar(int dt, const void* in, int in_planes, int p0, int np, int B, int H, int W,
                               float* dst, size_t view_stride, cudaStream_t st) {
  const size_t n = (size_t)B * np * H * W;
  if (n == 0) return cudaSuccess;
  const int grid = grid_for(n, 256);
  DLOC_BY_TYPE(dump_planar_kernel, grid, in_planes, p0, np, B, H, W, dst, view_stride)
  return cudaGetLastError();
}

cudaError_t launch_dloc_post(const float* maps, int n, int H, int W, int frame0, DlocPostParams pp, void* out48,
                             unsigned long long* counter, unsigned long long capacity, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  dim3 grid((W + PW_ - 1) / PW_, (H + PH_ - 1) / PH_, n);
  dloc_post_kernel<<<grid, PNT, 0, st>>>(maps, H, W, frame0, pp, (dloc_emitter*)out48, counter, capacity);
  return cudaGetLastError();
}

}  // namespace smlm
