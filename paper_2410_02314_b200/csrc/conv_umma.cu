// K2: one trunk layer on the 5th-generation tensor cores (tcgen05 / TMEM / TMA), sm_100a.
//     out = in + ReLU(conv3x3, dilation d, zero padding d (in; W) + b)        (smlm.h)
// bf16 activations and weights, fp32 accumulation in TMEM, one RNE rounding of the stored
// result (BASELINE.json north_star (b)).
//
// Dataflow ("row-chain walk"):  an implicit GEMM with M = 128 consecutive pixels of
// one image row, K = C input channels per tap, and - instead of N = C - N = 3C: the three
// vertical taps of one horizontal tap share their A operand.  Input row q of the chain
// r, r+d, r+2d, ... contributes
//     W[ky=0] to output row q+1,  W[ky=1] to output row q,  W[ky=2] to output row q-1
// (chain indices), so ONE tcgen05.mma  D[128 x 3C] += A[128 x 16] * B[16 x 3C]  feeds three
// output rows that live in three TMEM slots of C columns each.  Every input row is read from
// L2 once (one TMA box of (128+2d) pixels x C channels) and is used by 3 x C/16 MMAs of
// N = 3C, which keeps the tensor pipe - not the shared-memory operand fetch - the limiter
// (N = C would re-read the 4 KB A tile for every 1.5 KB of B).
//   * slot of output o = (step id of its centre input) % 3; the B operand is the window
//     [m] of the weight rows stored as (ky = 1, 0, 2, 1, 0) so that the rotation is just a
//     different start address;
//   * after the MMAs of step u the output whose centre was step u-1 is complete: the
//     epilogue warps tcgen05.ld its slot, re-initialise the slot with the bias
//     (tcgen05.st - the next output accumulates on top, so the bias add is free), release
//     it, then apply ReLU + residual, round to bf16 and store;
//   * two independent "lanes" per CTA (own TMEM slots, own smem stages, own epilogue
//     warps) alternate on the single MMA-issuing thread, so one lane's epilogue overlaps
//     the other lane's MMAs;
//   * work = the sequence of all (view, 128-px segment, residue, chain row) row-tiles, cut
//     into 2 x gridDim equal contiguous ranges: balanced for any shape, at the cost of two
//     halo steps per range/chain boundary.
// The activation layout act[b][C/8][y][x][8] makes a TMA box land in shared memory as the
// UMMA "K-major, no swizzle" operand: core matrix = 8 pixels x 16 B, contiguous, so a
// horizontal tap is a 16-byte-granular shift of the descriptor start address.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <vector>

#include "smlm_internal.cuh"

namespace smlm {
namespace {

constexpr int kThreads = 384;  // warp 0 TMA, 1 MMA, 2 TMEM alloc, 3 idle, 4-7 / 8-11 epilogue lane 0 / 1
constexpr int kTileM = 128;
constexpr int kMaxStages = 4;
constexpr int kTmemCols = 512;
constexpr int kLaneCols = 256;  // TMEM columns reserved per lane (3C <= 192)

// ------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0,
                                            int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(dst),
      "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
      "l"(reinterpret_cast<uint64_t>(src)), "r"(bytes), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                       uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tc_st16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
      "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// UMMA shared-memory descriptor, K-major, no swizzle (cute::UMMA::SmemDescriptor):
// core matrix = 8 rows x 16 B, rows 16 B apart; SBO = bytes between 8-row groups along M/N,
// LBO = bytes between the two core matrices along K; version 1 (Blackwell) in bits 46-47.
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo >> 4) & 0x3FFFu) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// instruction descriptor (cute::UMMA::InstrDescriptor), kind::f16: D fp32, A/B bf16, K-major
__host__ __device__ constexpr uint32_t umma_idesc(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// ------------------------------------------------------------------------------ work iterator
struct Geo {
  int B, H, W, d;
  int nseg;  // 128-pixel segments per row
  int Lmax;  // chain rows per residue: ceil(H / d)
  long long total;  // B * nseg * d * Lmax row-tiles
};

struct Step {
  int b, x0;
  int in_row, out_row;
  bool in_valid, out_valid;
};

// All roles of a lane walk the same deterministic sequence of steps.  A lane owns the
// contiguous range [g, g1) of row-tiles; inside one chain a run of n rows takes n + 2 steps
// (inputs i0-1 .. i0+n; the output of chain index o is complete after the step of input o+1).
struct LaneIter {
  long long g, g1;
  int i0, n, j, r, b, x0;
  bool active;
  __device__ void init(const Geo& geo, int lane_id, int nlanes) {
    g = geo.total * lane_id / nlanes;
    g1 = geo.total * (lane_id + 1) / nlanes;
    active = false;
  }
  __device__ bool next(const Geo& geo, Step& s) {
    if (!active) {
      if (g >= g1) return false;
      long long chain = g / geo.Lmax;
      i0 = (int)(g - chain * geo.Lmax);
      long long rem = g1 - g;
      n = geo.Lmax - i0 < rem ? geo.Lmax - i0 : (int)rem;
      r = (int)(chain % geo.d);
      long long t = chain / geo.d;
      x0 = (int)(t % geo.nseg) * kTileM;
      b = (int)(t / geo.nseg);
      j = 0;
      active = true;
    }
    const int q = i0 - 1 + j;
    s.b = b;
    s.x0 = x0;
    s.in_row = r + q * geo.d;
    s.in_valid = q >= 0 && s.in_row < geo.H;
    s.out_row = r + (q - 1) * geo.d;
    s.out_valid = j >= 2 && s.out_row < geo.H;
    if (++j == n + 2) {
      active = false;
      g += n;
    }
    return true;
  }
};

struct SmemLayout {
  uint32_t w_off, w_bytes;
  uint32_t stage_off, stage_bytes;  // per (lane, stage)
  uint32_t bias_off;
  uint32_t bar_off;
  uint32_t tmem_off;
  uint32_t total;
  int nstage;
};

__host__ __device__ inline SmemLayout smem_layout(int C, int d, int nstage) {
  SmemLayout L;
  L.w_off = 0;
  L.w_bytes = 30u * C * C;  // 3 kx * C/8 chunks * 5C rows * 16 B
  L.stage_bytes = (((uint32_t)(C / 8) * (kTileM + 2 * d) * 16u) + 127u) & ~127u;
  L.stage_off = (L.w_off + L.w_bytes + 127u) & ~127u;
  L.nstage = nstage;
  L.bias_off = L.stage_off + 2u * nstage * L.stage_bytes;
  L.bar_off = L.bias_off + (uint32_t)C * 4u;
  // barriers: wbar, per lane: full[kMaxStages], empty[kMaxStages], acc_full, acc_free
  L.tmem_off = L.bar_off + 8u * (1 + 2 * (2 * kMaxStages + 2));
  L.total = L.tmem_off + 16u;
  return L;
}

template <int C>
__global__ void __launch_bounds__(kThreads, 1)
    conv_umma_kernel(const __grid_constant__ CUtensorMap tmap, const __nv_bfloat16* __restrict__ in,
                     __nv_bfloat16* __restrict__ out, Geo geo, const uint8_t* __restrict__ wpack,
                     const float* __restrict__ bias, int nstage) {
  extern __shared__ uint8_t smem_raw[];
  const SmemLayout L = smem_layout(C, geo.d, nstage);
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 1023u) & ~1023u;  // the launch reserves 1 KB of slack for this
  uint8_t* smem = smem_raw + (sbase - sraw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int d = geo.d;

  const uint32_t wbar = sbase + L.bar_off;
  auto full_bar = [&](int ln, int s) { return sbase + L.bar_off + 8u * (1 + ln * (2 * kMaxStages + 2) + s); };
  auto empty_bar = [&](int ln, int s) { return sbase + L.bar_off + 8u * (1 + ln * (2 * kMaxStages + 2) + kMaxStages + s); };
  auto acc_full_bar = [&](int ln) { return sbase + L.bar_off + 8u * (1 + ln * (2 * kMaxStages + 2) + 2 * kMaxStages); };
  auto acc_free_bar = [&](int ln) { return sbase + L.bar_off + 8u * (1 + ln * (2 * kMaxStages + 2) + 2 * kMaxStages + 1); };
  auto stage_addr = [&](int ln, int s) { return sbase + L.stage_off + (uint32_t)(ln * nstage + s) * L.stage_bytes; };
  float* bias_s = reinterpret_cast<float*>(smem + L.bias_off);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + L.tmem_off);

  // ---- one-time setup
  if (threadIdx.x == 0) {
    mbar_init(wbar, 1);
    for (int ln = 0; ln < 2; ++ln) {
      for (int s = 0; s < kMaxStages; ++s) {
        mbar_init(full_bar(ln, s), 1);
        mbar_init(empty_bar(ln, s), 1);
      }
      mbar_init(acc_full_bar(ln), 1);
      mbar_init(acc_free_bar(ln), 4);  // one arrival per epilogue warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + L.tmem_off),
                 "n"(kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int i = threadIdx.x; i < C; i += kThreads) bias_s[i] = bias[i];
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const int nlanes = 2 * gridDim.x;

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (lane == 0) {
      // the layer's weights: one bulk copy stream into shared memory, resident for the launch
      mbar_expect_tx(wbar, L.w_bytes);
      for (uint32_t off = 0; off < L.w_bytes; off += 16384u) {
        uint32_t n = L.w_bytes - off < 16384u ? L.w_bytes - off : 16384u;
        bulk_load(sbase + L.w_off + off, wpack + off, n, wbar);
      }
      LaneIter it[2];
      it[0].init(geo, 2 * blockIdx.x, nlanes);
      it[1].init(geo, 2 * blockIdx.x + 1, nlanes);
      uint32_t cnt[2] = {0, 0};
      bool more[2] = {true, true};
      const uint32_t box_bytes = (uint32_t)(C / 8) * (kTileM + 2 * d) * 16u;
      while (more[0] || more[1]) {
#pragma unroll
        for (int ln = 0; ln < 2; ++ln) {
          if (!more[ln]) continue;
          Step s;
          more[ln] = it[ln].next(geo, s);
          if (!more[ln] || !s.in_valid) continue;
          const int st = cnt[ln] % nstage;
          mbar_wait(empty_bar(ln, st), ((cnt[ln] / nstage) & 1) ^ 1);
          mbar_expect_tx(full_bar(ln, st), box_bytes);
          tma_load_5d(stage_addr(ln, st), &tmap, full_bar(ln, st), 0, s.x0 - d, s.in_row, 0, s.b);
          cnt[ln]++;
        }
      }
    }
  } else if (warp == 1) {
    // =========================== MMA issuer ===========================
    if (lane == 0) {
      mbar_wait(wbar, 0);
      LaneIter it[2];
      it[0].init(geo, 2 * blockIdx.x, nlanes);
      it[1].init(geo, 2 * blockIdx.x + 1, nlanes);
      uint32_t cnt[2] = {0, 0}, u[2] = {0, 0};
      bool more[2] = {true, true};
      constexpr uint32_t idesc = umma_idesc(kTileM, 3 * C);
      const uint32_t plane = (uint32_t)(kTileM + 2 * d) * 16u;  // bytes between channel chunks (A)
      constexpr uint32_t wplane = 5u * C * 16u;                 // bytes between channel chunks (B)
      while (more[0] || more[1]) {
#pragma unroll
        for (int ln = 0; ln < 2; ++ln) {
          if (!more[ln]) continue;
          Step s;
          more[ln] = it[ln].next(geo, s);
          if (!more[ln]) continue;
          const uint32_t uu = u[ln]++;
          int st = 0;
          if (s.in_valid) {
            st = cnt[ln] % nstage;
            mbar_wait(full_bar(ln, st), (cnt[ln] / nstage) & 1);
            cnt[ln]++;
          }
          mbar_wait(acc_free_bar(ln), uu & 1);  // slot (uu+2)%3 re-initialised by the epilogue
          tc_fence_after();
          if (s.in_valid) {
            // rows stored as ky = (1,0,2,1,0): window start for uu%3 = 0,1,2 is block 0,2,1
            const uint32_t m = uu % 3u;
            const uint32_t win = m == 0 ? 0u : (m == 1 ? 2u : 1u);
            const uint32_t a0 = stage_addr(ln, st);
            const uint32_t b0 = sbase + L.w_off + win * C * 16u;
            const uint32_t dcol = tmem_base + (uint32_t)ln * kLaneCols;
#pragma unroll
            for (int kx = 0; kx < 3; ++kx) {
#pragma unroll
              for (int ks = 0; ks < C / 16; ++ks) {
                const uint64_t ad = umma_desc(a0 + (uint32_t)(2 * ks) * plane + (uint32_t)(kx * d) * 16u, plane, 128u);
                const uint64_t bd = umma_desc(b0 + (uint32_t)(kx * (C / 8) + 2 * ks) * wplane, wplane, 128u);
                tc_mma(dcol, ad, bd, idesc, 1u);
              }
            }
            tc_commit(empty_bar(ln, st));
          }
          tc_commit(acc_full_bar(ln));
        }
      }
    }
  } else if (warp >= 4) {
    // =========================== epilogue ===========================
    const int ln = (warp - 4) >> 2;
    const int qd = warp & 3;  // TMEM lane quadrant this warp may access
    const int px = qd * 32 + lane;
    const uint32_t tlane = tmem_base + ((uint32_t)(qd * 32) << 16) + (uint32_t)ln * kLaneCols;
    auto init_slot = [&](uint32_t slot) {
#pragma unroll
      for (int g16 = 0; g16 < C / 16; ++g16) {
        uint32_t v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = __float_as_uint(bias_s[g16 * 16 + i]);
        tc_st16(tlane + slot * C + g16 * 16, v);
      }
    };
    init_slot(0);
    init_slot(1);
    init_slot(2);
    tc_wait_st();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(acc_free_bar(ln));

    LaneIter it;
    it.init(geo, 2 * blockIdx.x + ln, nlanes);
    Step s;
    uint32_t u = 0;
    const size_t plane_px = (size_t)geo.H * geo.W;
    while (it.next(geo, s)) {
      const uint32_t uu = u++;
      const uint32_t slot = (uu + 2u) % 3u;  // output whose centre input was step uu-1
      const int x = s.x0 + px;
      const bool store = s.out_valid && x < geo.W;
      uint4 res[C / 8];
      size_t pix = 0;
      if (store) {
        pix = ((size_t)s.b * (C / 8) * geo.H + s.out_row) * geo.W + x;
        const uint4* rp = reinterpret_cast<const uint4*>(in);
#pragma unroll
        for (int k = 0; k < C / 8; ++k) res[k] = __ldg(rp + pix + (size_t)k * plane_px);
      }
      __syncwarp();  // the tcgen05 ld/st below are warp-collective (.sync.aligned)
      mbar_wait(acc_full_bar(ln), uu & 1);
      tc_fence_after();
      uint32_t acc[C];
      if (s.out_valid) {
#pragma unroll
        for (int g16 = 0; g16 < C / 16; ++g16)
          tc_ld16(tlane + slot * C + g16 * 16, *reinterpret_cast<uint32_t(*)[16]>(&acc[g16 * 16]));
        tc_wait_ld();
      }
      init_slot(slot);
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(acc_free_bar(ln));
      if (store) {
        uint4* op = reinterpret_cast<uint4*>(out);
#pragma unroll
        for (int k = 0; k < C / 8; ++k) {
          const uint32_t rw[4] = {res[k].x, res[k].y, res[k].z, res[k].w};
          uint32_t ow[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            float r0 = __uint_as_float(rw[i] << 16), r1 = __uint_as_float(rw[i] & 0xffff0000u);
            float v0 = r0 + fmaxf(__uint_as_float(acc[k * 8 + 2 * i]), 0.0f);
            float v1 = r1 + fmaxf(__uint_as_float(acc[k * 8 + 2 * i + 1]), 0.0f);
            __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
            ow[i] = *reinterpret_cast<uint32_t*>(&h);
          }
          op[pix + (size_t)k * plane_px] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
        }
      }
    }
  }

  // ---- teardown
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
  }
}

// ------------------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

uint16_t bf16_bits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

template <int C>
cudaError_t launch_c(const CUtensorMap& map, const void* in, void* out, Geo geo, const void* wpack,
                     const float* bias, int nstage, int grid, size_t smem, cudaStream_t st) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(conv_umma_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  conv_umma_kernel<C><<<grid, kThreads, smem, st>>>(map, (const __nv_bfloat16*)in, (__nv_bfloat16*)out, geo,
                                                    (const uint8_t*)wpack, bias, nstage);
  return cudaGetLastError();
}

}  // namespace

struct UmmaPlan {
  const void* buf[2];
  ActShape s;
  int n_sm;
  CUtensorMap maps[2][9];  // [buffer][dilation]
  bool have[2][9];
};

size_t umma_packed_weight_bytes(int C) { return (size_t)30 * C * C; }

// Shared-memory image of one layer's weights: for kx, input chunk kc: 5C rows of 16 B
// (8 input channels), rows = output channels of ky = 1, 0, 2, 1, 0.
void umma_pack_weights_host(int C, const float* w /*[C][C][3][3]*/, void* dst) {
  static const int ky_seq[5] = {1, 0, 2, 1, 0};
  uint16_t* o = static_cast<uint16_t*>(dst);
  for (int kx = 0; kx < 3; ++kx)
    for (int kc = 0; kc < C / 8; ++kc)
      for (int n = 0; n < 5 * C; ++n) {
        const int ky = ky_seq[n / C], co = n % C;
        for (int j = 0; j < 8; ++j) {
          const int ci = kc * 8 + j;
          o[(((size_t)(kx * (C / 8) + kc) * 5 * C) + n) * 8 + j] =
              bf16_bits(w[(((size_t)co * C + ci) * 3 + ky) * 3 + kx]);
        }
      }
}

UmmaPlan* umma_plan_create(const void* buf0, const void* buf1, ActShape s, int n_sm, char* err, size_t errlen) {
  if (!get_encode()) {
    snprintf(err, errlen, "cuTensorMapEncodeTiled not available from the driver");
    return nullptr;
  }
  if (s.C % 16 || s.C < 16 || s.C > 64) {
    snprintf(err, errlen, "channels must be 16/32/48/64");
    return nullptr;
  }
  UmmaPlan* p = new UmmaPlan;
  p->buf[0] = buf0;
  p->buf[1] = buf1;
  p->s = s;
  p->n_sm = n_sm;
  std::memset(p->have, 0, sizeof p->have);
  return p;
}

void umma_plan_destroy(UmmaPlan* p) { delete p; }

cudaError_t launch_conv_umma(UmmaPlan* p, int src, int dil, const void* wpack, const float* bias,
                             int /*band_rows*/, cudaStream_t st, char* err, size_t errlen) {
  if (!p || dil < 1 || dil > 8 || src < 0 || src > 1) return cudaErrorInvalidValue;
  const ActShape& s = p->s;
  if (s.B <= 0) return cudaSuccess;
  if (!p->have[src][dil]) {
    // act[b][k][y][x][8] as a rank-5 tensor (8, W, H, C/8, B); box = one row segment with its
    // horizontal halo, all channel chunks.  Out-of-bounds elements are zero-filled: that IS the
    // convolution's zero padding (and the ragged right edge).
    cuuint64_t gdim[5] = {8, (cuuint64_t)s.W, (cuuint64_t)s.H, (cuuint64_t)(s.C / 8), (cuuint64_t)s.B};
    cuuint64_t gstr[4] = {16, (cuuint64_t)s.W * 16, (cuuint64_t)s.W * s.H * 16,
                          (cuuint64_t)s.W * s.H * (s.C / 8) * 16};
    cuuint32_t box[5] = {8, (cuuint32_t)(kTileM + 2 * dil), 1, (cuuint32_t)(s.C / 8), 1};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = get_encode()(&p->maps[src][dil], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(p->buf[src]),
                              gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      snprintf(err, errlen, "cuTensorMapEncodeTiled failed (%d) for %dx%dx%dx%d d=%d", (int)r, s.B, s.C, s.H, s.W, dil);
      return cudaErrorInvalidValue;
    }
    p->have[src][dil] = true;
  }
  Geo geo;
  geo.B = s.B;
  geo.H = s.H;
  geo.W = s.W;
  geo.d = dil;
  geo.nseg = (s.W + kTileM - 1) / kTileM;
  geo.Lmax = (s.H + dil - 1) / dil;
  geo.total = (long long)s.B * geo.nseg * dil * geo.Lmax;
  // stages: as many as fit next to the resident weights (<= kMaxStages)
  int nstage = kMaxStages;
  SmemLayout L = smem_layout(s.C, dil, nstage);
  while (nstage > 1 && L.total + 1024 > 227u * 1024u) L = smem_layout(s.C, dil, --nstage);
  if (L.total + 1024 > 227u * 1024u) {
    snprintf(err, errlen, "shared memory budget exceeded");
    return cudaErrorInvalidValue;
  }
  // at least ~12 row-tiles per lane, at most one CTA per SM
  long long want = (geo.total + 23) / 24;
  int grid = (int)(want < 1 ? 1 : (want > p->n_sm ? p->n_sm : want));
  const size_t smem = L.total + 1024;
  const void* in = p->buf[src];
  void* out = const_cast<void*>(p->buf[src ^ 1]);
  switch (s.C) {
    case 16: return launch_c<16>(p->maps[src][dil], in, out, geo, wpack, bias, nstage, grid, smem, st);
    case 32: return launch_c<32>(p->maps[src][dil], in, out, geo, wpack, bias, nstage, grid, smem, st);
    case 48: return launch_c<48>(p->maps[src][dil], in, out, geo, wpack, bias, nstage, grid, smem, st);
    case 64: return launch_c<64>(p->maps[src][dil], in, out, geo, wpack, bias, nstage, grid, smem, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace smlm
