// K2: one trunk layer on the 5th-generation tensor cores (tcgen05 / TMEM / TMA), sm_100a.
//     out = in + ReLU(conv3x3, dilation d, zero padding d (in; W) + b)        (smlm.h)
// bf16 activations and weights, fp32 accumulation in TMEM, one RNE rounding of the stored
// result (BASELINE.json north_star (b)).
//
// Dataflow ("row-chain walk"):  an implicit GEMM with M = 128
// consecutive pixels of one image row, K = C input channels per tap, and - instead of
// N = C - N = 3C: the three vertical taps of one horizontal tap share their A operand.
// Input row q of the chain r, r+d, r+2d, ... contributes
//     W[ky=0] to output row q+1,  W[ky=1] to output row q,  W[ky=2] to output row q-1
// (chain indices), so ONE tcgen05.mma  D[128 x 3C] += A[128 x 16] * B[16 x 3C]  feeds three
// output rows that live in three TMEM slots of C columns each.  Every input row is fetched
// once (C/8 bulk copies of (128+2d) pixels x 16 B) and is used by 3 x C/16 MMAs of N = 3C,
// which keeps the tensor pipe - not the shared-memory operand fetch - the limiter (N = C
// would re-read the 4 KB A tile for every 1.5 KB of B).
//   * slot of output o = (step id of its centre input) % 3; the B operand is the window
//     [m] of the weight rows stored as (ky = 1, 0, 2, 1, 0) so that the rotation is just a
//     different start address;
//   * after the MMAs of step u the output whose centre was step u-1 is complete: the
//     epilogue warps tcgen05.ld its slot, re-initialise the slot with the bias
//     (tcgen05.st - the next output accumulates on top, so the bias add is free), release
//     it, then apply ReLU + residual (read from the shared-memory stage, not from L2),
//     round to bf16 and store; the last layer also evaluates the detection head (HEAD);
//   * two independent "lanes" per CTA, each with its own producer warp, MMA-issuing warp,
//     four epilogue warps, TMEM slots and shared-memory stages: one lane's epilogue
//     overlaps the other lane's MMAs, and two issuing warps keep the tensor queue fed;
//   * work = the sequence of all (view, 128-px segment, residue, chain row) row-tiles, cut
//     into 2 x gridDim equal contiguous ranges: balanced for any shape, at the cost of two
//     halo steps per range/chain boundary;
//   * consecutive layers are chained by programmatic dependent launch: the prologue and the
//     weight load of layer l+1 overlap the tail of layer l.
// The activation layout act[b][C/8][y][x][8] makes a row segment of one chunk plane land in
// shared memory as the UMMA "K-major, no swizzle" operand: core matrix = 8 pixels x 16 B,
// contiguous, so a horizontal tap is a 16-byte-granular shift of the descriptor start address.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <vector>

#include "smlm_internal.cuh"

namespace smlm {
namespace {

constexpr int kThreads = 384;  // warps 0 / 2: TMA lane 0 / 1 (2 also owns TMEM alloc), 1 / 3: MMA lane 0 / 1, 4-7 / 8-11: epilogue
constexpr int kTileM = 128;
constexpr int kMaxStages = 6;
constexpr int kTmemCols = 512;
constexpr int kLaneCols = 256;  // TMEM columns reserved per lane (3C <= 192)
constexpr int kMaxDevices = 64;

// zero source for the padded parts of a row segment: at most (127 + 8) pixels x 16 B
__device__ __align__(16) uint4 g_zeros[160];

// Optional per-CTA cycle accounting (-DSMLM_PROF, used by ad-hoc probes only): slot i of CTA b
// is g_prof[b * 16 + i].
#ifdef SMLM_PROF
__device__ unsigned long long g_prof[1024 * 16];
#define PROF_DECL long long prof_acc[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}
#define PROF_T(var) const long long var = clock64()
#define PROF_ADD(i, v) prof_acc[i] += (long long)(v)
#define PROF_WAIT(i, stmt)          \
  do {                              \
    long long t0_ = clock64();      \
    stmt;                           \
    prof_acc[i] += clock64() - t0_; \
  } while (0)
#define PROF_FLUSH(cond)                                                             \
  if (cond) {                                                                        \
    for (int i_ = 0; i_ < 16; ++i_)                                                  \
      if (prof_acc[i_]) g_prof[blockIdx.x * 16 + i_] += (unsigned long long)prof_acc[i_]; \
  }
#else
#define PROF_DECL
#define PROF_T(var)
#define PROF_ADD(i, v)
#define PROF_WAIT(i, stmt) stmt
#define PROF_FLUSH(cond)
#endif

// ------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "elect.sync _|p, 0xffffffff;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(pred));
  return pred != 0;
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

// A lane owns the contiguous range [g, g1) of row-tiles and walks it as RUNS: n consecutive
// rows i0 .. i0+n-1 of one chain (view b, segment x0, residue r).  A run takes n + 2 steps
// j = 0 .. n+1: step j brings in chain row q = i0-1+j (image row r + q d, skipped when it is
// outside the image) and completes the output whose centre was the previous step's row
// (valid for j >= 2).  All roles of a lane walk the same deterministic sequence.
struct Run {
  int b, x0, r, i0, n;
};
struct LaneRuns {
  long long g, g1;
  __device__ void init(const Geo& geo, int lane_id, int nlanes) {
    g = geo.total * lane_id / nlanes;
    g1 = geo.total * (lane_id + 1) / nlanes;
  }
  __device__ bool next(const Geo& geo, Run& run) {
    if (g >= g1) return false;
    const long long chain = g / geo.Lmax;
    run.i0 = (int)(g - chain * geo.Lmax);
    const long long rem = g1 - g;
    run.n = geo.Lmax - run.i0 < rem ? geo.Lmax - run.i0 : (int)rem;
    run.r = (int)(chain % geo.d);
    const long long t = chain / geo.d;
    run.x0 = (int)(t % geo.nseg) * kTileM;
    run.b = (int)(t / geo.nseg);
    g += run.n;
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
  L.bar_off = L.bias_off + (uint32_t)(2 * C + 4) * 4u;  // layer bias, detection-head row + its bias
  // barriers: wbar, per lane: full[kMaxStages], empty[kMaxStages], acc_full, acc_free
  L.tmem_off = L.bar_off + 8u * (1 + 2 * (2 * kMaxStages + 2));
  L.total = L.tmem_off + 16u;
  return L;
}

// HEAD: the layer is the last one of the trunk; the epilogue additionally evaluates the
// detection head o_p = b_p + sum_c w_p[c] a[c] on the ROUNDED output values (same order and
// fmaf chain as head_post.cu, so both produce the same bits) and stores it as an fp32 map:
// K3 then reads 4 B/px instead of 2C B/px.
template <int C, bool HEAD>
__global__ void __launch_bounds__(kThreads, 1)
    conv_umma_kernel(const __nv_bfloat16* __restrict__ in, __nv_bfloat16* __restrict__ out, Geo geo,
                     const uint8_t* __restrict__ wpack, const float* __restrict__ bias, int nstage,
                     const float* __restrict__ head_w, const float* __restrict__ head_b,
                     float* __restrict__ logit) {
  extern __shared__ uint8_t smem_raw[];
  const SmemLayout L = smem_layout(C, geo.d, nstage);
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 1023u) & ~1023u;  // the launch reserves 1 KB of slack for this
  uint8_t* smem = smem_raw + (sbase - sraw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int d = geo.d;
  PROF_T(t_begin);
  PROF_DECL;

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
        mbar_init(empty_bar(ln, s), 5);  // MMA commit + one arrival per epilogue warp
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
  if (HEAD) {
    for (int i = threadIdx.x; i < C; i += kThreads) bias_s[C + i] = head_w[i];
    if (threadIdx.x == 0) bias_s[2 * C] = head_b[0];
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  // Programmatic dependent launch: everything above (barriers, TMEM, bias) and the weight
  // load below touch nothing the previous layer's kernel writes, so they overlap its tail.
  // Let the next layer's kernel start its own prologue as soon as SMs free up ...
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  const int nlanes = 2 * gridDim.x;

  // The two single-thread roles run with the whole warp converged and one elected lane
  // issuing: every operand below is warp-uniform, so the compiler keeps descriptors and
  // addresses in uniform registers (inside an `if (lane == 0)` region it falls back to a
  // per-instruction R2UR broadcast loop, ~19 instructions per MMA: the issue thread, not
  // the tensor pipe, was then the limiter - profiles/conv_umma_r1_full.md).
  if (warp == 0 || warp == 2) {
    // =========================== TMA producers: warp 0 -> lane 0, warp 2 -> lane 1 ========
    const int ln = warp >> 1;
    if (warp == 0 && elect_one()) {
      // the layer's weights: one bulk copy stream into shared memory, resident for the launch
      mbar_expect_tx(wbar, L.w_bytes);
      for (uint32_t off = 0; off < L.w_bytes; off += 16384u) {
        uint32_t n = L.w_bytes - off < 16384u ? L.w_bytes - off : 16384u;
        bulk_load(sbase + L.w_off + off, wpack + off, n, wbar);
      }
    }
    __syncwarp();
    // ... and wait for the previous layer's kernel to have finished (it wrote `in` and was
    // still reading `out`) before the first activation access.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // One input row segment = C/8 contiguous runs of (128 + 2d) pixels x 16 B in the
    // chunk-planar layout: one 1-D bulk copy each (a tensor-map box with a 16-byte inner
    // dimension costs one 32-byte sector request per pixel-chunk, twice the L2 traffic).
    // The parts of the segment outside the row are the convolution's zero padding (and the
    // ragged right edge): they are bulk-copied from a block of zeros, for the first `nstage`
    // loads after the segment changes - after that every stage already holds them.
    const uint32_t plane = (uint32_t)(kTileM + 2 * d) * 16u;
    const size_t plane_bytes = (size_t)geo.H * geo.W * 16u;
    const size_t row_step = (size_t)d * geo.W * 16u;
    const uint8_t* in_b = reinterpret_cast<const uint8_t*>(in);
    LaneRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    Run run;
    uint32_t st = 0, empty_par = 1;
    int last_x0 = -1, fills_left = 0;
    while (runs.next(geo, run)) {
      const int xl = run.x0 - d, xr = run.x0 + kTileM + d;
      const int lo = xl > 0 ? xl : 0, hi = xr < geo.W ? xr : geo.W;
      const uint32_t pre = (uint32_t)(lo - xl) * 16u, mid = (uint32_t)(hi - lo) * 16u,
                     post = (uint32_t)(xr - hi) * 16u;
      if (run.x0 != last_x0) {
        last_x0 = run.x0;
        fills_left = (pre | post) ? nstage : 0;
      }
      int row = run.r + (run.i0 - 1) * d;
      const uint8_t* src = in_b + ((size_t)run.b * (C / 8) * geo.H * geo.W + (long long)row * geo.W + lo) * 16;
      for (int j = 0; j < run.n + 2; ++j, row += d, src += row_step) {
        if (row < 0 || row >= geo.H) continue;
        const uint32_t dst = stage_addr(ln, st);
        const uint32_t bar = full_bar(ln, st);
        const bool fill = fills_left > 0;
        PROF_WAIT(1, mbar_wait(empty_bar(ln, st), empty_par));
        if (elect_one()) {
          mbar_expect_tx(bar, (uint32_t)(C / 8) * (fill ? plane : mid));
#pragma unroll
          for (int k = 0; k < C / 8; ++k)
            bulk_load(dst + (uint32_t)k * plane + pre, src + (size_t)k * plane_bytes, mid, bar);
          if (fill) {
#pragma unroll
            for (int k = 0; k < C / 8; ++k) {
              if (pre) bulk_load(dst + (uint32_t)k * plane, g_zeros, pre, bar);
              if (post) bulk_load(dst + (uint32_t)k * plane + pre + mid, g_zeros, post, bar);
            }
          }
        }
        __syncwarp();
        fills_left -= fill ? 1 : 0;
        if (++st == (uint32_t)nstage) {
          st = 0;
          empty_par ^= 1u;
        }
      }
    }
  } else if (warp == 1 || warp == 3) {
    // =========================== MMA issuers: warp 1 -> lane 0, warp 3 -> lane 1 ==========
    // One issuing warp per lane: the tensor pipe's instruction queue is short, so while one
    // warp is busy with barriers and bookkeeping between two steps the other one's MMAs keep
    // the pipe fed (the lanes are independent: own TMEM columns, own stages).
    const int ln = warp >> 1;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    PROF_ADD(0, clock64() - t_begin);
    PROF_WAIT(2, mbar_wait(wbar, 0));
    constexpr uint32_t idesc = umma_idesc(kTileM, 3 * C);
    const uint32_t plane16 = (uint32_t)(kTileM + 2 * d);  // (bytes between channel chunks of A) / 16
    constexpr uint32_t wplane16 = 5u * C;                 // same for B
    // descriptor = {hi: SBO = 128 B, version 1; lo: LBO << 16 | start address >> 4}
    constexpr uint32_t desc_hi = (128u >> 4) | (1u << 14);
    const uint32_t a_lo_base = (plane16 << 16) | (((sbase + L.stage_off) >> 4) & 0x3FFFu);
    const uint32_t b_lo_base = (wplane16 << 16) | (((sbase + L.w_off) >> 4) & 0x3FFFu);
    const uint32_t stage16 = L.stage_bytes >> 4;
    const uint32_t dcol = __shfl_sync(0xffffffffu, tmem_base, 0) + (uint32_t)ln * kLaneCols;
    LaneRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    Run run;
    uint32_t st = 0, full_par = 0, free_par = 0, m = 0;
    while (runs.next(geo, run)) {
      int row = run.r + (run.i0 - 1) * d;
      for (int j = 0; j < run.n + 2; ++j, row += d) {
        const bool in_valid = row >= 0 && row < geo.H;
        if (in_valid) PROF_WAIT(3, mbar_wait(full_bar(ln, st), full_par));
        PROF_WAIT(4, mbar_wait(acc_free_bar(ln), free_par));  // slot (u+2)%3 re-initialised by the epilogue
        free_par ^= 1u;
        tc_fence_after();
        // rows stored as ky = (1,0,2,1,0): window start for u%3 = 0,1,2 is block 0,2,1
        const uint32_t win = m == 0 ? 0u : (m == 1 ? 2u : 1u);
        const uint32_t a_lo = a_lo_base + ((uint32_t)ln * nstage + st) * stage16;
        const uint32_t b_lo = b_lo_base + win * C;
        PROF_T(t_issue);
        if (elect_one()) {
          if (in_valid) {
#pragma unroll
            for (int kx = 0; kx < 3; ++kx) {
#pragma unroll
              for (int ks = 0; ks < C / 16; ++ks) {
                const uint32_t al = a_lo + (uint32_t)(2 * ks) * plane16 + (uint32_t)(kx * d);
                const uint32_t bl = b_lo + (uint32_t)(kx * (C / 8) + 2 * ks) * wplane16;
                tc_mma(dcol, ((uint64_t)desc_hi << 32) | al, ((uint64_t)desc_hi << 32) | bl, idesc, 1u);
              }
            }
            tc_commit(empty_bar(ln, st));
          }
          tc_commit(acc_full_bar(ln));
        }
        __syncwarp();
        PROF_ADD(8, clock64() - t_issue);
        if (in_valid && ++st == (uint32_t)nstage) {
          st = 0;
          full_par ^= 1u;
        }
        m = m == 2 ? 0u : m + 1u;
      }
    }
    PROF_ADD(5, clock64() - t_begin);
  } else if (warp >= 4) {
    // =========================== epilogue ===========================
    const int ln = (warp - 4) >> 2;
    const int qd = warp & 3;  // TMEM lane quadrant this warp may access
    asm volatile("griddepcontrol.wait;" ::: "memory");
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

    const size_t plane_px = (size_t)geo.H * geo.W;
    const uint32_t plane = (uint32_t)(kTileM + 2 * d) * 16u;
    // The residual operand of an output row is its own centre input row, which the previous
    // step of this lane staged in shared memory: it is read from there (no second trip to
    // L2).  Two policies for handing that stage back to the producer (the empty barrier
    // counts the MMA commit plus one arrival per epilogue warp):
    //   kEarly (C = 64, where only 2-3 stages per lane fit): the epilogue of step u - whose
    //     acc_full says MMA(u) is done with stage(u) - copies the 128 centre pixels into
    //     registers for step u+1 and releases the stage at once; holding it until step u+1
    //     would cost one stage of prefetch depth (measured: 0.8 -> 1.2 PFLOP/s at C = 64).
    //     The copy is a generic-proxy read that the TMA refill (async proxy) must not
    //     overtake: fence.proxy.async before the arrive.  Without it the arrive is issued
    //     behind loads still in flight and the refill raced with them (measured).
    //   otherwise (6 stages): step u+1 reads the residual straight from stage(u) and releases
    //     it after use; no extra registers, no fence (3 % faster at C = 48).
    constexpr bool kEarly = C >= 64;
    LaneRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    Run run;
    uint32_t slot = 2, acc_par = 0, st = 0, prev_st = 0;
    bool prev_valid = false;
    uint4 res[C / 8];
#pragma unroll
    for (int k = 0; k < C / 8; ++k) res[k] = make_uint4(0u, 0u, 0u, 0u);
    while (runs.next(geo, run)) {
      const int x = run.x0 + px;
      int row = run.r + (run.i0 - 1) * d;  // input row of the step; the output row is row - d
      uint4* orow = reinterpret_cast<uint4*>(out) +
                    ((size_t)run.b * (C / 8) * geo.H * geo.W + (long long)(row - d) * geo.W + x);
      for (int j = 0; j < run.n + 2; ++j, row += d, orow += (size_t)d * geo.W) {
        const bool in_valid = row >= 0 && row < geo.H;
        const bool out_valid = j >= 2 && row - d < geo.H;
        const bool store = out_valid && x < geo.W;
        PROF_WAIT(6, mbar_wait(acc_full_bar(ln), acc_par));
        acc_par ^= 1u;
        tc_fence_after();
        PROF_T(t_tm0);
        uint32_t acc[C];
        if (out_valid) {
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
        PROF_ADD(9, clock64() - t_tm0);
        PROF_T(t_post0);
        // (the stage was filled by the async proxy; its full barrier was observed by this
        // lane's MMA warp, whose tcgen05.commit on acc_full this thread has observed in turn)
        const uint4* rprev = reinterpret_cast<const uint4*>(smem + (stage_addr(ln, prev_st) - sbase) +
                                                            (uint32_t)(d + px) * 16u);
        if (store) {
          float lg = HEAD ? bias_s[2 * C] : 0.0f;
#pragma unroll
          for (int k = 0; k < C / 8; ++k) {
            const uint4 rk = kEarly ? res[k] : rprev[(size_t)k * (plane / 16u)];
            const uint32_t rw[4] = {rk.x, rk.y, rk.z, rk.w};
            uint32_t ow[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              float r0 = __uint_as_float(rw[i] << 16), r1 = __uint_as_float(rw[i] & 0xffff0000u);
              float v0 = r0 + fmaxf(__uint_as_float(acc[k * 8 + 2 * i]), 0.0f);
              float v1 = r1 + fmaxf(__uint_as_float(acc[k * 8 + 2 * i + 1]), 0.0f);
              __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
              ow[i] = *reinterpret_cast<uint32_t*>(&h);
              if (HEAD) {
                lg = fmaf(__uint_as_float(ow[i] << 16), bias_s[C + k * 8 + 2 * i], lg);
                lg = fmaf(__uint_as_float(ow[i] & 0xffff0000u), bias_s[C + k * 8 + 2 * i + 1], lg);
              }
            }
            orow[(size_t)k * plane_px] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
          }
          if (HEAD) logit[((size_t)run.b * geo.H + (row - d)) * geo.W + x] = lg;
        }
        if (kEarly) {
          if (in_valid) {
            const uint4* rp = reinterpret_cast<const uint4*>(smem + (stage_addr(ln, st) - sbase) +
                                                             (uint32_t)(d + px) * 16u);
#pragma unroll
            for (int k = 0; k < C / 8; ++k) res[k] = rp[(size_t)k * (plane / 16u)];
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(ln, st));
          }
        } else if (prev_valid) {
          __syncwarp();  // the residual was consumed above (real data dependence), so the
          if (lane == 0) mbar_arrive(empty_bar(ln, prev_st));  // loads are done before this arrive
        }
        prev_valid = in_valid;
        if (in_valid) {
          prev_st = st;
          if (++st == (uint32_t)nstage) st = 0;
        }
        PROF_ADD(10, clock64() - t_post0);
        slot = slot == 2 ? 0u : slot + 1u;
      }
    }
  }

  // ---- teardown
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) PROF_ADD(7, clock64() - t_begin);
  PROF_FLUSH(threadIdx.x == 0 || threadIdx.x == 32 || threadIdx.x == 128)
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
  }
}

// ------------------------------------------------------------------------------ host side
uint16_t bf16_bits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

template <int C, bool HEAD>
cudaError_t launch_ch(const void* in, void* out, Geo geo, const void* wpack, const float* bias, int nstage,
                      int grid, size_t smem, const float* head_w, const float* head_b, float* logit,
                      cudaStream_t st) {
  static bool attr_done[kMaxDevices] = {};  // the attribute is per device
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (!attr_done[dev]) {
    cudaError_t e = cudaFuncSetAttribute(conv_umma_kernel<C, HEAD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         227 * 1024);
    if (e != cudaSuccess) return e;
    attr_done[dev] = true;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, conv_umma_kernel<C, HEAD>, (const __nv_bfloat16*)in, (__nv_bfloat16*)out,
                            geo, (const uint8_t*)wpack, bias, nstage, head_w, head_b, logit);
}
template <int C>
cudaError_t launch_c(const void* in, void* out, Geo geo, const void* wpack, const float* bias, int nstage,
                     int grid, size_t smem, const float* head_w, const float* head_b, float* logit,
                     cudaStream_t st) {
  return logit ? launch_ch<C, true>(in, out, geo, wpack, bias, nstage, grid, smem, head_w, head_b, logit, st)
               : launch_ch<C, false>(in, out, geo, wpack, bias, nstage, grid, smem, head_w, head_b, logit, st);
}

}  // namespace

struct UmmaPlan {
  const void* buf[2];
  ActShape s;
  int n_sm;
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
  if (s.C % 16 || s.C < 16 || s.C > 64) {
    snprintf(err, errlen, "channels must be 16/32/48/64");
    return nullptr;
  }
  UmmaPlan* p = new UmmaPlan;
  p->buf[0] = buf0;
  p->buf[1] = buf1;
  p->s = s;
  p->n_sm = n_sm;
  return p;
}

void umma_plan_destroy(UmmaPlan* p) { delete p; }

cudaError_t launch_conv_umma(UmmaPlan* p, int src, int dil, const void* wpack, const float* bias,
                             const float* head_w, const float* head_b, float* logit, cudaStream_t st,
                             char* err, size_t errlen) {
  if (!p || dil < 1 || dil > 8 || src < 0 || src > 1) return cudaErrorInvalidValue;
  const ActShape& s = p->s;
  if (s.B <= 0) return cudaSuccess;
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
  // (>= 2 for any overlap of load and MMA)
  while (nstage > 2 && L.total + 1024 > 227u * 1024u) L = smem_layout(s.C, dil, --nstage);
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
    case 16: return launch_c<16>(in, out, geo, wpack, bias, nstage, grid, smem, head_w, head_b, logit, st);
    case 32: return launch_c<32>(in, out, geo, wpack, bias, nstage, grid, smem, head_w, head_b, logit, st);
    case 48: return launch_c<48>(in, out, geo, wpack, bias, nstage, grid, smem, head_w, head_b, logit, st);
    case 64: return launch_c<64>(in, out, geo, wpack, bias, nstage, grid, smem, head_w, head_b, logit, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace smlm
