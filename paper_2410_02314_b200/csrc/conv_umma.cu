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
//     weight load of layer l+1 overlap the tail of layer l;
//   * STEM variant (first layer): K1 is folded in.  No activation map is read: the lane's
//     epilogue warps (one pixel per thread) and its producer warp (the 2d halo pixels)
//     compute a_0 = act(conv3x3(xhat) + b_0) for the row segment of a step two steps ahead
//     of the MMAs, straight from the uint16 frame, and write it as bf16 into the stage in
//     operand layout; the residual of the layer is that same stage;
//   * HEAD variant (last layer): K3's heads are folded in.  The activation map is NOT
//     stored; the epilogue evaluates the detection logit of every pixel (fp32 map, 4 B/px)
//     and, for pixels above the threshold only, the other heads (one 32-byte record per
//     candidate pixel): K3 reads logits and candidate records, no activations.
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
constexpr int kLaneBars = 2 * kMaxStages + 2 + 2 * 3;  // mbarriers per lane (SmemLayout)
constexpr int kMaxDilation = 8;

// zero source for the padded parts of a row segment: at most (127 + 8) pixels x 16 B
__device__ __align__(16) uint4 g_zeros[160];

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


// The steps of a lane whose input row lies inside the image, in walk order: exactly the
// steps that occupy a shared-memory stage.
struct Step {
  int b, x0, row;
};
struct ValidSteps {
  LaneRuns runs;
  Run run;
  int j, row;
  bool have_run;
  __device__ void init(const Geo& geo, int lane_id, int nlanes) {
    runs.init(geo, lane_id, nlanes);
    have_run = false;
  }
  __device__ bool next(const Geo& geo, Step& s) {
    for (;;) {
      if (!have_run) {
        if (!runs.next(geo, run)) return false;
        have_run = true;
        j = 0;
        row = run.r + (run.i0 - 1) * geo.d;
      }
      while (j < run.n + 2) {
        const int r = row;
        ++j;
        row += geo.d;
        if (r >= 0 && r < geo.H) {
          s.b = run.b;
          s.x0 = run.x0;
          s.row = r;
          return true;
        }
      }
      have_run = false;
    }
  }
};

// ------------------------------------------------------------------------------ STEM (K1 folded in)
// smlm.h: xhat = ((adu - offset) / gain) / norm_scale, 0 outside the FRAME;
// a_0 = act(b_0 + sum_{ky,kx} W_0[c][ky][kx] xhat[y+ky-1][x+kx-1]), taps in (ky, kx) order with
// one fmaf each - the same chain as stem.cu, so both kernels produce the same bits.
__device__ __forceinline__ unsigned long long pack2f(float lo, float hi) {
  return ((unsigned long long)__float_as_uint(hi) << 32) | __float_as_uint(lo);
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b,
                                                    unsigned long long c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
// One pixel of a_0, all C channels, rounded to bf16 and written to the stage in operand
// layout (chunk k of the pixel at dst + k * plane).  Two channels per fma.rn.f32x2 (two
// independent IEEE fp32 FMAs).  valid == false (pixel outside the window): zeros.
template <int C>
__device__ __forceinline__ void stem_pixel(const float (&xv)[9], const float* ws, const float* bs,
                                           int relu, bool valid, uint8_t* dst, uint32_t plane) {
  unsigned long long xx[9];
#pragma unroll
  for (int t = 0; t < 9; ++t) xx[t] = pack2f(xv[t], xv[t]);
#pragma unroll 2
  for (int k = 0; k < C / 8; ++k) {
    const ulonglong2 b01 = *reinterpret_cast<const ulonglong2*>(bs + k * 8);
    const ulonglong2 b23 = *reinterpret_cast<const ulonglong2*>(bs + k * 8 + 4);
    unsigned long long acc[4] = {b01.x, b01.y, b23.x, b23.y};
#pragma unroll
    for (int t = 0; t < 9; ++t) {
      const ulonglong2 w01 = *reinterpret_cast<const ulonglong2*>(ws + t * C + k * 8);
      const ulonglong2 w23 = *reinterpret_cast<const ulonglong2*>(ws + t * C + k * 8 + 4);
      acc[0] = ffma2(xx[t], w01.x, acc[0]);
      acc[1] = ffma2(xx[t], w01.y, acc[1]);
      acc[2] = ffma2(xx[t], w23.x, acc[2]);
      acc[3] = ffma2(xx[t], w23.y, acc[3]);
    }
    uint32_t ow[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float v0 = __uint_as_float((uint32_t)acc[i]), v1 = __uint_as_float((uint32_t)(acc[i] >> 32));
      if (relu) {
        v0 = fmaxf(v0, 0.0f);
        v1 = fmaxf(v1, 0.0f);
      }
      __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
      ow[i] = valid ? *reinterpret_cast<uint32_t*>(&h) : 0u;
    }
    *reinterpret_cast<uint4*>(dst + (size_t)k * plane) = make_uint4(ow[0], ow[1], ow[2], ow[3]);
  }
}

constexpr int kPatchSlots = 3;  // STEM: ring of normalised input patches per lane

struct SmemLayout {
  uint32_t w_off, w_bytes;
  uint32_t stage_off, stage_bytes;  // per (lane, stage)
  uint32_t bias_off;  // float: layer bias [C], detection-head row [C], other head rows [C][8], head bias [8]
  uint32_t stem_off;  // float: stem weights [9][C], stem bias [C]
  uint32_t patch_off, patch_bytes, patch_row;  // STEM: per (lane, slot): float xhat[3][patch_row], int x0
  uint32_t bar_off;
  uint32_t tmem_off;
  uint32_t total;
  int nstage;
};

__host__ __device__ inline SmemLayout smem_layout(int C, int d, int nstage, bool stem) {
  SmemLayout L;
  L.w_off = 0;
  L.w_bytes = 30u * C * C;  // 3 kx * C/8 chunks * 5C rows * 16 B
  L.stage_bytes = (((uint32_t)(C / 8) * (kTileM + 2 * d) * 16u) + 127u) & ~127u;
  L.stage_off = (L.w_off + L.w_bytes + 127u) & ~127u;
  L.nstage = nstage;
  L.bias_off = L.stage_off + 2u * nstage * L.stage_bytes;
  L.stem_off = L.bias_off + (uint32_t)(10 * C + 8) * 4u;
  L.patch_off = L.stem_off + (uint32_t)(10 * C) * 4u;
  L.patch_row = (uint32_t)(kTileM + 2 * d + 2 + 3) & ~3u;  // the segment plus the stem's own 1-px halo
  L.patch_bytes = stem ? (3u * L.patch_row + 4u) * 4u : 0u;
  L.bar_off = L.patch_off + 2u * kPatchSlots * L.patch_bytes;
  // barriers: wbar, per lane: full[kMaxStages], empty[kMaxStages], acc_full, acc_free,
  // patch_full[kPatchSlots], patch_empty[kPatchSlots]
  L.tmem_off = L.bar_off + 8u * (1 + 2 * kLaneBars);
  L.total = L.tmem_off + 16u;
  return L;
}

// HEAD: the layer is the last one of the trunk.  The epilogue evaluates the heads on the ROUNDED
// output values (same order and fmaf chain as head_post.cu, so both produce the same bits):
// the detection logit o_p for every pixel, the other heads for pixels with o_p > lthr; the
// activation map itself is not stored.
// STEM: the layer is the first one; its input a_0 is computed in the kernel (see above).
template <int C, bool HEAD, bool STEM>
__global__ void __launch_bounds__(kThreads, 1)
    conv_umma_kernel(const __nv_bfloat16* __restrict__ in, __nv_bfloat16* __restrict__ out, Geo geo,
                     const uint8_t* __restrict__ wpack, const float* __restrict__ bias, int nstage,
                     const HeadArgs ha, const StemArgs sa) {
  extern __shared__ uint8_t smem_raw[];
  const SmemLayout L = smem_layout(C, geo.d, nstage, STEM);
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 1023u) & ~1023u;  // the launch reserves 1 KB of slack for this
  uint8_t* smem = smem_raw + (sbase - sraw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int d = geo.d;

  const uint32_t wbar = sbase + L.bar_off;
  auto lane_bar = [&](int ln, int i) { return sbase + L.bar_off + 8u * (1 + ln * kLaneBars + i); };
  auto full_bar = [&](int ln, int s) { return lane_bar(ln, s); };
  auto empty_bar = [&](int ln, int s) { return lane_bar(ln, kMaxStages + s); };
  auto acc_full_bar = [&](int ln) { return lane_bar(ln, 2 * kMaxStages); };
  auto acc_free_bar = [&](int ln) { return lane_bar(ln, 2 * kMaxStages + 1); };
  auto patch_full_bar = [&](int ln, int s) { return lane_bar(ln, 2 * kMaxStages + 2 + s); };
  auto patch_empty_bar = [&](int ln, int s) { return lane_bar(ln, 2 * kMaxStages + 2 + kPatchSlots + s); };
  auto patch_ptr = [&](int ln, int s) {
    return reinterpret_cast<float*>(smem + L.patch_off + (uint32_t)(ln * kPatchSlots + s) * L.patch_bytes);
  };
  auto stage_addr = [&](int ln, int s) { return sbase + L.stage_off + (uint32_t)(ln * nstage + s) * L.stage_bytes; };
  float* bias_s = reinterpret_cast<float*>(smem + L.bias_off);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + L.tmem_off);

  // ---- one-time setup
  if (threadIdx.x == 0) {
    mbar_init(wbar, 1);
    for (int ln = 0; ln < 2; ++ln) {
      for (int s = 0; s < kMaxStages; ++s) {
        // full: the TMA transaction count, or (STEM) the four epilogue warps
        mbar_init(full_bar(ln, s), STEM ? 4 : 1);
        mbar_init(empty_bar(ln, s), 5);  // MMA commit + one arrival per epilogue warp
      }
      mbar_init(acc_full_bar(ln), 1);
      mbar_init(acc_free_bar(ln), 4);  // one arrival per epilogue warp
      for (int s = 0; s < kPatchSlots; ++s) {
        mbar_init(patch_full_bar(ln, s), 1);   // the producer warp
        mbar_init(patch_empty_bar(ln, s), 4);  // one arrival per epilogue warp
      }
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
  float* head_s = bias_s + C;        // detection head row [C]
  float* headq_s = bias_s + 2 * C;   // [C][8]: rows 1 .. n_h-1 of channel c, zero padded
  float* headb_s = bias_s + 10 * C;  // [8]: head biases 0 .. n_h-1, zero padded
  if (HEAD) {
    for (int i = threadIdx.x; i < C; i += kThreads) head_s[i] = ha.w[i];
    for (int i = threadIdx.x; i < 8 * C; i += kThreads) {
      const int c = i >> 3, h = 1 + (i & 7);
      headq_s[i] = h < ha.n_h ? ha.w[h * C + c] : 0.0f;
    }
    if (threadIdx.x < 8) headb_s[threadIdx.x] = (int)threadIdx.x < ha.n_h ? ha.b[threadIdx.x] : 0.0f;
  }
  float* stem_w_s = reinterpret_cast<float*>(smem + L.stem_off);  // [9][C]
  float* stem_b_s = stem_w_s + 9 * C;
  if (STEM) {
    for (int i = threadIdx.x; i < 9 * C; i += kThreads) stem_w_s[i] = sa.w[i];
    for (int i = threadIdx.x; i < C; i += kThreads) stem_b_s[i] = sa.b[i];
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
    if (STEM) {
      // STEM producer.  Per valid step: (1) the normalised input patch xhat[3][130 + 2d] (rows
      // row-1, row, row+1; columns x0-d-1 .. x0+128+d) goes to a ring in shared memory, from
      // which the epilogue threads take the inputs of their pixel (and of the 2d halo pixels
      // of the segment, which they share out by channel).  When a step continues the previous
      // one with d = 1, two of its three rows are the previous patch's rows 1 and 2 (copied
      // inside shared memory) and only the new row is loaded.  The global loads of step s+1
      // are in flight while step s is processed (two register sets, loop unrolled by two),
      // and the warp runs as far ahead as the rings allow: it is off the critical path.
      const int pcols = kTileM + 2 * d + 2;      // patch columns in use
      constexpr int NJ = (kTileM + 2 * kMaxDilation + 2 + 31) / 32;  // column passes per row
      ValidSteps steps;
      steps.init(geo, 2 * blockIdx.x + ln, nlanes);
      uint32_t ps = 0, pempty_par = 1;
      struct Raw {
        uint16_t adu[3][NJ];
        float om[3][NJ], gm[3][NJ];
      };
      // (uniform branches on `reuse`: predicated-off instructions would still cost issue slots)
      auto issue = [&](const Step& sp, bool reuse, Raw& rw) {
        const View v = view_of(sa.vs, sp.b, geo.H, geo.W);
        const uint16_t* frame = sa.frames + (size_t)(v.frame - sa.frame_base) * sa.vs.Hf * sa.vs.Wf;
        const int fx0 = v.wx0 + sp.x0 - d - 1 + lane;
        auto load_row = [&](int py, uint16_t (&adu)[NJ], float (&om)[NJ], float (&gm)[NJ]) {
          const int fy = v.wy0 + sp.row - 1 + py;
          const bool row_ok = fy >= 0 && fy < sa.vs.Hf;
          const size_t rowq = (size_t)(row_ok ? fy : 0) * sa.vs.Wf;
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            const int fx = fx0 + 32 * j;
            const bool ok = row_ok && lane + 32 * j < pcols && fx >= 0 && fx < sa.vs.Wf;
            const size_t q = rowq + (ok ? fx : 0);
            adu[j] = ok ? __ldg(frame + q) : (uint16_t)0;  // (0 - 0) / 1 normalises to exactly 0
            om[j] = ok ? (sa.np.offset_map ? __ldg(sa.np.offset_map + q) : sa.np.offset) : 0.0f;
            gm[j] = ok ? (sa.np.offset_map ? __ldg(sa.np.gain_map + q) : sa.np.gain) : 1.0f;
          }
        };
        if (!reuse) {
          load_row(0, rw.adu[0], rw.om[0], rw.gm[0]);
          load_row(1, rw.adu[1], rw.om[1], rw.gm[1]);
        }
        load_row(2, rw.adu[2], rw.om[2], rw.gm[2]);
      };
      auto process = [&](const Step& sp, bool reuse, const Raw& rw) {
        float* patch = patch_ptr(ln, ps);
        const float* prev = patch_ptr(ln, ps == 0 ? kPatchSlots - 1 : ps - 1);
        mbar_wait(patch_empty_bar(ln, ps), pempty_par);
        auto norm_row = [&](int py, const uint16_t (&adu)[NJ], const float (&om)[NJ], const float (&gm)[NJ]) {
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            const int pxx = lane + 32 * j;
            if (pxx < pcols)
              patch[py * L.patch_row + pxx] = (((float)adu[j] - om[j]) / gm[j]) / sa.np.norm_scale;
          }
        };
        if (reuse) {
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            const int pxx = lane + 32 * j;
            if (pxx < pcols) {
              patch[pxx] = prev[L.patch_row + pxx];
              patch[L.patch_row + pxx] = prev[2 * L.patch_row + pxx];
            }
          }
        } else {
          norm_row(0, rw.adu[0], rw.om[0], rw.gm[0]);
          norm_row(1, rw.adu[1], rw.om[1], rw.gm[1]);
        }
        norm_row(2, rw.adu[2], rw.om[2], rw.gm[2]);
        if (lane == 0) reinterpret_cast<int*>(patch)[3 * L.patch_row] = sp.x0;
        __syncwarp();
        if (lane == 0) mbar_arrive(patch_full_bar(ln, ps));
        if (++ps == (uint32_t)kPatchSlots) {
          ps = 0;
          pempty_par ^= 1u;
        }
      };
      // a step continues the previous one (same view and segment, next row) iff d == 1
      auto continues = [&](const Step& a, const Step& b) {
        return d == 1 && b.b == a.b && b.x0 == a.x0 && b.row == a.row + 1;
      };
      Raw rA, rB;
      Step sA{0, 0, 0}, sB{0, 0, 0};
      bool reA = false, reB = false;
      bool haveA = steps.next(geo, sA), haveB = false;
      if (haveA) issue(sA, false, rA);
      while (haveA) {
        haveB = steps.next(geo, sB);
        reB = haveB && continues(sA, sB);
        if (haveB) issue(sB, reB, rB);
        process(sA, reA, rA);
        if (!haveB) break;
        haveA = steps.next(geo, sA);
        reA = haveA && continues(sB, sA);
        if (haveA) issue(sA, reA, rA);
        process(sB, reB, rB);
      }
    } else {
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
          mbar_wait(empty_bar(ln, st), empty_par);
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
    }
  } else if (warp == 1 || warp == 3) {
    // =========================== MMA issuers: warp 1 -> lane 0, warp 3 -> lane 1 ==========
    // One issuing warp per lane: the tensor pipe's instruction queue is short, so while one
    // warp is busy with barriers and bookkeeping between two steps the other one's MMAs keep
    // the pipe fed (the lanes are independent: own TMEM columns, own stages).
    const int ln = warp >> 1;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    mbar_wait(wbar, 0);
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
        if (in_valid) mbar_wait(full_bar(ln, st), full_par);
        mbar_wait(acc_free_bar(ln), free_par);  // slot (u+2)%3 re-initialised by the epilogue
        free_par ^= 1u;
        tc_fence_after();
        // rows stored as ky = (1,0,2,1,0): window start for u%3 = 0,1,2 is block 0,2,1
        const uint32_t win = m == 0 ? 0u : (m == 1 ? 2u : 1u);
        const uint32_t a_lo = a_lo_base + ((uint32_t)ln * nstage + st) * stage16;
        const uint32_t b_lo = b_lo_base + win * C;
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
        if (in_valid && ++st == (uint32_t)nstage) {
          st = 0;
          full_par ^= 1u;
        }
        m = m == 2 ? 0u : m + 1u;
      }
    }
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

    // STEM: this thread computes pixel x0 + px of a_0 for the segment of the valid step that is
    // two steps ahead of the one being retired (the MMAs of the step in between are running
    // meanwhile).  Its nine inputs come from the producer warp's patch ring.
    uint32_t sst = 0, sempty_par = 1, sps = 0, spfull_par = 0;
    long long stems_left = 0;
    auto stem_advance = [&]() {
      if (stems_left <= 0) return;
      --stems_left;
      const float* patch = patch_ptr(ln, sps);
      mbar_wait(patch_full_bar(ln, sps), spfull_par);
      float xv[9];
#pragma unroll
      for (int t = 0; t < 9; ++t) xv[t] = patch[(t / 3) * L.patch_row + d + px + t % 3];
      const int x0 = reinterpret_cast<const int*>(patch)[3 * L.patch_row];
      mbar_wait(empty_bar(ln, sst), sempty_par);
      uint8_t* stage = smem + (stage_addr(ln, sst) - sbase);
      const uint32_t splane = (uint32_t)(kTileM + 2 * d) * 16u;
      // the 2d halo pixels of the segment (positions [0, d) and [d + 128, 128 + 2d)): one
      // (pixel, channel) output per thread and pass, the same fmaf chain
      for (int o = px; o < 2 * d * C; o += kTileM) {
        const int h = o / C, c = o - h * C;
        const int pos = h < d ? h : kTileM + h;  // position in the (128 + 2d)-pixel segment
        const int x = x0 - d + pos;              // window coordinate
        float a = stem_b_s[c];
#pragma unroll
        for (int t = 0; t < 9; ++t)
          a = fmaf(patch[(t / 3) * L.patch_row + pos + t % 3], stem_w_s[t * C + c], a);
        if (sa.relu) a = fmaxf(a, 0.0f);
        const __nv_bfloat16 hb = __float2bfloat16_rn(a);
        const uint16_t bits = (x >= 0 && x < geo.W) ? *reinterpret_cast<const uint16_t*>(&hb) : (uint16_t)0;
        *reinterpret_cast<uint16_t*>(stage + (size_t)(c >> 3) * splane + (size_t)pos * 16u + (c & 7) * 2) = bits;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(patch_empty_bar(ln, sps));
      stem_pixel<C>(xv, stem_w_s, stem_b_s, sa.relu, x0 + px < geo.W, stage + (size_t)(d + px) * 16u, splane);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(full_bar(ln, sst));
      if (++sst == (uint32_t)nstage) {
        sst = 0;
        sempty_par ^= 1u;
      }
      if (++sps == (uint32_t)kPatchSlots) {
        sps = 0;
        spfull_par ^= 1u;
      }
    };
    if (STEM) {
      ValidSteps cnt;  // number of valid steps of this lane
      cnt.init(geo, 2 * blockIdx.x + ln, nlanes);
      Step tmp;
      while (cnt.next(geo, tmp)) ++stems_left;
      stem_advance();
      stem_advance();
    }

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
        mbar_wait(acc_full_bar(ln), acc_par);
        acc_par ^= 1u;
        tc_fence_after();
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
        // (the stage was filled by the async proxy; its full barrier was observed by this
        // lane's MMA warp, whose tcgen05.commit on acc_full this thread has observed in turn)
        const uint4* rprev = reinterpret_cast<const uint4*>(smem + (stage_addr(ln, prev_st) - sbase) +
                                                            (uint32_t)(d + px) * 16u);
        if (store) {
          float lg = HEAD ? headb_s[0] : 0.0f;
          uint32_t orw[HEAD ? C / 2 : 1];  // HEAD: the rounded output row stays in registers
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
                lg = fmaf(__uint_as_float(ow[i] << 16), head_s[k * 8 + 2 * i], lg);
                lg = fmaf(__uint_as_float(ow[i] & 0xffff0000u), head_s[k * 8 + 2 * i + 1], lg);
                orw[k * 4 + i] = ow[i];
              }
            }
            if (!HEAD) orow[(size_t)k * plane_px] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
          }
          if (HEAD) {
            const size_t q = ((size_t)run.b * geo.H + (row - d)) * geo.W + x;
            ha.logit[q] = lg;
            if (lg > ha.lthr) {
              // candidate: the other heads, each the same fmaf chain over the channels as
              // head_post.cu, two heads per fma.rn.f32x2 (independent IEEE fp32 FMAs)
              unsigned long long a12 = pack2f(headb_s[1], headb_s[2]), a34 = pack2f(headb_s[3], headb_s[4]),
                                 a5 = pack2f(headb_s[5], 0.0f);
              const bool six = ha.n_h == 6;
#pragma unroll
              for (int c2 = 0; c2 < C / 2; ++c2) {
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                  const float av = __uint_as_float(half ? (orw[c2] & 0xffff0000u) : (orw[c2] << 16));
                  const unsigned long long aa = pack2f(av, av);
                  const float* wq = headq_s + (2 * c2 + half) * 8;
                  const ulonglong2 w14 = *reinterpret_cast<const ulonglong2*>(wq);
                  a12 = ffma2(aa, w14.x, a12);
                  a34 = ffma2(aa, w14.y, a34);
                  if (six) a5 = ffma2(aa, *reinterpret_cast<const unsigned long long*>(wq + 4), a5);
                }
              }
              float4* cq = reinterpret_cast<float4*>(ha.cand) + q * 2;
              cq[0] = make_float4(__uint_as_float((uint32_t)a12), __uint_as_float((uint32_t)(a12 >> 32)),
                                  __uint_as_float((uint32_t)a34), __uint_as_float((uint32_t)(a34 >> 32)));
              cq[1] = make_float4(__uint_as_float((uint32_t)a5), 0.0f, 0.0f, 0.0f);
            }
          }
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
          if (STEM) stem_advance();
        }
        slot = slot == 2 ? 0u : slot + 1u;
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
uint16_t bf16_bits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

template <int C, bool HEAD, bool STEM>
cudaError_t launch_chs(const void* in, void* out, Geo geo, const void* wpack, const float* bias, int nstage,
                       int grid, size_t smem, const HeadArgs& ha, const StemArgs& sa, cudaStream_t st) {
  static bool attr_done[kMaxDevices] = {};  // the attribute is per device
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (!attr_done[dev]) {
    cudaError_t e = cudaFuncSetAttribute(conv_umma_kernel<C, HEAD, STEM>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
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
  return cudaLaunchKernelEx(&cfg, conv_umma_kernel<C, HEAD, STEM>, (const __nv_bfloat16*)in,
                            (__nv_bfloat16*)out, geo, (const uint8_t*)wpack, bias, nstage, ha, sa);
}
template <int C>
cudaError_t launch_c(const void* in, void* out, Geo geo, const void* wpack, const float* bias, int nstage,
                     int grid, size_t smem, const HeadArgs* ha, const StemArgs* sa, cudaStream_t st) {
  const HeadArgs h0{};
  const StemArgs s0{};
  if (ha && sa) return launch_chs<C, true, true>(in, out, geo, wpack, bias, nstage, grid, smem, *ha, *sa, st);
  if (ha) return launch_chs<C, true, false>(in, out, geo, wpack, bias, nstage, grid, smem, *ha, s0, st);
  if (sa) return launch_chs<C, false, true>(in, out, geo, wpack, bias, nstage, grid, smem, h0, *sa, st);
  return launch_chs<C, false, false>(in, out, geo, wpack, bias, nstage, grid, smem, h0, s0, st);
}

// stages: as many as fit next to the resident weights (<= kMaxStages; >= 2 for any overlap of
// load and MMA; the STEM variant computes two steps ahead and needs >= 3)
int pick_stages(int C, int dil, bool stem) {
  int nstage = kMaxStages;
  const int min_stage = stem ? 3 : 2;
  while (nstage >= min_stage && smem_layout(C, dil, nstage, stem).total + 1024 > 227u * 1024u) --nstage;
  return nstage >= min_stage ? nstage : 0;
}

}  // namespace

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

bool conv_umma_supports(int C, int dil, bool stem) {
  return C >= 16 && C <= 64 && C % 16 == 0 && dil >= 1 && dil <= kMaxDilation && pick_stages(C, dil, stem) > 0;
}

cudaError_t launch_conv_umma(const void* in, void* out, ActShape s, int dil, const void* wpack,
                             const float* bias, const HeadArgs* head, const StemArgs* stem, int n_sm,
                             cudaStream_t st, char* err, size_t errlen) {
  if (dil < 1 || dil > kMaxDilation || s.C % 16 || s.C < 16 || s.C > 64) {
    snprintf(err, errlen, "unsupported channels / dilation");
    return cudaErrorInvalidValue;
  }
  if (s.B <= 0) return cudaSuccess;
  Geo geo;
  geo.B = s.B;
  geo.H = s.H;
  geo.W = s.W;
  geo.d = dil;
  geo.nseg = (s.W + kTileM - 1) / kTileM;
  geo.Lmax = (s.H + dil - 1) / dil;
  geo.total = (long long)s.B * geo.nseg * dil * geo.Lmax;
  const int nstage = pick_stages(s.C, dil, stem != nullptr);
  if (nstage == 0) {
    snprintf(err, errlen, "shared memory budget exceeded");
    return cudaErrorInvalidValue;
  }
  const SmemLayout L = smem_layout(s.C, dil, nstage, stem != nullptr);
  // at least ~12 row-tiles per lane, at most one CTA per SM
  long long want = (geo.total + 23) / 24;
  int grid = (int)(want < 1 ? 1 : (want > n_sm ? n_sm : want));
  const size_t smem = L.total + 1024;
  switch (s.C) {
    case 16: return launch_c<16>(in, out, geo, wpack, bias, nstage, grid, smem, head, stem, st);
    case 32: return launch_c<32>(in, out, geo, wpack, bias, nstage, grid, smem, head, stem, st);
    case 48: return launch_c<48>(in, out, geo, wpack, bias, nstage, grid, smem, head, stem, st);
    case 64: return launch_c<64>(in, out, geo, wpack, bias, nstage, grid, smem, head, stem, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace smlm
