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
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <type_traits>
#include <vector>

#include "smlm_internal.cuh"
#include "umma_ptx.cuh"

namespace smlm {
namespace {

// warps 0-7 / 8-15: epilogue of lane 0 / 1; 16 / 18: producer of lane 0 / 1 (18 also owns the TMEM
// allocation), 17 / 19: MMA issuer of lane 0 / 1.  Eight epilogue warps per lane: warp pair
// (q, q + 4) shares TMEM lane quadrant q (32 pixels of the row tile) and splits the channels
// in halves.  The epilogue's instruction stream is latency-bound (about 4.5 cycles per
// instruction with so few warps per scheduler: profiles/), and its length per step, not the
// MMA time, set the pace of a lane; half the channels per thread halve it.
constexpr int kThreads = 640;
constexpr int kEpiWarps = 8;  // per lane
constexpr int kTileM = 128;
constexpr int kMaxStages = 6;
constexpr int kTmemCols = 512;
constexpr int kLaneCols = 256;  // TMEM columns reserved per lane (3C <= 192)
constexpr int kMaxDevices = 64;
constexpr int kLaneBars = 2 * kMaxStages + 2;  // mbarriers per lane (SmemLayout)
constexpr int kMaxDilation = 16;  // the paper's dilation set is (2, 4, 8, 16)

// zero source for the padded parts of a row segment: at most (127 + 16) pixels x 16 B
__device__ __align__(16) uint4 g_zeros[160];

using namespace ptx;

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
// Chunk k (8 channels) of a_0 for the four pixels lane, lane + 32, lane + 64, lane + 96 of a
// 128-pixel segment, rounded to bf16 and written to the stage in operand layout.  One warp
// per chunk: every weight fetched from shared memory (a broadcast read costs a full
// wavefront per 4 bytes) serves four pixels, and the shared-memory pipe - which the tensor
// core's operand fetch needs - sees a quarter of the traffic of a pixel-per-thread mapping.
// Two channels per fma.rn.f32x2 (two independent IEEE fp32 FMAs); per channel the chain is
// bias, then the nine taps in (ky, kx) order - the same as stem.cu, so the bits agree.
template <int C>
__device__ __forceinline__ void stem_chunk4(const float* const (&rows)[3], int d, int lane, int k,
                                            const float* ws, const float* bs, int relu, int x0, int W,
                                            uint8_t* stage, uint32_t plane) {
  unsigned long long acc[4][4];
  {
    const ulonglong2 b01 = *reinterpret_cast<const ulonglong2*>(bs + k * 8);
    const ulonglong2 b23 = *reinterpret_cast<const ulonglong2*>(bs + k * 8 + 4);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      acc[p][0] = b01.x;
      acc[p][1] = b01.y;
      acc[p][2] = b23.x;
      acc[p][3] = b23.y;
    }
  }
#pragma unroll
  for (int t = 0; t < 9; ++t) {
    const ulonglong2 w01 = *reinterpret_cast<const ulonglong2*>(ws + t * C + k * 8);
    const ulonglong2 w23 = *reinterpret_cast<const ulonglong2*>(ws + t * C + k * 8 + 4);
    const float* prow = rows[t / 3] + d + lane + t % 3;
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const float x = prow[32 * p];
      const unsigned long long xx = pack2f(x, x);
      acc[p][0] = ffma2(xx, w01.x, acc[p][0]);
      acc[p][1] = ffma2(xx, w01.y, acc[p][1]);
      acc[p][2] = ffma2(xx, w23.x, acc[p][2]);
      acc[p][3] = ffma2(xx, w23.y, acc[p][3]);
    }
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    uint32_t ow[4];
    const bool valid = x0 + lane + 32 * p < W;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float v0 = __uint_as_float((uint32_t)acc[p][i]), v1 = __uint_as_float((uint32_t)(acc[p][i] >> 32));
      if (relu) {
        v0 = fmaxf(v0, 0.0f);
        v1 = fmaxf(v1, 0.0f);
      }
      __nv_bfloat162 h = __floats2bfloat162_rn(v0, v1);
      ow[i] = valid ? *reinterpret_cast<uint32_t*>(&h) : 0u;
    }
    *reinterpret_cast<uint4*>(stage + (size_t)k * plane + (size_t)(d + lane + 32 * p) * 16u) =
        make_uint4(ow[0], ow[1], ow[2], ow[3]);
  }
}

constexpr int kRingRows = 8;  // STEM: ring of normalised input rows per lane

struct SmemLayout {
  uint32_t w_off, w_bytes;
  uint32_t stage_off, stage_bytes;  // per (lane, stage)
  uint32_t xch_off;   // HEAD: float [2 lanes][128 px][8] partial head sums of the upper channel half
  uint32_t stem_off;  // STEM: float stem weights [9][C], stem bias [C]
  uint32_t patch_off, patch_bytes, patch_row;  // STEM: per lane: float xhat[kRingRows][patch_row]
  uint32_t raw_off;   // STEM: uint32 raw[2 lanes][2 sets][5 fields][256 threads] (cp.async landing slots)
  uint32_t bar_off;
  uint32_t tmem_off;
  uint32_t total;
  int nstage;
};

__host__ __device__ inline SmemLayout smem_layout(int C, int d, int nstage, bool stem, bool head) {
  SmemLayout L;
  L.w_off = 0;
  L.w_bytes = 30u * C * C;  // 3 kx * C/8 chunks * 5C rows * 16 B
  L.stage_bytes = (((uint32_t)(C / 8) * (kTileM + 2 * d) * 16u) + 127u) & ~127u;
  L.stage_off = (L.w_off + L.w_bytes + 127u) & ~127u;
  L.nstage = nstage;
  L.xch_off = L.stage_off + 2u * nstage * L.stage_bytes;
  L.stem_off = L.xch_off + (head ? 2u * kTileM * 8u * 4u : 0u);
  L.patch_off = L.stem_off + (stem ? (uint32_t)(10 * C) * 4u : 0u);
  L.patch_row = (uint32_t)(kTileM + 2 * d + 2 + 3) & ~3u;  // the segment plus the stem's own 1-px halo
  L.patch_bytes = stem ? (uint32_t)kRingRows * L.patch_row * 4u : 0u;
  L.raw_off = L.patch_off + 2u * L.patch_bytes;
  L.bar_off = L.raw_off + (stem ? 2u * 2u * 5u * 256u * 4u : 0u);
  // barriers: wbar, per lane: full[kMaxStages], empty[kMaxStages], acc_full, acc_free
  L.tmem_off = L.bar_off + 8u * (1 + 2 * kLaneBars);
  L.total = L.tmem_off + 16u;
  return L;
}

// HEAD: the layer is the last one of the trunk.  The epilogue evaluates the heads on the ROUNDED
// output values (same order and fmaf chain as head_post.cu, so both produce the same bits):
// the detection logit o_p for every pixel, the other heads for pixels with o_p > lthr; the
// activation map itself is not stored.
// STEM: the layer is the first one; its input a_0 is computed in the kernel (see above).
template <int C, bool HEAD, bool STEM, bool F16>
__global__ void __launch_bounds__(kThreads, 1)
    conv_umma_kernel(const __nv_bfloat16* __restrict__ in, __nv_bfloat16* __restrict__ out, Geo geo,
                     const uint8_t* __restrict__ wpack, int nstage, const __grid_constant__ LayerConst lc,
                     const __grid_constant__ HeadArgs ha, const __grid_constant__ StemArgs sa) {
  extern __shared__ uint8_t smem_raw[];
  const SmemLayout L = smem_layout(C, geo.d, nstage, STEM, HEAD);
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 1023u) & ~1023u;  // the launch reserves 1 KB of slack for this
  uint8_t* smem = smem_raw + (sbase - sraw);
  // Role of a warp.  The schedulers favour the highest warp id among eligible warps, so the
  // four single-thread roles (which feed the tensor pipe and must never queue behind the
  // epilogue's long instruction streams) take the top ids: role 0 / 2 = producer of lane 0 / 1,
  // 1 / 3 = MMA issuer of lane 0 / 1; warps 0 .. 15 are the epilogue (quadrant = warp % 4).
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int role = warp - 2 * kEpiWarps;  // < 0: epilogue
  const int d = geo.d;

  const uint32_t wbar = sbase + L.bar_off;
  auto lane_bar = [&](int ln, int i) { return sbase + L.bar_off + 8u * (1 + ln * kLaneBars + i); };
  auto full_bar = [&](int ln, int s) { return lane_bar(ln, s); };
  auto empty_bar = [&](int ln, int s) { return lane_bar(ln, kMaxStages + s); };
  auto acc_full_bar = [&](int ln) { return lane_bar(ln, 2 * kMaxStages); };
  auto acc_free_bar = [&](int ln) { return lane_bar(ln, 2 * kMaxStages + 1); };
  auto stage_addr = [&](int ln, int s) { return sbase + L.stage_off + (uint32_t)(ln * nstage + s) * L.stage_bytes; };
  auto ring_row = [&](int ln, int r) {
    return reinterpret_cast<float*>(smem + L.patch_off + (uint32_t)ln * L.patch_bytes) +
           (size_t)(r & (kRingRows - 1)) * L.patch_row;
  };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + L.tmem_off);

  // ---- one-time setup
  if (threadIdx.x == 0) {
    mbar_init(wbar, 1);
    for (int ln = 0; ln < 2; ++ln) {
      for (int s = 0; s < kMaxStages; ++s) {
        // full: the TMA transaction count, or (STEM) the epilogue warps
        mbar_init(full_bar(ln, s), STEM ? kEpiWarps : 1);
        mbar_init(empty_bar(ln, s), 1 + kEpiWarps);  // MMA commit + one arrival per epilogue warp
      }
      mbar_init(acc_full_bar(ln), 1);
      mbar_init(acc_free_bar(ln), kEpiWarps);  // one arrival per epilogue warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (role == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + L.tmem_off),
                 "n"(kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  float* stem_w_s = reinterpret_cast<float*>(smem + L.stem_off);  // [9][C]
  float* stem_b_s = stem_w_s + 9 * C;
  if (STEM) {
    for (int i = threadIdx.x; i < 9 * C; i += kThreads) stem_w_s[i] = sa.w[i / C][i % C];
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
  if (role == 0 || role == 2) {
    // =========================== TMA producers: warp 0 -> lane 0, warp 2 -> lane 1 ========
    const int ln = role >> 1;
    if (role == 0 && elect_one()) {
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
      // (the lane's epilogue warps produce the input themselves, see below)
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
  } else if (role == 1 || role == 3) {
    // =========================== MMA issuers: warp 1 -> lane 0, warp 3 -> lane 1 ==========
    // One issuing warp per lane: the tensor pipe's instruction queue is short, so while one
    // warp is busy with barriers and bookkeeping between two steps the other one's MMAs keep
    // the pipe fed (the lanes are independent: own TMEM columns, own stages).
    const int ln = role >> 1;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    mbar_wait(wbar, 0);
    constexpr uint32_t idesc = umma_idesc(kTileM, 3 * C, F16);
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
  } else {
    // =========================== epilogue ===========================
    const int e = warp;
    const int ln = e >> 3;       // lane of the CTA
    const int qd = warp & 3;     // TMEM lane quadrant this warp may access
    const int half = (e >> 2) & 1;
    constexpr int CH = C / 2;    // channels per thread
    constexpr int KH = C / 16;   // 8-channel chunks per thread
    const int k0 = half * KH;    // first chunk
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int px = qd * 32 + lane;
    const uint32_t tlane = tmem_base + ((uint32_t)(qd * 32) << 16) + (uint32_t)ln * kLaneCols + (uint32_t)(half * CH);
    // the CH accumulator columns of this thread: groups of 16 (and one of 8 when CH % 16 == 8)
    auto ld_cols = [&](uint32_t slot, uint32_t (&acc)[CH]) {
#pragma unroll
      for (int g = 0; g + 16 <= CH; g += 16)
        tc_ld16(tlane + slot * C + g, *reinterpret_cast<uint32_t(*)[16]>(&acc[g]));
      if (CH % 16) tc_ld8(tlane + slot * C + (CH - 8), *reinterpret_cast<uint32_t(*)[8]>(&acc[CH - 8]));
    };
    // a finished slot is re-armed with zeros (registers only); the bias is added below
    auto init_slot = [&](uint32_t slot) {
      const uint32_t z16[16] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
      const uint32_t z8[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
#pragma unroll
      for (int g = 0; g + 16 <= CH; g += 16) tc_st16(tlane + slot * C + g, z16);
      if (CH % 16) tc_st8(tlane + slot * C + (CH - 8), z8);
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

    // STEM (K1 folded in): the lane's 256 epilogue threads build the layer's input themselves.
    // For the valid step that is two steps ahead of the one being retired (the MMAs of the
    // step in between are running meanwhile) they need the normalised rows row-1, row, row+1,
    // columns x0-d-1 .. x0+128+d.  Rows live in a ring in shared memory; when a step continues
    // the previous one with d = 1 only its last row is new.  One thread per aligned 32-bit
    // word of a raw uint16 row (two pixels; plus the two offset / gain values of a per-pixel
    // camera): the words are fetched with cp.async one call ahead into the thread's own
    // shared-memory slots - asynchronous copies stay in flight across the fences and barrier
    // arrivals of a step, which ordinary loads do not - and normalised into the ring now.  A
    // 256-thread named barrier makes the rows visible; then warp = channel chunk, thread =
    // four pixels compute a_0 into the stage (stem_chunk4), plus the 2d halo pixels shared out
    // by channel.  (A word may straddle the end of a row, so up to two bytes beyond the last
    // pixel of the frame buffer are read; they are never used.)
    struct StemPend {
      Step sp;
      int base;    // ring slot of the step's first row
      bool reuse;  // rows 0 and 1 are the previous step's rows 1 and 2
    };
    const int ew = e & 7;            // epilogue warp within the lane: the stem's channel chunk
    const int et = ew * 32 + lane;   // thread within the lane's epilogue
    const int pcols = kTileM + 2 * d + 2;
    const int aw = pcols / 2 + 1;    // words that cover a row of pcols pixels at any alignment
    const int lane_bar = 9 + ln;
    // this thread's word: row 2 (the new row) for et < aw, row 0 for aw <= et < 2 aw, row 1 next
    const int my_py = et < aw ? 2 : (et < 2 * aw ? 0 : (et < 3 * aw ? 1 : -1));
    const int my_w = et < aw ? et : (et < 2 * aw ? et - aw : et - 2 * aw);
    uint32_t* raw_base = reinterpret_cast<uint32_t*>(smem + L.raw_off) + (size_t)ln * 2 * 5 * 256 + et;
    ValidSteps ssteps;
    StemPend pend{{0, 0, 0}, 0, false};
    bool have_pend = false;
    int sset = 0;
    uint32_t sst = 0, sempty_par = 1;
    // pixel column (in the patch) of the first pixel of this thread's word, and its frame position
    auto word_geom = [&](const StemPend& pd, int& col0, long long& q0, bool& row_ok, const uint16_t*& frame) {
      const View v = view_of(sa.vs, pd.sp.b, geo.H, geo.W);
      frame = sa.frames + (size_t)(v.frame - sa.frame_base) * sa.vs.Hf * sa.vs.Wf;
      const int fy = v.wy0 + pd.sp.row - 1 + my_py, fx0 = v.wx0 + pd.sp.x0 - d - 1;
      row_ok = fy >= 0 && fy < sa.vs.Hf;
      const long long qrow = (long long)fy * sa.vs.Wf + fx0;  // pixel index of patch column 0
      // alignment of patch column 0 inside its 32-bit word: 0 or 1 pixels
      const int sh = (int)((reinterpret_cast<uintptr_t>(frame + qrow) >> 1) & 1);
      col0 = 2 * my_w - sh;
      q0 = qrow + col0;
    };
    auto stem_issue = [&](const StemPend& pd, int set) {
      if (my_py < 0 || (pd.reuse && my_py != 2)) return;
      int col0;
      long long q0;
      bool row_ok;
      const uint16_t* frame;
      word_geom(pd, col0, q0, row_ok, frame);
      uint32_t* slot = raw_base + (size_t)set * 5 * 256;
      const View v = view_of(sa.vs, pd.sp.b, geo.H, geo.W);
      const int fxa = v.wx0 + pd.sp.x0 - d - 1 + col0;  // frame x of the word's first pixel
      const bool in0 = row_ok && col0 >= 0 && col0 < pcols && fxa >= 0 && fxa < sa.vs.Wf;
      const bool in1 = row_ok && col0 + 1 >= 0 && col0 + 1 < pcols && fxa + 1 >= 0 && fxa + 1 < sa.vs.Wf;
      if (in0 || in1) cp_async4(smem_u32(slot), frame + q0);
      if (sa.np.offset_map) {
        if (in0) {
          cp_async4(smem_u32(slot + 256), sa.np.offset_map + q0);
          cp_async4(smem_u32(slot + 3 * 256), sa.np.gain_map + q0);
        }
        if (in1) {
          cp_async4(smem_u32(slot + 2 * 256), sa.np.offset_map + q0 + 1);
          cp_async4(smem_u32(slot + 4 * 256), sa.np.gain_map + q0 + 1);
        }
      }
    };
    auto stem_store = [&](const StemPend& pd, int set) {
      if (my_py < 0 || (pd.reuse && my_py != 2)) return;
      int col0;
      long long q0;
      bool row_ok;
      const uint16_t* frame;
      word_geom(pd, col0, q0, row_ok, frame);
      const View v = view_of(sa.vs, pd.sp.b, geo.H, geo.W);
      const int fxa = v.wx0 + pd.sp.x0 - d - 1 + col0;
      const uint32_t* slot = raw_base + (size_t)set * 5 * 256;
      const uint32_t wv = slot[0];
      float* rowp = ring_row(ln, pd.base + my_py);
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int col = col0 + i;
        if (col < 0 || col >= pcols) continue;
        const bool in = row_ok && fxa + i >= 0 && fxa + i < sa.vs.Wf;
        float xh = 0.0f;
        if (in) {
          const float adu = (float)(i ? (wv >> 16) : (wv & 0xffffu));
          const float om = sa.np.offset_map ? __uint_as_float(slot[(1 + i) * 256]) : sa.np.offset;
          const float gm = sa.np.offset_map ? __uint_as_float(slot[(3 + i) * 256]) : sa.np.gain;
          xh = ((adu - om) / gm) / sa.np.norm_scale;
        }
        rowp[col] = xh;
      }
    };
    auto stem_advance = [&]() {
      if (!have_pend) return;
      cp_async_wait_all();  // this thread's words of the pending step (issued one call ago)
      stem_store(pend, sset);
      StemPend nx;
      const bool have_next = ssteps.next(geo, nx.sp);
      if (have_next) {
        nx.reuse = d == 1 && nx.sp.b == pend.sp.b && nx.sp.x0 == pend.sp.x0 && nx.sp.row == pend.sp.row + 1;
        nx.base = pend.base + (nx.reuse ? 1 : 3);
        stem_issue(nx, sset ^ 1);  // in flight until the next call
      }
      cp_async_commit();
      asm volatile("bar.sync %0, 256;" ::"r"(lane_bar) : "memory");
      const float* const rows[3] = {ring_row(ln, pend.base), ring_row(ln, pend.base + 1),
                                    ring_row(ln, pend.base + 2)};
      const int x0 = pend.sp.x0;
      mbar_wait(empty_bar(ln, sst), sempty_par);
      uint8_t* stage = smem + (stage_addr(ln, sst) - sbase);
      if (ew < C / 8) stem_chunk4<C>(rows, d, lane, ew, stem_w_s, stem_b_s, sa.relu, x0, geo.W, stage, plane);
      // the 2d halo pixels of the segment (positions [0, d) and [d + 128, 128 + 2d)): one
      // (pixel, channel) output per thread and pass, the same fmaf chain
      for (int o = et; o < 2 * d * C; o += 32 * kEpiWarps) {
        const int h = o / C, c = o - h * C;
        const int pos = h < d ? h : kTileM + h;  // position in the (128 + 2d)-pixel segment
        const int x = x0 - d + pos;              // window coordinate
        float a = stem_b_s[c];
#pragma unroll
        for (int t = 0; t < 9; ++t) a = fmaf(rows[t / 3][pos + t % 3], stem_w_s[t * C + c], a);
        if (sa.relu) a = fmaxf(a, 0.0f);
        const __nv_bfloat16 hb = __float2bfloat16_rn(a);
        const uint16_t bits = (x >= 0 && x < geo.W) ? *reinterpret_cast<const uint16_t*>(&hb) : (uint16_t)0;
        *reinterpret_cast<uint16_t*>(stage + (size_t)(c >> 3) * plane + (size_t)pos * 16u + (c & 7) * 2) = bits;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(full_bar(ln, sst));
      if (++sst == (uint32_t)nstage) {
        sst = 0;
        sempty_par ^= 1u;
      }
      pend = nx;
      have_pend = have_next;
      sset ^= 1;
    };
    if (STEM) {
      ssteps.init(geo, 2 * blockIdx.x + ln, nlanes);
      have_pend = ssteps.next(geo, pend.sp);
      if (have_pend) stem_issue(pend, sset);
      cp_async_commit();
      stem_advance();
      stem_advance();
    }

    // HEAD: every head is the sum of two fmaf chains, one per channel half (head_post.cu
    // evaluates the same two chains), so the warp pair exchanges partial sums: half 1 hands
    // its six partials to half 0 through shared memory (one 64-thread named barrier).
    float* xch = reinterpret_cast<float*>(smem + L.xch_off) + (size_t)(ln * kTileM + px) * 8;
    const int pair_bar = 1 + ln * 4 + qd;

    LaneRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    Run run;
    uint32_t slot = 2, acc_par = 0, st = 0, prev_st = 0;
    bool prev_valid = false;
    uint4 res[KH];
#pragma unroll
    for (int k = 0; k < KH; ++k) res[k] = make_uint4(0u, 0u, 0u, 0u);
    while (runs.next(geo, run)) {
      const int x = run.x0 + px;
      int row = run.r + (run.i0 - 1) * d;  // input row of the step; the output row is row - d
      uint4* orow = reinterpret_cast<uint4*>(out) +
                    (((size_t)run.b * (C / 8) + k0) * geo.H * geo.W + (long long)(row - d) * geo.W + x);
      for (int j = 0; j < run.n + 2; ++j, row += d, orow += (size_t)d * geo.W) {
        const bool in_valid = row >= 0 && row < geo.H;
        const bool out_valid = j >= 2 && row - d < geo.H;
        const bool store = out_valid && x < geo.W;
        mbar_wait(acc_full_bar(ln), acc_par);
        acc_par ^= 1u;
        tc_fence_after();
        uint32_t acc[CH];
        if (out_valid) {
          ld_cols(slot, acc);
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
        // ReLU(acc + bias) + residual, one RNE rounding, store; HEAD: this half's partial sums
        // of the six heads on the rounded values.  Specialised on the channel half so that
        // bias and head weights are compile-time-indexed kernel parameters.
        float hp[6] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
        auto post = [&](auto HALF) {
          constexpr int kHalf = decltype(HALF)::value;
          if (HEAD && kHalf == 0) {
#pragma unroll
            for (int h = 0; h < 6; ++h) hp[h] = ha.b[h];
          }
#pragma unroll
          for (int kk = 0; kk < KH; ++kk) {
            constexpr int kc0 = kHalf * KH;
            const uint4 rk = kEarly ? res[kk] : rprev[(size_t)(kc0 + kk) * (plane / 16u)];
            const uint32_t rw[4] = {rk.x, rk.y, rk.z, rk.w};
            uint32_t ow[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int c0 = (kc0 + kk) * 8 + 2 * i;
              float r0, r1;
              unpack2<F16>(rw[i], r0, r1);
              float v0 = r0 + fmaxf(__uint_as_float(acc[kk * 8 + 2 * i]) + lc.bias[c0], 0.0f);
              float v1 = r1 + fmaxf(__uint_as_float(acc[kk * 8 + 2 * i + 1]) + lc.bias[c0 + 1], 0.0f);
              ow[i] = pack2<F16>(v0, v1);
              if (HEAD) {
                float a0, a1;
                unpack2<F16>(ow[i], a0, a1);
#pragma unroll
                for (int h = 0; h < 6; ++h) hp[h] = fmaf(a0, ha.w[c0][h], hp[h]);
#pragma unroll
                for (int h = 0; h < 6; ++h) hp[h] = fmaf(a1, ha.w[c0 + 1][h], hp[h]);
              }
            }
            if (!HEAD) orow[(size_t)kk * plane_px] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
          }
        };
        if (store) {
          if (half == 0) post(std::integral_constant<int, 0>{});
          else post(std::integral_constant<int, 1>{});
        }
        if (HEAD && out_valid) {
          if (half == 1) {
            *reinterpret_cast<float4*>(xch) = make_float4(hp[0], hp[1], hp[2], hp[3]);
            *reinterpret_cast<float2*>(xch + 4) = make_float2(hp[4], hp[5]);
          }
          asm volatile("bar.sync %0, 64;" ::"r"(pair_bar) : "memory");
          if (half == 0 && store) {
            const float4 o03 = *reinterpret_cast<const float4*>(xch);
            const float2 o45 = *reinterpret_cast<const float2*>(xch + 4);
            const float lg = hp[0] + o03.x;
            const size_t q = ((size_t)run.b * geo.H + (row - d)) * geo.W + x;
            ha.logit[q] = lg;
            if (lg > ha.lthr) {  // candidate record: heads 1 .. 5 (pre-activation; zero beyond n_h)
              float4* cq = reinterpret_cast<float4*>(ha.cand) + q * 2;
              cq[0] = make_float4(hp[1] + o03.y, hp[2] + o03.z, hp[3] + o03.w, hp[4] + o45.x);
              cq[1] = make_float4(hp[5] + o45.y, 0.0f, 0.0f, 0.0f);
            }
          }
          asm volatile("bar.sync %0, 64;" ::"r"(pair_bar) : "memory");  // xch may be rewritten
        }
        if (kEarly) {
          if (in_valid) {
            const uint4* rp = reinterpret_cast<const uint4*>(smem + (stage_addr(ln, st) - sbase) +
                                                             (uint32_t)(d + px) * 16u);
#pragma unroll
            for (int kk = 0; kk < KH; ++kk) res[kk] = rp[(size_t)(k0 + kk) * (plane / 16u)];
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
  if (role == 2) {
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

uint16_t f16_bits(float f) {
  const __half h = __float2half_rn(f);
  uint16_t u;
  std::memcpy(&u, &h, 2);
  return u;
}

template <int C, bool HEAD, bool STEM, bool F16>
cudaError_t launch_chs(const void* in, void* out, Geo geo, const void* wpack, const LayerConst& lc, int nstage,
                       int grid, size_t smem, const HeadArgs& ha, const StemArgs& sa, cudaStream_t st) {
  static bool attr_done[kMaxDevices] = {};  // the attribute is per device
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (!attr_done[dev]) {
    cudaError_t e = cudaFuncSetAttribute(conv_umma_kernel<C, HEAD, STEM, F16>,
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
  return cudaLaunchKernelEx(&cfg, conv_umma_kernel<C, HEAD, STEM, F16>, (const __nv_bfloat16*)in,
                            (__nv_bfloat16*)out, geo, (const uint8_t*)wpack, nstage, lc, ha, sa);
}
template <int C>
cudaError_t launch_c(bool f16, const void* in, void* out, Geo geo, const void* wpack, const LayerConst& lc,
                     int nstage, int grid, size_t smem, const HeadArgs* ha, const StemArgs* sa, cudaStream_t st) {
  static const HeadArgs h0{};
  static const StemArgs s0{};
  if (f16) {  // the STEM variant exists in bf16 only (api.cu keeps K1 a kernel of its own in fp16)
    if (sa) return cudaErrorInvalidValue;
    if (ha) return launch_chs<C, true, false, true>(in, out, geo, wpack, lc, nstage, grid, smem, *ha, s0, st);
    return launch_chs<C, false, false, true>(in, out, geo, wpack, lc, nstage, grid, smem, h0, s0, st);
  }
  if (ha && sa) return launch_chs<C, true, true, false>(in, out, geo, wpack, lc, nstage, grid, smem, *ha, *sa, st);
  if (ha) return launch_chs<C, true, false, false>(in, out, geo, wpack, lc, nstage, grid, smem, *ha, s0, st);
  if (sa) return launch_chs<C, false, true, false>(in, out, geo, wpack, lc, nstage, grid, smem, h0, *sa, st);
  return launch_chs<C, false, false, false>(in, out, geo, wpack, lc, nstage, grid, smem, h0, s0, st);
}

// stages: as many as fit next to the resident weights (<= kMaxStages; >= 2 for any overlap of
// load and MMA; the STEM variant computes two steps ahead and needs >= 3)
int pick_stages(int C, int dil, bool stem, bool head) {
  int nstage = kMaxStages;
  const int min_stage = stem ? 3 : 2;
  while (nstage >= min_stage && smem_layout(C, dil, nstage, stem, head).total + 1024 > 227u * 1024u) --nstage;
  return nstage >= min_stage ? nstage : 0;
}

}  // namespace

size_t umma_packed_weight_bytes(int C) { return (size_t)30 * C * C; }

// Shared-memory image of one layer's weights: for kx, input chunk kc: 5C rows of 16 B
// (8 input channels), rows = output channels of ky = 1, 0, 2, 1, 0.
float round_to_act(float v, int dt) {
  uint32_t u;
  if (dt == ACT_BF16) u = (uint32_t)bf16_bits(v) << 16;
  else if (dt == ACT_F16) return __half2float(__float2half_rn(v));
  else return v;
  float r;
  std::memcpy(&r, &u, 4);
  return r;
}

void umma_pack_weights_host(int C, const float* w /*[C][C][3][3]*/, void* dst, bool f16) {
  static const int ky_seq[5] = {1, 0, 2, 1, 0};
  uint16_t* o = static_cast<uint16_t*>(dst);
  for (int kx = 0; kx < 3; ++kx)
    for (int kc = 0; kc < C / 8; ++kc)
      for (int n = 0; n < 5 * C; ++n) {
        const int ky = ky_seq[n / C], co = n % C;
        for (int j = 0; j < 8; ++j) {
          const int ci = kc * 8 + j;
          const float v = w[(((size_t)co * C + ci) * 3 + ky) * 3 + kx];
          o[(((size_t)(kx * (C / 8) + kc) * 5 * C) + n) * 8 + j] = f16 ? f16_bits(v) : bf16_bits(v);
        }
      }
}

bool conv_umma_supports(int C, int dil, bool stem) {
  return C >= 16 && C <= 64 && C % 16 == 0 && dil >= 1 && dil <= kMaxDilation && pick_stages(C, dil, stem, true) > 0;
}

cudaError_t launch_conv_umma(bool f16, const void* in, void* out, ActShape s, int dil, const void* wpack,
                             const LayerConst& lc, const HeadArgs* head, const StemArgs* stem, int n_sm,
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
  const int nstage = pick_stages(s.C, dil, stem != nullptr, head != nullptr);
  if (nstage == 0) {
    snprintf(err, errlen, "shared memory budget exceeded");
    return cudaErrorInvalidValue;
  }
  const SmemLayout L = smem_layout(s.C, dil, nstage, stem != nullptr, head != nullptr);
  // at least ~12 row-tiles per lane, at most one CTA per SM
  long long want = (geo.total + 23) / 24;
  int grid = (int)(want < 1 ? 1 : (want > n_sm ? n_sm : want));
  const size_t smem = L.total + 1024;
  switch (s.C) {
    case 16: return launch_c<16>(f16, in, out, geo, wpack, lc, nstage, grid, smem, head, stem, st);
    case 32: return launch_c<32>(f16, in, out, geo, wpack, lc, nstage, grid, smem, head, stem, st);
    case 48: return launch_c<48>(f16, in, out, geo, wpack, lc, nstage, grid, smem, head, stem, st);
    case 64: return launch_c<64>(f16, in, out, geo, wpack, lc, nstage, grid, smem, head, stem, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace smlm
