// Dense-block layer of the paper's own topology (dloc.h; "each layer [utilizes]
// outputs from all preceding layers", P:144 dilations 2-4-8-16) on the tcgen05 tensor cores:
//     out[co] = ReLU(b[co] + sum_{ci, ky, kx} w[co][ci][ky][kx] in[ci][y + (ky-1) d][x + (kx-1) d])
// with C_in = C0 + i G input channels (a range of planes of the block's concatenation buffer)
// and only C_out = G (16 or 32) output channels, written to the next planes of the SAME buffer.
//
// The generic kernel of conv_gen.cu handles this shape badly (profiles/launches_dloc_r2.md):
// one work item per output row fetches every input row three times, and an MMA with N = 16
// re-reads its 4 KB A tile for 512 B of B.  This kernel is the row-chain walk of conv_umma.cu
// for C_in != C_out: M = 128 pixels of one row, one MMA D[128 x 3 C_out] += A[128 x 16]
// B[16 x 3 C_out] feeds the three output rows that share the input row (three TMEM slots of
// C_out columns), a lane walks the rows r, r+d, r+2d, ... of one residue class, every input
// row is fetched ONCE (C_in / 8 bulk copies of (128 + 2d) pixels x 16 B) and the layer's
// weights stay resident in shared memory (<= 46 KB).  No residual (the dense concatenation is
// the skip), so the epilogue never touches the stages.  Two lanes per CTA as in conv_umma.cu:
// warps 0-3 / 4-7 epilogue of lane 0 / 1 (one TMEM lane quadrant each), 8 / 10 TMA producer,
// 9 / 11 MMA issuer.  The layer is HBM-bound: 2 C_in + 2 C_out bytes per pixel.
//
// STEM variant (K1 of smlm.h on the tensor cores; BASELINE.json north_star (a)): uint16 unpack,
// ((adu - offset) / gain) / norm_scale and the 3x3 stem convolution 1 -> C in one kernel that is
// bound by its HBM WRITE (2 B in, 2C B out per pixel) instead of by fp32 FMA issue (stem.cu: 670
// thread-instructions per pixel).  No map is read: the lane's producer warp computes the
// operand row itself.  fp32 accuracy on 16-bit tensor cores by splitting: xhat = x_h + x_m + x_l
// and w = w_h + w_m + w_l into three 16-bit pieces each (24 of fp32's 24 mantissa bits with
// bf16), and letting six of the K = 16 input channels carry the pairings (x_h w_h), (x_h w_m),
// (x_m w_h), (x_h w_l), (x_l w_h), (x_m w_m); the dropped ones are below 2^-24 relative.  The
// products are exact in the fp32 accumulator, so a_0 differs from the fmaf chain of stem.cu
// only in summation order (~1 fp32 ulp).  One MMA per horizontal tap and row: the tensor work
// is nothing, the kernel streams.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>

#include "dloc_internal.cuh"
#include "umma_ptx.cuh"

namespace smlm {
namespace {

using namespace ptx;

constexpr int kThreads = 384;   // 12 warps
constexpr int kStemThreads = 576;  // STEM: + 3 more operand-building warps per lane (warps 12-14 / 15-17)
constexpr int kStemProd = 4;       // producer warps per lane in the STEM variant
constexpr int kEpiWarps = 4;    // per lane
constexpr int kTileM = 128;
constexpr int kMaxStages = 4;
constexpr int kTmemCols = 512;
constexpr int kLaneCols = 256;  // TMEM columns reserved per lane (3 C_out <= 192)
constexpr int kLaneBars = 2 * kMaxStages + 2;
constexpr int kMaxDevices = 64;

__device__ __align__(16) uint4 g_czeros[160];  // zero source for the padded parts of a row segment

struct CGeo {
  int B, H, W, d;         // d: row step of a chain = vertical dilation (1 for a 1x1 convolution)
  int dx;                 // horizontal dilation = x halo of a row segment (0 for a 1x1 convolution)
  int nseg, Lmax;
  long long total;
  int CI;                 // input channels (multiple of 16)
  int in_planes;          // planes per view of the input buffer
  int out_planes, co_plane0;
  float* out_f32;         // != nullptr: planar fp32 maps [B][n_valid][H][W] instead (the head maps of dloc.h)
  int n_valid;
};

struct CRun {
  int b, x0, r, i0, n;
};
struct CRuns {
  long long g, g1;
  __device__ void init(const CGeo& geo, int lane_id, int nlanes) {
    g = geo.total * lane_id / nlanes;
    g1 = geo.total * (lane_id + 1) / nlanes;
  }
  __device__ bool next(const CGeo& geo, CRun& run) {
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

struct CSmem {
  uint32_t w_bytes, stage_off, stage_bytes, bar_off, tmem_off, total;
};
__host__ __device__ inline CSmem chain_smem(int CI, int CO, int kx_taps, int dx, int nstage) {
  CSmem L;
  L.w_bytes = (uint32_t)kx_taps * (CI / 8) * 5u * CO * 16u;
  L.stage_bytes = (((uint32_t)(CI / 8) * (kTileM + 2 * dx) * 16u) + 127u) & ~127u;
  L.stage_off = (L.w_bytes + 127u) & ~127u;
  L.bar_off = L.stage_off + 2u * nstage * L.stage_bytes;
  L.tmem_off = L.bar_off + 8u * (1 + 2 * kLaneBars);
  L.total = L.tmem_off + 16u;
  return L;
}

// STEM: where the operand rows come from (the frames, not a map)
struct StemSrc {
  const uint16_t* frames;  // device; frame f of the call at frames + (f - frame_base) Hf Wf
  int frame_base;
  ViewSet vs;
  NormParams np;
};

// max(v, 0) and the RNE rounding of two values in one conversion (low half = first argument)
template <bool F16>
__device__ __forceinline__ uint32_t pack2_relu(float lo, float hi) {
  uint32_t d;
  if (F16) asm("cvt.rn.relu.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  else asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

// 16-bit pieces of v: v ~ h + m + l
template <bool F16>
__device__ __forceinline__ void split3(float v, uint32_t& h, uint32_t& m, uint32_t& l) {
  if (F16) {
    const __half a = __float2half_rn(v);
    const float r1 = v - __half2float(a);
    const __half b = __float2half_rn(r1);
    const __half c = __float2half_rn(r1 - __half2float(b));
    h = __half_as_ushort(a);
    m = __half_as_ushort(b);
    l = __half_as_ushort(c);
  } else {
    const __nv_bfloat16 a = __float2bfloat16_rn(v);
    const float r1 = v - __bfloat162float(a);
    const __nv_bfloat16 b = __float2bfloat16_rn(r1);
    const __nv_bfloat16 c = __float2bfloat16_rn(r1 - __bfloat162float(b));
    h = __bfloat16_as_ushort(a);
    m = __bfloat16_as_ushort(b);
    l = __bfloat16_as_ushort(c);
  }
}

// KX = 3: 3x3 convolution.  KX = 1: 1x1 convolution (the transition of a dense block) run through
// the same walk - one tap, no x halo, the weight rows of ky = 0 and ky = 2 are zero; the layer is
// HBM-bound by a wide margin, so the idle two thirds of each MMA's N do not show.
template <int CO, bool F16, int KX, bool STEM>
__global__ void __launch_bounds__(STEM ? kStemThreads : kThreads, 1)
    conv_chain_kernel(const uint8_t* __restrict__ in, uint8_t* __restrict__ out, CGeo geo,
                      const uint8_t* __restrict__ wpack, int nstage, const __grid_constant__ LayerConst lc, int relu,
                      const __grid_constant__ StemSrc ss) {
  extern __shared__ uint8_t smem_raw[];
  const int d = geo.d, dx = geo.dx, CI = geo.CI;
  const CSmem L = chain_smem(CI, CO, KX, dx, nstage);
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - sraw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int role = warp - 2 * kEpiWarps;  // < 0: epilogue; 0 / 2 producer of lane 0 / 1, 1 / 3 MMA issuer

  const uint32_t wbar = sbase + L.bar_off;
  auto lane_bar = [&](int ln, int i) { return sbase + L.bar_off + 8u * (1 + ln * kLaneBars + i); };
  auto full_bar = [&](int ln, int s) { return lane_bar(ln, s); };
  auto empty_bar = [&](int ln, int s) { return lane_bar(ln, kMaxStages + s); };
  auto acc_full_bar = [&](int ln) { return lane_bar(ln, 2 * kMaxStages); };
  auto acc_free_bar = [&](int ln) { return lane_bar(ln, 2 * kMaxStages + 1); };
  auto stage_addr = [&](int ln, int s) { return sbase + L.stage_off + (uint32_t)(ln * nstage + s) * L.stage_bytes; };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + L.tmem_off);
  const uint32_t plane_bytes_s = (uint32_t)(kTileM + 2 * dx) * 16u;  // one channel chunk of a stage
  // does the step of window row `row` bring in a row?  A map row must lie inside the window; a
  // STEM row inside the FRAME (smlm.h: xhat = 0 outside the frame - a window's neighbour rows
  // are real pixels, as in stem.cu)
  auto row_valid = [&](int wy0, int row) {
    if (STEM) return row >= -1 && row <= geo.H && wy0 + row >= 0 && wy0 + row < ss.vs.Hf;
    return row >= 0 && row < geo.H;
  };
  if (STEM) {
    // the second K chunk (channels 8-15) of every stage is constant: channels 8, 9, 10 = 1 (they
    // carry the three pieces of the bias through the centre tap), the rest 0
    uint4* zs = reinterpret_cast<uint4*>(smem + L.stage_off);
    const uint32_t one = F16 ? 0x3C00u : 0x3F80u;
    const uint32_t per_stage = L.stage_bytes / 16u, per_plane = plane_bytes_s / 16u;
    const uint32_t nz = 2u * nstage * per_stage;
    for (uint32_t i = threadIdx.x; i < nz; i += kStemThreads) {
      const uint32_t in_stage = i % per_stage;
      const bool chunk1 = in_stage >= per_plane && in_stage < 2u * per_plane;
      zs[i] = chunk1 ? make_uint4(one | (one << 16), one, 0u, 0u) : make_uint4(0u, 0u, 0u, 0u);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }

  if (threadIdx.x == 0) {
    mbar_init(wbar, 1);
    for (int ln = 0; ln < 2; ++ln) {
      for (int s = 0; s < kMaxStages; ++s) {
        mbar_init(full_bar(ln, s), STEM ? kStemProd : 1);  // the TMA transaction count, or the operand-building warps
        mbar_init(empty_bar(ln, s), 1);  // the MMA commit only: no residual, the epilogue never reads a stage
      }
      mbar_init(acc_full_bar(ln), 1);
      mbar_init(acc_free_bar(ln), kEpiWarps);
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
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int nlanes = 2 * gridDim.x;
  const uint32_t plane = (uint32_t)(kTileM + 2 * dx) * 16u;

  if (role == 0 || role == 2 || role >= 4) {
    // =========================== TMA producers (STEM: the warps that build the operand rows)
    const int ln = role >= 4 ? (role - 4) / (kStemProd - 1) : role >> 1;
    const int sp = role >= 4 ? 1 + (role - 4) % (kStemProd - 1) : 0;  // STEM: which quarter of the positions
    if (role == 0 && elect_one()) {
      mbar_expect_tx(wbar, L.w_bytes);
      for (uint32_t off = 0; off < L.w_bytes; off += 16384u) {
        const uint32_t n = L.w_bytes - off < 16384u ? L.w_bytes - off : 16384u;
        bulk_load(sbase + off, wpack + off, n, wbar);
      }
    }
    __syncwarp();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t plane_bytes = (size_t)geo.H * geo.W * 16u;
    const size_t row_step = (size_t)d * geo.W * 16u;
    const int nk = CI / 8;
    CRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    CRun run;
    uint32_t st = 0, empty_par = 1;
    int last_x0 = -1, fills_left = 0;
    if (STEM) {
      // The warp builds the operand row of every valid step: 130 positions (x0 - 1 .. x0 + 128),
      // lane l owns positions l, l + 32, ...  The raw values of the NEXT valid step are loaded
      // before this step's arithmetic, so the global latency hides behind it.
      constexpr int NP = 2;  // positions sp * 32 + lane, and (the two halo positions 128, 129) + 128
      const size_t fpx = (size_t)ss.vs.Hf * ss.vs.Wf;
      struct Raw {
        float adu[NP], om[NP], gm[NP];
        bool in[NP];
      };
      auto fetch = [&](int b, int x0, int row, Raw& r) {
        const View v = view_of(ss.vs, b, geo.H, geo.W);
        const uint16_t* frame = ss.frames + (size_t)(v.frame - ss.frame_base) * fpx;
        const int fy = v.wy0 + row;
#pragma unroll
        for (int i = 0; i < NP; ++i) {
          const int p = sp * 32 + lane + 128 * i;
          const int fx = v.wx0 + x0 - 1 + p;
          r.in[i] = p < kTileM + 2 && fx >= 0 && fx < ss.vs.Wf;
          const size_t q = r.in[i] ? (size_t)fy * ss.vs.Wf + fx : 0;
          r.adu[i] = r.in[i] ? (float)__ldg(frame + q) : 0.0f;
          r.om[i] = (r.in[i] && ss.np.offset_map) ? __ldg(ss.np.offset_map + q) : ss.np.offset;
          r.gm[i] = (r.in[i] && ss.np.offset_map) ? __ldg(ss.np.gain_map + q) : ss.np.gain;
        }
      };
      // iterator over the valid steps of this lane, in walk order
      bool have_run = false;
      int j = 0, row = 0, wy0 = 0;
      auto next_step = [&](int& b, int& x0, int& rrow) {
        for (;;) {
          if (!have_run) {
            if (!runs.next(geo, run)) return false;
            have_run = true;
            j = 0;
            row = run.r + (run.i0 - 1) * d;
            wy0 = view_of(ss.vs, run.b, geo.H, geo.W).wy0;
          }
          while (j < run.n + 2) {
            const int r0 = row;
            ++j;
            row += d;
            if (row_valid(wy0, r0)) {
              b = run.b;
              x0 = run.x0;
              rrow = r0;
              return true;
            }
          }
          have_run = false;
        }
      };
      int b0, x00, r00;
      bool have = next_step(b0, x00, r00);
      Raw cur;
      if (have) fetch(b0, x00, r00, cur);
      while (have) {
        int b1, x01, r01;
        const bool have_next = next_step(b1, x01, r01);
        Raw nxt;
        if (have_next) fetch(b1, x01, r01, nxt);
        mbar_wait(empty_bar(ln, (int)st), empty_par);
        uint8_t* dst = smem + (stage_addr(ln, (int)st) - sbase);
#pragma unroll
        for (int i = 0; i < NP; ++i) {
          const int p = sp * 32 + lane + 128 * i;
          if (p >= kTileM + 2) continue;
          uint4 o = make_uint4(0u, 0u, 0u, 0u);
          if (cur.in[i]) {
            const float xh = ((cur.adu[i] - cur.om[i]) / cur.gm[i]) / ss.np.norm_scale;  // the oracle's operation order (G5)
            uint32_t h, m, l;
            split3<F16>(xh, h, m, l);
            o = make_uint4(h | (h << 16), m | (h << 16), l | (m << 16), 0u);  // (x_h, x_h, x_m, x_h, x_l, x_m, 0, 0)
          }
          *reinterpret_cast<uint4*>(dst + (size_t)p * 16u) = o;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(full_bar(ln, (int)st));
        if (++st == (uint32_t)nstage) {
          st = 0;
          empty_par ^= 1u;
        }
        cur = nxt;
        have = have_next;
      }
    } else
    while (runs.next(geo, run)) {
      const int xl = run.x0 - dx, xr = run.x0 + kTileM + dx;
      const int lo = xl > 0 ? xl : 0, hi = xr < geo.W ? xr : geo.W;
      const uint32_t pre = (uint32_t)(lo - xl) * 16u, mid = (uint32_t)(hi - lo) * 16u, post = (uint32_t)(xr - hi) * 16u;
      if (run.x0 != last_x0) {
        last_x0 = run.x0;
        fills_left = (pre | post) ? nstage : 0;
      }
      int row = run.r + (run.i0 - 1) * d;
      const uint8_t* src = in + ((size_t)run.b * geo.in_planes * geo.H * geo.W + (long long)row * geo.W + lo) * 16;
      for (int j = 0; j < run.n + 2; ++j, row += d, src += row_step) {
        if (row < 0 || row >= geo.H) continue;
        const uint32_t dst = stage_addr(ln, (int)st);
        const uint32_t bar = full_bar(ln, (int)st);
        const bool fill = fills_left > 0;
        mbar_wait(empty_bar(ln, (int)st), empty_par);
        if (elect_one()) {
          mbar_expect_tx(bar, (uint32_t)nk * (fill ? plane : mid));
          for (int k = 0; k < nk; ++k) bulk_load(dst + (uint32_t)k * plane + pre, src + (size_t)k * plane_bytes, mid, bar);
          if (fill) {
            for (int k = 0; k < nk; ++k) {
              if (pre) bulk_load(dst + (uint32_t)k * plane, g_czeros, pre, bar);
              if (post) bulk_load(dst + (uint32_t)k * plane + pre + mid, g_czeros, post, bar);
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
  } else if (role == 1 || role == 3) {
    // =========================== MMA issuers
    const int ln = role >> 1;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    mbar_wait(wbar, 0);
    constexpr uint32_t idesc = umma_idesc(kTileM, 3 * CO, F16);
    const uint32_t plane16 = (uint32_t)(kTileM + 2 * dx);
    constexpr uint32_t wplane16 = 5u * CO;
    constexpr uint32_t desc_hi = (128u >> 4) | (1u << 14);
    const uint32_t a_lo_base = (plane16 << 16) | (((sbase + L.stage_off) >> 4) & 0x3FFFu);
    const uint32_t b_lo_base = (wplane16 << 16) | ((sbase >> 4) & 0x3FFFu);
    const uint32_t stage16 = L.stage_bytes >> 4;
    const uint32_t dcol = __shfl_sync(0xffffffffu, tmem_base, 0) + (uint32_t)ln * kLaneCols;
    const int nks = CI / 16;
    CRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    CRun run;
    uint32_t st = 0, full_par = 0, free_par = 0, m = 0;
    while (runs.next(geo, run)) {
      int row = run.r + (run.i0 - 1) * d;
      const int wy0 = STEM ? view_of(ss.vs, run.b, geo.H, geo.W).wy0 : 0;
      for (int j = 0; j < run.n + 2; ++j, row += d) {
        const bool in_valid = row_valid(wy0, row);
        if (in_valid) mbar_wait(full_bar(ln, (int)st), full_par);
        mbar_wait(acc_free_bar(ln), free_par);
        free_par ^= 1u;
        tc_fence_after();
        const uint32_t win = m == 0 ? 0u : (m == 1 ? 2u : 1u);  // rows stored as ky = (1,0,2,1,0)
        const uint32_t a_lo = a_lo_base + ((uint32_t)ln * nstage + st) * stage16;
        const uint32_t b_lo = b_lo_base + win * CO;
        if (elect_one()) {
          if (in_valid) {
#pragma unroll
            for (int kx = 0; kx < KX; ++kx) {
              for (int ks = 0; ks < nks; ++ks) {
                const uint32_t al = a_lo + (uint32_t)(2 * ks) * plane16 + (uint32_t)(kx * dx);
                const uint32_t bl = b_lo + (uint32_t)(kx * (CI / 8) + 2 * ks) * wplane16;
                tc_mma(dcol, ((uint64_t)desc_hi << 32) | al, ((uint64_t)desc_hi << 32) | bl, idesc, 1u);
              }
            }
            tc_commit(empty_bar(ln, (int)st));
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
    // =========================== epilogue: ReLU(acc + bias), one RNE rounding, store
    const int ln = warp >> 2;
    const int qd = warp & 3;
    const int px = qd * 32 + lane;
    const uint32_t tlane = tmem_base + ((uint32_t)(qd * 32) << 16) + (uint32_t)ln * kLaneCols;
    auto zero_slot = [&](uint32_t slot) {
      const uint32_t z16[16] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
#pragma unroll
      for (int g = 0; g < CO; g += 16) tc_st16(tlane + slot * CO + g, z16);
    };
    zero_slot(0);
    zero_slot(1);
    zero_slot(2);
    tc_wait_st();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(acc_free_bar(ln));
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t plane_px = (size_t)geo.H * geo.W;
    CRuns runs;
    runs.init(geo, 2 * blockIdx.x + ln, nlanes);
    CRun run;
    uint32_t slot = 2, acc_par = 0;
    while (runs.next(geo, run)) {
      const int x = run.x0 + px;
      int row = run.r + (run.i0 - 1) * d;  // input row of the step; the output row is row - d
      uint4* orow = reinterpret_cast<uint4*>(out) +
                    (((size_t)run.b * geo.out_planes + geo.co_plane0) * geo.H * geo.W + (long long)(row - d) * geo.W + x);
      for (int j = 0; j < run.n + 2; ++j, row += d, orow += (size_t)d * geo.W) {
        const bool out_valid = j >= 2 && row - d < geo.H;
        mbar_wait(acc_full_bar(ln), acc_par);
        acc_par ^= 1u;
        tc_fence_after();
        uint32_t acc[CO];
        if (out_valid) {
#pragma unroll
          for (int g = 0; g < CO; g += 16) tc_ld16(tlane + slot * CO + g, *reinterpret_cast<uint32_t(*)[16]>(&acc[g]));
          tc_wait_ld();
        }
        zero_slot(slot);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(acc_free_bar(ln));
        if (out_valid && x < geo.W && geo.out_f32) {
          // head maps: pre-activation fp32 values, planar (a warp writes 32 consecutive pixels of one map)
          float* o = geo.out_f32 + ((size_t)run.b * geo.n_valid * geo.H + (row - d)) * geo.W + x;
#pragma unroll
          for (int c = 0; c < CO; ++c)
            if (c < geo.n_valid) {
              float v = __uint_as_float(acc[c]) + (STEM ? 0.0f : lc.bias[c]);
              if (relu) v = fmaxf(v, 0.0f);
              o[(size_t)c * plane_px] = v;
            }
        } else if (out_valid && x < geo.W) {
#pragma unroll
          for (int kk = 0; kk < CO / 8; ++kk) {
            uint32_t ow[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int c0 = kk * 8 + 2 * i;
              if (STEM) {
                // the bias came in through the MMA (three constant-one input channels), the ReLU
                // rides on the conversion: two instructions per channel pair less in the one loop
                // that sets the pace of this HBM-bound kernel
                const float v0 = __uint_as_float(acc[c0]), v1 = __uint_as_float(acc[c0 + 1]);
                ow[i] = relu ? pack2_relu<F16>(v0, v1) : pack2<F16>(v0, v1);
              } else {
                float v0 = __uint_as_float(acc[c0]) + lc.bias[c0];
                float v1 = __uint_as_float(acc[c0 + 1]) + lc.bias[c0 + 1];
                if (relu) {
                  v0 = fmaxf(v0, 0.0f);
                  v1 = fmaxf(v1, 0.0f);
                }
                ow[i] = pack2<F16>(v0, v1);
              }
            }
            orow[(size_t)kk * plane_px] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
          }
        }
        slot = slot == 2 ? 0u : slot + 1u;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (role == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
  }
}

int pick_chain_stages(int CI, int CO, int k, int d) {
  int nstage = kMaxStages;
  while (nstage >= 2 && chain_smem(CI, CO, k, k == 3 ? d : 0, nstage).total + 1024 > 227u * 1024u) --nstage;
  return nstage >= 2 ? nstage : 0;
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

template <int CO, bool F16, int KX, bool STEM>
cudaError_t launch_t(const ConvGen& a, CGeo geo, const void* wpack, const LayerConst& lc, int nstage, int grid,
                     size_t smem, const StemSrc& ss, cudaStream_t st) {
  static bool attr_done[kMaxDevices] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (!attr_done[dev]) {
    cudaError_t e = cudaFuncSetAttribute(conv_chain_kernel<CO, F16, KX, STEM>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_done[dev] = true;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(STEM ? kStemThreads : kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, conv_chain_kernel<CO, F16, KX, STEM>, (const uint8_t*)a.in, (uint8_t*)a.out, geo,
                            (const uint8_t*)wpack, nstage, lc, a.relu, ss);
}

}  // namespace

bool conv_chain_supports(int CI, int CO, int k, int d) {
  const bool shape = (k == 3 && (CO == 16 || CO == 32)) || (k == 1 && (CO == 16 || CO == 32 || CO == 48) && d == 1);
  return shape && CI % 16 == 0 && CI >= 16 && CI <= 256 && d >= 1 && d <= 16 && pick_chain_stages(CI, CO, k, d) > 0;
}

size_t conv_chain_packed_bytes(int CI, int CO, int k) { return (size_t)k * (CI / 8) * 5 * CO * 16; }

// w_oihw [CO_real][CI][k][k] fp32 -> shared-memory image: for kx, input chunk kc: 5 CO rows of
// 16 B (8 input channels), rows = output channels of ky = 1, 0, 2, 1, 0; rows >= CO_real zero.
// k = 1: one kx tap, the rows of ky = 0 and ky = 2 zero.
void conv_chain_pack_host(int CI, int CO, int CO_real, int k, const float* w, void* dst, bool f16) {
  static const int ky_seq[5] = {1, 0, 2, 1, 0};
  uint16_t* o = static_cast<uint16_t*>(dst);
  for (int kx = 0; kx < k; ++kx)
    for (int kc = 0; kc < CI / 8; ++kc)
      for (int n = 0; n < 5 * CO; ++n) {
        const int ky = ky_seq[n / CO], co = n % CO;
        for (int j = 0; j < 8; ++j) {
          const int ci = kc * 8 + j;
          float v = 0.0f;
          if (co < CO_real) {
            if (k == 3) v = w[(((size_t)co * CI + ci) * 3 + ky) * 3 + kx];
            else if (ky == 1) v = w[(size_t)co * CI + ci];
          }
          o[(((size_t)(kx * (CI / 8) + kc) * 5 * CO) + n) * 8 + j] = bits16(v, f16);
        }
      }
}

cudaError_t launch_conv_chain(bool f16, const ConvGen& a, const void* wpack, const LayerConst& lc, int n_sm,
                              cudaStream_t st) {
  if (!conv_chain_supports(a.CI, a.CO, a.k, a.d) || a.ci_plane0 != 0) return cudaErrorInvalidValue;
  if (a.B <= 0) return cudaSuccess;
  CGeo geo;
  geo.B = a.B;
  geo.H = a.H;
  geo.W = a.W;
  geo.d = a.d;
  geo.dx = a.k == 3 ? a.d : 0;
  geo.nseg = (a.W + kTileM - 1) / kTileM;
  geo.Lmax = (a.H + a.d - 1) / a.d;
  geo.total = (long long)a.B * geo.nseg * a.d * geo.Lmax;
  geo.CI = a.CI;
  geo.in_planes = a.in_planes;
  geo.out_planes = a.out_planes;
  geo.out_f32 = a.out_f32;
  geo.n_valid = a.n_valid;
  geo.co_plane0 = a.co_plane0;
  const int nstage = pick_chain_stages(a.CI, a.CO, a.k, a.d);
  const size_t smem = chain_smem(a.CI, a.CO, a.k, geo.dx, nstage).total + 1024;
  long long want = (geo.total + 23) / 24;
  const int grid = (int)(want < 1 ? 1 : (want > n_sm ? n_sm : want));
  static const StemSrc ss0{};
#define SMLM_CHAIN_CASE(CC, KK)                                                                     \
  if (a.CO == CC && a.k == KK)                                                                     \
    return f16 ? launch_t<CC, true, KK, false>(a, geo, wpack, lc, nstage, grid, smem, ss0, st)     \
               : launch_t<CC, false, KK, false>(a, geo, wpack, lc, nstage, grid, smem, ss0, st);
  SMLM_CHAIN_CASE(16, 3)
  SMLM_CHAIN_CASE(32, 3)
  SMLM_CHAIN_CASE(16, 1)
  SMLM_CHAIN_CASE(32, 1)
  SMLM_CHAIN_CASE(48, 1)
#undef SMLM_CHAIN_CASE
  return cudaErrorInvalidValue;
}

// ---------------------------------------------------------------------------- K1 on the tensor cores
bool stem_umma_supports(int C, int in_frames) {
  return in_frames == 1 && (C == 16 || C == 32 || C == 48 || C == 64) && pick_chain_stages(16, C, 3, 1) > 0;
}

size_t stem_umma_packed_bytes(int C) { return conv_chain_packed_bytes(16, C, 3); }

// w_stem [9][C] fp32 (tap ky * 3 + kx, channel) -> the chain kernel's image for C_in = 16: input
// channel j of chunk 0 carries the weight piece that pairs with the x piece of the same j
// (x_h w_h, x_h w_m, x_m w_h, x_h w_l, x_l w_h, x_m w_m); everything else zero.
void stem_umma_pack_host(int C, const float* w_stem, const float* b_stem, void* dst, bool f16) {
  static const int ky_seq[5] = {1, 0, 2, 1, 0};
  static const int wpiece[8] = {0, 1, 0, 2, 0, 1, -1, -1};  // h, m, h, l, h, m
  uint16_t* o = static_cast<uint16_t*>(dst);
  auto val16 = [&](uint16_t bits) {
    if (f16) return __half2float(__ushort_as_half(bits));
    uint32_t u = (uint32_t)bits << 16;
    float f;
    std::memcpy(&f, &u, 4);
    return f;
  };
  for (int kx = 0; kx < 3; ++kx)
    for (int kc = 0; kc < 2; ++kc)
      for (int n = 0; n < 5 * C; ++n) {
        const int ky = ky_seq[n / C], co = n % C;
        // chunk 0: the weight of the tap; chunk 1 (constant-one channels): the bias, at the centre tap only
        const float w = kc == 0 ? w_stem[(size_t)(ky * 3 + kx) * C + co] : ((ky == 1 && kx == 1) ? b_stem[co] : 0.0f);
        uint16_t piece[3];
        piece[0] = bits16(w, f16);
        const float r1 = w - val16(piece[0]);
        piece[1] = bits16(r1, f16);
        piece[2] = bits16(r1 - val16(piece[1]), f16);
        for (int j = 0; j < 8; ++j) {
          uint16_t v = 0;
          if (kc == 0 && wpiece[j] >= 0) v = piece[wpiece[j]];
          if (kc == 1 && j < 3) v = piece[j];
          o[(((size_t)(kx * 2 + kc) * 5 * C) + n) * 8 + j] = v;
        }
      }
}

cudaError_t launch_stem_umma(bool f16, const uint16_t* frames, int frame_base, ViewSet vs, ActShape s, NormParams np,
                             const void* wpack, const LayerConst& lc, int relu, void* act, int n_sm,
                             cudaStream_t st) {
  if (!stem_umma_supports(s.C, vs.in_frames <= 1 ? 1 : vs.in_frames)) return cudaErrorInvalidValue;
  if (s.B <= 0) return cudaSuccess;
  ConvGen a{};
  a.in = nullptr;
  a.out = act;
  a.CI = 16;
  a.CO = s.C;
  a.B = s.B;
  a.H = s.H;
  a.W = s.W;
  a.k = 3;
  a.d = 1;
  a.relu = relu;
  CGeo geo;
  geo.B = s.B;
  geo.H = s.H;
  geo.W = s.W;
  geo.d = 1;
  geo.dx = 1;
  geo.nseg = (s.W + kTileM - 1) / kTileM;
  geo.Lmax = s.H;
  geo.total = (long long)s.B * geo.nseg * geo.Lmax;
  geo.CI = 16;
  geo.in_planes = 0;
  geo.out_planes = (s.CT > 0 ? s.CT : s.C) / 8;
  geo.out_f32 = nullptr;
  geo.n_valid = 0;
  geo.co_plane0 = 0;
  StemSrc ss;
  ss.frames = frames;
  ss.frame_base = frame_base;
  ss.vs = vs;
  ss.np = np;
  const int nstage = pick_chain_stages(16, s.C, 3, 1);
  const size_t smem = chain_smem(16, s.C, 3, 1, nstage).total + 1024;
  long long want = (geo.total + 23) / 24;
  const int grid = (int)(want < 1 ? 1 : (want > n_sm ? n_sm : want));
#define SMLM_STEM_CASE(CC)                                                                       \
  if (s.C == CC)                                                                                 \
    return f16 ? launch_t<CC, true, 3, true>(a, geo, wpack, lc, nstage, grid, smem, ss, st)      \
               : launch_t<CC, false, 3, true>(a, geo, wpack, lc, nstage, grid, smem, ss, st);
  SMLM_STEM_CASE(16)
  SMLM_STEM_CASE(32)
  SMLM_STEM_CASE(48)
  SMLM_STEM_CASE(64)
#undef SMLM_STEM_CASE
  return cudaErrorInvalidValue;
}

}  // namespace smlm
