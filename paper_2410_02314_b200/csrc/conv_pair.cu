// K2 pair: two consecutive trunk layers with dilations (d, 2d) in ONE kernel, sm_100a
// (SURVEY.md 8(f)-1 "deeper fusion to remove activation round-trips").
//     mid = in  + ReLU(conv3x3 dil d  (in;  W_A) + b_A)
//     out = mid + ReLU(conv3x3 dil 2d (mid; W_B) + b_B)
// `mid` never reaches HBM: layer A's epilogue writes each finished row, rounded to the storage
// type exactly as conv_umma.cu stores it, into shared memory in tcgen05 operand layout, and
// layer B's MMAs consume it from there; it is also layer B's residual.  Per pixel the pair
// moves 2C bytes in and 2C bytes out instead of twice that, which takes the trunk off the HBM
// roof (profiles/).  Results are bit-identical to two conv_umma launches: same operands, same
// accumulation order per output, same rounding points.
//
// Both layers use the row-chain walk of conv_umma.cu (M = 128 pixels of one row, N = 3C: one
// MMA feeds three output rows held in three TMEM slots).  Chain of layer A: rows r, r+d, r+2d,
// ... (index i).  Its outputs alternate between the two chains of layer B (dilation 2d) that
// cover the same rows: B chain s = i & 1.  TMEM: 3 slots for A + 3 per B chain = 9C columns
// (432 at C = 48), so one pair pipeline per CTA; it still overlaps like the two lanes of
// conv_umma.cu because A's MMAs run under B's epilogue and vice versa, and the two B chains
// let B's MMA of row i+1 start before row i's epilogue has released its slot.
//
// The x halo of layer B (2d pixels of `mid` on each side of a 128-pixel segment) is NOT
// recomputed: the segments of a row sit on the CTAs of one thread-block cluster (cluster
// size = segments per row <= 8, CTA rank = segment), which walk the same rows in lock-step;
// A's epilogue stores its edge pixels into the neighbour CTA's stage through distributed
// shared memory, and the stage's full / empty mbarriers count the neighbours' arrivals
// (remote mbarrier.arrive, tcgen05.commit multicast).
//
// Warps: 0-7 epilogue of A, 8-15 epilogue of B (warp pair (q, q+4) = TMEM lane quadrant q,
// channel halves), 16 TMA producer, 17 MMA issuer of A, 18 MMA issuer of B (+ TMEM allocation).
#include <algorithm>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <type_traits>

#include "smlm_internal.cuh"
#include "umma_ptx.cuh"

namespace smlm {
namespace {

using namespace ptx;

constexpr int kThreads = 608;
constexpr int kEpiWarps = 8;  // per layer
constexpr int kTileM = 128;
constexpr int kMaxSt = 4;     // stages per ring
constexpr int kTmemCols = 512;
constexpr int kMaxDevices = 64;
constexpr int kMaxCluster = 8;  // portable cluster size
constexpr int kNumBars = 23 + 2 * kMaxSt;  // + the peer's stage-full relays (cta_group::2)

// zero source for the padded parts of an input row segment: at most (127 + 8) pixels x 16 B
__device__ __align__(16) uint4 g_pzeros[160];

struct PGeo {
  int B, H, W, d;   // d: dilation of layer A (layer B: 2d)
  int nseg;         // 128-pixel segments per row = cluster size
  int Lmax;         // chain rows per residue of layer A: ceil(H / d)
  long long total;  // B * d * Lmax rows (each spans the whole cluster)
};

// A cluster owns the contiguous range [g, g1) of rows (in chain order) and walks it as runs:
// n consecutive rows i0 .. i0+n-1 of one A chain (view b, residue r) are OUTPUT rows of the
// pair.  A run takes n + 6 steps of layer A (inputs i0-3 .. i0+n+2, giving mid rows i0-2 ..
// i0+n+1) and n + 4 steps of layer B.
struct PRun {
  int b, r, i0, n;
};
struct PRuns {
  long long g, g1;
  __device__ void init(const PGeo& geo, int cid, int ncl) {
    g = geo.total * cid / ncl;
    g1 = geo.total * (cid + 1) / ncl;
  }
  __device__ bool next(const PGeo& geo, PRun& run) {
    if (g >= g1) return false;
    const long long chain = g / geo.Lmax;
    run.i0 = (int)(g - chain * geo.Lmax);
    const long long rem = g1 - g;
    run.n = geo.Lmax - run.i0 < rem ? geo.Lmax - run.i0 : (int)rem;
    run.r = (int)(chain % geo.d);
    run.b = (int)(chain / geo.d);
    g += run.n;
    return true;
  }
};

struct PSmem {
  uint32_t wA_off, wB_off, w_bytes;   // per layer
  uint32_t stA_off, stA_bytes;        // input row segments of layer A (TMA)
  uint32_t stB_off, stB_bytes;        // `mid` row segments (written by A's epilogue)
  uint32_t xch_off;                   // HEAD: float [2][128 px][8]
  uint32_t scr_off;                   // HEAD: uint4 [C/16][256 threads]: the B epilogue's rounded outputs, parked
  uint32_t bar_off, tmem_off, total;
};

// cta_group::2: of every 5C-row weight plane a CTA holds the rows its half of the three N = 3C
// windows needs: rows [pr NH, pr NH + 2C + NH), NH = 3C/2, pr = rank in the pair
__host__ __device__ constexpr uint32_t pair_wrows(int C, bool cg2) { return cg2 ? 2u * C + 3u * C / 2u : 5u * C; }

__host__ __device__ inline PSmem pair_smem(int C, int d, int nA, int nB, bool head, bool cg2) {
  PSmem L;
  L.w_bytes = 3u * (C / 8) * pair_wrows(C, cg2) * 16u;
  L.wA_off = 0;
  L.wB_off = L.w_bytes;
  L.stA_bytes = (((uint32_t)(C / 8) * (kTileM + 2 * d) * 16u) + 127u) & ~127u;
  L.stB_bytes = (((uint32_t)(C / 8) * (kTileM + 4 * d) * 16u) + 127u) & ~127u;
  L.stA_off = (2u * L.w_bytes + 127u) & ~127u;
  L.stB_off = L.stA_off + (uint32_t)nA * L.stA_bytes;
  L.xch_off = L.stB_off + (uint32_t)nB * L.stB_bytes;
  L.scr_off = L.xch_off + (head ? 2u * kTileM * 8u * 4u : 0u);  // two step parities
  L.bar_off = L.scr_off + (head ? (uint32_t)(C / 16) * 256u * 16u : 0u);
  L.tmem_off = L.bar_off + 8u * kNumBars;
  L.total = L.tmem_off + 16u;
  return L;
}

// mbarrier wait with a watchdog: a protocol error traps (launch failure) instead of hanging
// the device.  ~10 s at 2 GHz; no legitimate wait inside one launch comes near it.
template <bool CLUSTER>
__device__ __forceinline__ void wait_bar(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  long long t0 = 0;
  for (;;) {
    if (CLUSTER)
      asm volatile(
          "{\n.reg .pred p;\nmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2, %3;\n"
          "selp.u32 %0, 1, 0, p;\n}\n"
          : "=r"(ok)
          : "r"(bar), "r"(parity), "r"(0x989680u)
          : "memory");
    else
      asm volatile(
          "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
          "selp.u32 %0, 1, 0, p;\n}\n"
          : "=r"(ok)
          : "r"(bar), "r"(parity), "r"(0x989680u)
          : "memory");
    if (ok) return;
    const long long t = clock64();
    if (t0 == 0) t0 = t;
    else if (t - t0 > 20000000000ll) __trap();
  }
}

// cta_group::2: one MMA over the CTA pair (ranks 2k, 2k+1 of the cluster = two adjacent
// segments): D[256 x N], A rows 0-127 / 128-255 and D from the leader's / the peer's shared
// memory and TMEM at the same addresses, B's N columns split between the two CTAs.
__device__ __forceinline__ void tc_mma2(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, 1, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc)
      : "memory");
}
__device__ __forceinline__ void tc_commit2_mc(uint32_t bar, uint16_t mask) {
  asm volatile(
      "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
      "h"(mask)
      : "memory");
}
template <int C, bool HEAD, bool F16, bool CG2>
__global__ void __launch_bounds__(kThreads, 1)
    conv_pair_kernel(const __nv_bfloat16* __restrict__ in, __nv_bfloat16* __restrict__ out, PGeo geo,
                     const uint8_t* __restrict__ wpackA, const uint8_t* __restrict__ wpackB, int nA, int nB,
                     const __grid_constant__ LayerConst lcA, const __grid_constant__ LayerConst lcB,
                     const __grid_constant__ HeadArgs ha) {
  extern __shared__ uint8_t smem_raw[];
  const int d = geo.d, dB = 2 * geo.d;
  const PSmem L = pair_smem(C, d, nA, nB, HEAD, CG2);
  const uint32_t sraw = smem_u32(smem_raw);
  const uint32_t sbase = (sraw + 1023u) & ~1023u;  // the launch reserves 1 KB of slack for this
  uint8_t* smem = smem_raw + (sbase - sraw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = (int)cluster_ctarank();  // = segment of the row
  const int nseg = geo.nseg;
  const bool has_left = rank > 0, has_right = rank + 1 < nseg;
  const int nnb = 1 + (has_left ? 1 : 0) + (has_right ? 1 : 0);
  const int cid = blockIdx.x / nseg, ncl = gridDim.x / nseg;
  const int x0 = rank * kTileM;
  // cta_group::2: the even rank of a pair issues the MMAs of both CTAs
  const int pr = rank & 1;
  const bool leader = !CG2 || pr == 0;
  const uint32_t leader_rank = (uint32_t)(rank & ~1);

  auto bar = [&](int i) { return sbase + L.bar_off + 8u * (uint32_t)i; };
  const uint32_t wbar = bar(0);
  auto fullA = [&](int s) { return bar(1 + s); };
  auto emptyA = [&](int s) { return bar(1 + kMaxSt + s); };
  auto fullB = [&](int s) { return bar(1 + 2 * kMaxSt + s); };
  auto emptyB = [&](int s) { return bar(1 + 3 * kMaxSt + s); };
  const uint32_t accA_full = bar(1 + 4 * kMaxSt), accA_free = bar(2 + 4 * kMaxSt);
  auto accB_full = [&](int s) { return bar(3 + 4 * kMaxSt + s); };
  auto accB_free = [&](int s) { return bar(5 + 4 * kMaxSt + s); };
  auto fullAp = [&](int s) { return bar(7 + 4 * kMaxSt + s); };  // leader: the peer's input stage s is full
  auto fullBp = [&](int s) { return bar(7 + 5 * kMaxSt + s); };  // leader: the peer's mid stage s is full
  // B's MMA commits arrive once per CTA (cta_group::1) or once per pair (cta_group::2) that
  // touches this CTA's neighbourhood {rank-1, rank, rank+1}
  const int ncommit = CG2 ? 1 + ((pr == 0 ? has_left : has_right) ? 1 : 0) : nnb;
  auto stA = [&](int s) { return sbase + L.stA_off + (uint32_t)s * L.stA_bytes; };
  auto stB = [&](int s) { return sbase + L.stB_off + (uint32_t)s * L.stB_bytes; };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + L.tmem_off);

  const uint32_t planeA = (uint32_t)(kTileM + 2 * d) * 16u;   // bytes between channel chunks
  const uint32_t planeB = (uint32_t)(kTileM + 2 * dB) * 16u;

  // ---- one-time setup
  if (threadIdx.x == 0) {
    mbar_init(wbar, 1);
    for (int s = 0; s < kMaxSt; ++s) {
      mbar_init(fullA(s), 1);                 // the TMA transaction count
      mbar_init(emptyA(s), 1 + kEpiWarps);    // MMA commit + A's epilogue warps (residual copied out)
      // mid stage: written by this CTA's 8 A-epilogue warps (arrivals) and by the edge threads
      // of each neighbour (st.async: transaction bytes); read by the B MMAs and B epilogue
      // warps of this CTA - and the stages of the neighbours, which this CTA also writes,
      // must be free too
      mbar_init(fullB(s), kEpiWarps);
      mbar_init(emptyB(s), ncommit + kEpiWarps * nnb);
      mbar_init(fullAp(s), 1);
      mbar_init(fullBp(s), 1);
    }
    mbar_init(accA_full, 1);
    mbar_init(accA_free, CG2 ? 2 * kEpiWarps : kEpiWarps);  // cta_group::2: both CTAs' epilogues, on the leader
    for (int s = 0; s < 2; ++s) {
      mbar_init(accB_full(s), 1);
      mbar_init(accB_free(s), CG2 ? 2 * kEpiWarps : kEpiWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 18) {
    if (CG2) {  // the same warp of both CTAs, the same destination offset
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + L.tmem_off),
                   "n"(kTmemCols)
                   : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + L.tmem_off),
                   "n"(kTmemCols)
                   : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  // the mid stages start as zeros: positions outside the frame (left of segment 0, right of the
  // last segment) are never written and ARE the zero padding of layer B
  {
    uint4* zb = reinterpret_cast<uint4*>(smem + L.stB_off);
    const uint32_t nz = (uint32_t)nB * L.stB_bytes / 16u;
    for (uint32_t i = threadIdx.x; i < nz; i += kThreads) zb[i] = make_uint4(0u, 0u, 0u, 0u);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  cluster_sync_all();  // every CTA's barriers and stages exist before any remote access
  const uint32_t tmem_base = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == 16) {
    // =========================== TMA producer (layer A's input rows, both layers' weights)
    if (elect_one()) {
      mbar_expect_tx(wbar, 2u * L.w_bytes);
      if (CG2) {  // per (kx, input chunk) plane: the rows of this CTA's halves of the three windows
        const uint32_t prow = pair_wrows(C, true) * 16u, skip = (uint32_t)pr * (3u * C / 2u) * 16u;
        for (uint32_t pl = 0; pl < 3u * (C / 8); ++pl) {
          bulk_load(sbase + L.wA_off + pl * prow, wpackA + pl * (5u * C * 16u) + skip, prow, wbar);
          bulk_load(sbase + L.wB_off + pl * prow, wpackB + pl * (5u * C * 16u) + skip, prow, wbar);
        }
      } else {
        for (uint32_t off = 0; off < L.w_bytes; off += 16384u) {
          const uint32_t n = L.w_bytes - off < 16384u ? L.w_bytes - off : 16384u;
          bulk_load(sbase + L.wA_off + off, wpackA + off, n, wbar);
          bulk_load(sbase + L.wB_off + off, wpackB + off, n, wbar);
        }
      }
    }
    __syncwarp();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t plane_bytes = (size_t)geo.H * geo.W * 16u;
    const size_t row_step = (size_t)d * geo.W * 16u;
    const uint8_t* in_b = reinterpret_cast<const uint8_t*>(in);
    const int xl = x0 - d, xr = x0 + kTileM + d;
    const int lo = xl > 0 ? xl : 0, hi = xr < geo.W ? xr : geo.W;
    const uint32_t pre = (uint32_t)(lo - xl) * 16u, mid = (uint32_t)(hi - lo) * 16u,
                   post = (uint32_t)(xr - hi) * 16u;
    int fills_left = (pre | post) ? nA : 0;  // zero padding: once per stage, it stays
    PRuns runs;
    runs.init(geo, cid, ncl);
    PRun run;
    uint32_t st = 0, par = 1;
    while (runs.next(geo, run)) {
      int row = run.r + (run.i0 - 3) * d;
      const uint8_t* src = in_b + ((long long)run.b * (C / 8) * geo.H * geo.W + (long long)row * geo.W + lo) * 16;
      for (int t = 0; t < run.n + 6; ++t, row += d, src += row_step) {
        if (row < 0 || row >= geo.H) continue;
        const uint32_t dst = stA((int)st);
        const uint32_t fb = fullA((int)st);
        const bool fill = fills_left > 0;
        wait_bar<false>(emptyA((int)st), par);
        if (elect_one()) {
          mbar_expect_tx(fb, (uint32_t)(C / 8) * (fill ? planeA : mid));
#pragma unroll
          for (int k = 0; k < C / 8; ++k)
            bulk_load(dst + (uint32_t)k * planeA + pre, src + (size_t)k * plane_bytes, mid, fb);
          if (fill) {
#pragma unroll
            for (int k = 0; k < C / 8; ++k) {
              if (pre) bulk_load(dst + (uint32_t)k * planeA, g_pzeros, pre, fb);
              if (post) bulk_load(dst + (uint32_t)k * planeA + pre + mid, g_pzeros, post, fb);
            }
          }
        }
        __syncwarp();
        fills_left -= fill ? 1 : 0;
        if (++st == (uint32_t)nA) {
          st = 0;
          par ^= 1u;
        }
      }
    }
  } else if (warp == 17) {
    // =========================== MMA issuer of layer A
    asm volatile("griddepcontrol.wait;" ::: "memory");
    wait_bar<false>(wbar, 0);
    constexpr uint32_t idesc = umma_idesc(CG2 ? 2 * kTileM : kTileM, 3 * C, F16);
    const uint32_t plane16 = planeA >> 4;
    constexpr uint32_t wplane16 = pair_wrows(C, CG2);
    const uint16_t pair_mask = (uint16_t)(3u << leader_rank);
    const uint32_t relayA = CG2 && !leader ? mapa(fullAp(0), leader_rank) : 0u;
    constexpr uint32_t desc_hi = (128u >> 4) | (1u << 14);
    const uint32_t a_lo_base = (plane16 << 16) | (((sbase + L.stA_off) >> 4) & 0x3FFFu);
    const uint32_t b_lo_base = (wplane16 << 16) | (((sbase + L.wA_off) >> 4) & 0x3FFFu);
    const uint32_t stage16 = L.stA_bytes >> 4;
    const uint32_t dcol = __shfl_sync(0xffffffffu, tmem_base, 0);
    PRuns runs;
    runs.init(geo, cid, ncl);
    PRun run;
    uint32_t st = 0, full_par = 0, free_par = 0, m = 0;
    while (runs.next(geo, run)) {
      int row = run.r + (run.i0 - 3) * d;
      for (int t = 0; t < run.n + 6; ++t, row += d) {
        const bool in_valid = row >= 0 && row < geo.H;
        if (in_valid) wait_bar<false>(fullA((int)st), full_par);
        if (CG2 && !leader) {
          // the peer of a pair issues nothing: it tells the leader that its stage has landed
          if (in_valid && elect_one()) mbar_arrive_cluster(relayA + 8u * st);
          __syncwarp();
          if (in_valid && ++st == (uint32_t)nA) {
            st = 0;
            full_par ^= 1u;
          }
          continue;
        }
        if (CG2 && in_valid) wait_bar<false>(fullAp((int)st), full_par);
        wait_bar<false>(accA_free, free_par);
        free_par ^= 1u;
        tc_fence_after();
        const uint32_t win = m == 0 ? 0u : (m == 1 ? 2u : 1u);
        const uint32_t a_lo = a_lo_base + st * stage16;
        const uint32_t b_lo = b_lo_base + win * C;
        if (elect_one()) {
          if (in_valid) {
#pragma unroll
            for (int kx = 0; kx < 3; ++kx) {
#pragma unroll
              for (int ks = 0; ks < C / 16; ++ks) {
                const uint32_t al = a_lo + (uint32_t)(2 * ks) * plane16 + (uint32_t)(kx * d);
                const uint32_t bl = b_lo + (uint32_t)(kx * (C / 8) + 2 * ks) * wplane16;
                if (CG2) tc_mma2(dcol, ((uint64_t)desc_hi << 32) | al, ((uint64_t)desc_hi << 32) | bl, idesc);
                else tc_mma(dcol, ((uint64_t)desc_hi << 32) | al, ((uint64_t)desc_hi << 32) | bl, idesc, 1u);
              }
            }
            if (CG2) tc_commit2_mc(emptyA((int)st), pair_mask);
            else tc_commit(emptyA((int)st));
          }
          if (CG2) tc_commit2_mc(accA_full, pair_mask);
          else tc_commit(accA_full);
        }
        __syncwarp();
        if (in_valid && ++st == (uint32_t)nA) {
          st = 0;
          full_par ^= 1u;
        }
        m = m == 2 ? 0u : m + 1u;
      }
    }
  } else if (warp == 18) {
    // =========================== MMA issuer of layer B (two interleaved chains)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    wait_bar<false>(wbar, 0);
    constexpr uint32_t idesc = umma_idesc(CG2 ? 2 * kTileM : kTileM, 3 * C, F16);
    const uint32_t plane16 = planeB >> 4;
    constexpr uint32_t wplane16 = pair_wrows(C, CG2);
    const uint16_t pair_mask = (uint16_t)(3u << leader_rank);
    const uint32_t relayB = CG2 && !leader ? mapa(fullBp(0), leader_rank) : 0u;
    constexpr uint32_t desc_hi = (128u >> 4) | (1u << 14);
    const uint32_t a_lo_base = (plane16 << 16) | (((sbase + L.stB_off) >> 4) & 0x3FFFu);
    const uint32_t b_lo_base = (wplane16 << 16) | (((sbase + L.wB_off) >> 4) & 0x3FFFu);
    const uint32_t stage16 = L.stB_bytes >> 4;
    const uint32_t dcol0 = __shfl_sync(0xffffffffu, tmem_base, 0) + 3u * C;
    // who hears that this CTA's (cta_group::2: this pair's) MMAs are done with a mid stage: the
    // CTAs that write into it
    const uint16_t mask = CG2 ? (uint16_t)((3u << leader_rank) | (leader_rank > 0 ? 1u << (leader_rank - 1) : 0u) |
                                           ((int)leader_rank + 2 < nseg ? 1u << (leader_rank + 2) : 0u))
                              : (uint16_t)((1u << rank) | (has_left ? 1u << (rank - 1) : 0u) |
                                           (has_right ? 1u << (rank + 1) : 0u));
    PRuns runs;
    runs.init(geo, cid, ncl);
    PRun run;
    uint32_t st = 0, full_par = 0;
    uint32_t free_par0 = 0, free_par1 = 0, m0 = 0, m1 = 0;
    while (runs.next(geo, run)) {
      int row = run.r + (run.i0 - 2) * d;
      for (int u = 0; u < run.n + 4; ++u, row += d) {
        const int s = u & 1;
        const bool in_valid = row >= 0 && row < geo.H;
        if (in_valid) {
          wait_bar<true>(fullB((int)st), full_par);
          // the neighbours' st.async data, observed through the barrier, before the MMAs read it
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        if (CG2 && !leader) {
          if (in_valid && elect_one()) mbar_arrive_cluster(relayB + 8u * st);
          __syncwarp();
          if (in_valid && ++st == (uint32_t)nB) {
            st = 0;
            full_par ^= 1u;
          }
          continue;
        }
        if (CG2 && in_valid) wait_bar<false>(fullBp((int)st), full_par);
        wait_bar<false>(accB_free(s), s ? free_par1 : free_par0);
        if (s) free_par1 ^= 1u;
        else free_par0 ^= 1u;
        tc_fence_after();
        const uint32_t m = s ? m1 : m0;
        const uint32_t win = m == 0 ? 0u : (m == 1 ? 2u : 1u);
        const uint32_t a_lo = a_lo_base + st * stage16;
        const uint32_t b_lo = b_lo_base + win * C;
        const uint32_t dcol = dcol0 + (uint32_t)s * 3u * C;
        if (elect_one()) {
          if (in_valid) {
#pragma unroll
            for (int kx = 0; kx < 3; ++kx) {
#pragma unroll
              for (int ks = 0; ks < C / 16; ++ks) {
                const uint32_t al = a_lo + (uint32_t)(2 * ks) * plane16 + (uint32_t)(kx * dB);
                const uint32_t bl = b_lo + (uint32_t)(kx * (C / 8) + 2 * ks) * wplane16;
                if (CG2) tc_mma2(dcol, ((uint64_t)desc_hi << 32) | al, ((uint64_t)desc_hi << 32) | bl, idesc);
                else tc_mma(dcol, ((uint64_t)desc_hi << 32) | al, ((uint64_t)desc_hi << 32) | bl, idesc, 1u);
              }
            }
            if (CG2) tc_commit2_mc(emptyB((int)st), mask);
            else if (nnb > 1) tc_commit_mc(emptyB((int)st), mask);
            else tc_commit(emptyB((int)st));
          }
          if (CG2) tc_commit2_mc(accB_full(s), pair_mask);
          else tc_commit(accB_full(s));
        }
        __syncwarp();
        if (in_valid && ++st == (uint32_t)nB) {
          st = 0;
          full_par ^= 1u;
        }
        if (s) m1 = m1 == 2 ? 0u : m1 + 1u;
        else m0 = m0 == 2 ? 0u : m0 + 1u;
      }
    }
  } else {
    // =========================== epilogues
    const bool isB = warp >= kEpiWarps;
    const int qd = warp & 3;            // TMEM lane quadrant this warp may access
    const int half = (warp >> 2) & 1;   // channel half
    constexpr int CH = C / 2;           // channels per thread
    constexpr int KH = C / 16;          // 8-channel chunks per thread
    const int k0 = half * KH;
    const int px = qd * 32 + lane;
    const int x = x0 + px;
    const uint32_t tlane = tmem_base + ((uint32_t)(qd * 32) << 16) + (uint32_t)(half * CH);
    auto ld_cols = [&](uint32_t col, uint32_t (&acc)[CH]) {
#pragma unroll
      for (int g = 0; g + 16 <= CH; g += 16) tc_ld16(tlane + col + g, *reinterpret_cast<uint32_t(*)[16]>(&acc[g]));
      if (CH % 16) tc_ld8(tlane + col + (CH - 8), *reinterpret_cast<uint32_t(*)[8]>(&acc[CH - 8]));
    };
    auto zero_cols = [&](uint32_t col) {
      const uint32_t z16[16] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
      const uint32_t z8[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
#pragma unroll
      for (int g = 0; g + 16 <= CH; g += 16) tc_st16(tlane + col + g, z16);
      if (CH % 16) tc_st8(tlane + col + (CH - 8), z8);
    };

    if (!isB) {
      // ----------------------- epilogue of layer A: TMEM -> mid row in shared memory
      for (int sl = 0; sl < 3; ++sl) zero_cols((uint32_t)(sl * C));
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      // cta_group::2: the accumulator-free signals of both CTAs go to the leader, who issues
      const uint32_t accA_free_t = CG2 && !leader ? mapa(accA_free, leader_rank) : accA_free;
      auto arrive_accA_free = [&]() {
        if (CG2 && !leader) mbar_arrive_cluster(accA_free_t);
        else mbar_arrive(accA_free);
      };
      if (lane == 0) arrive_accA_free();
      // where this thread's pixel goes: own stage at dB + px; the first / last dB pixels of the
      // segment are also the right / left halo of the left / right neighbour's stage
      const bool to_left = has_left && px < dB, to_right = has_right && px >= kTileM - dB;
      const uint32_t own_off = (uint32_t)(dB + px) * 16u;
      const uint32_t rem_off = to_left ? (uint32_t)(dB + kTileM + px) * 16u : (uint32_t)(px - (kTileM - dB)) * 16u;
      const uint32_t rem_rank = to_left ? (uint32_t)(rank - 1) : (uint32_t)(rank + 1);
      const uint32_t rem_base = (to_left || to_right) ? mapa(sbase + L.stB_off, rem_rank) : 0u;
      const uint32_t rem_bar0 = (to_left || to_right) ? mapa(fullB(0), rem_rank) : 0u;
      // bytes the neighbours send into one stage of this CTA: dB pixels x C channels each
      const uint32_t halo_tx = (uint32_t)(nnb - 1) * (uint32_t)dB * (uint32_t)C * 2u;
      PRuns runs;
      runs.init(geo, cid, ncl);
      PRun run;
      uint32_t slot = 2, acc_par = 0, st = 0, bst = 0, bpar = 1;
      uint4 res[KH];
#pragma unroll
      for (int k = 0; k < KH; ++k) res[k] = make_uint4(0u, 0u, 0u, 0u);
      while (runs.next(geo, run)) {
        int row = run.r + (run.i0 - 3) * d;  // input row of the step; the finished mid row is row - d
        for (int t = 0; t < run.n + 6; ++t, row += d) {
          const bool in_valid = row >= 0 && row < geo.H;
          const bool mid_valid = t >= 2 && row - d >= 0 && row - d < geo.H;
          wait_bar<false>(accA_full, acc_par);
          acc_par ^= 1u;
          tc_fence_after();
          uint32_t acc[CH];
          if (mid_valid) {
            ld_cols(slot * C, acc);
            tc_wait_ld();
          }
          zero_cols(slot * C);
          tc_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) arrive_accA_free();
          // the residual of the mid row that the NEXT step finishes is this step's input row:
          // copy its centre pixels out now (conv_umma.cu, kEarly policy); the stage goes back
          // to the producer together with the mid stage's arrival below
          uint4 res_next[KH];
          if (in_valid) {
            const uint4* rp = reinterpret_cast<const uint4*>(smem + (stA((int)st) - sbase) + (uint32_t)(d + px) * 16u);
#pragma unroll
            for (int kk = 0; kk < KH; ++kk) res_next[kk] = rp[(size_t)(k0 + kk) * (planeA / 16u)];
          }
          if (mid_valid) {
            wait_bar<false>(emptyB((int)bst), bpar);  // this stage is free here and in the neighbours
            uint8_t* own = smem + (stB((int)bst) - sbase) + own_off;
            const uint32_t rem = rem_base + bst * L.stB_bytes + rem_off;
            const uint32_t rem_bar = rem_bar0 + 8u * bst;
            const uint32_t keep = x < geo.W ? 0xffffffffu : 0u;  // beyond the row: B's zero padding
            auto post = [&](auto HALF) {
              constexpr int kHalf = decltype(HALF)::value;
#pragma unroll
              for (int kk = 0; kk < KH; ++kk) {
                constexpr int kc0 = kHalf * KH;
                const uint32_t rw[4] = {res[kk].x, res[kk].y, res[kk].z, res[kk].w};
                uint32_t ow[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  const int c0 = (kc0 + kk) * 8 + 2 * i;
                  float r0, r1;
                  unpack2<F16>(rw[i], r0, r1);
                  const float v0 = r0 + fmaxf(__uint_as_float(acc[kk * 8 + 2 * i]) + lcA.bias[c0], 0.0f);
                  const float v1 = r1 + fmaxf(__uint_as_float(acc[kk * 8 + 2 * i + 1]) + lcA.bias[c0 + 1], 0.0f);
                  ow[i] = pack2<F16>(v0, v1) & keep;
                }
                const uint4 o = make_uint4(ow[0], ow[1], ow[2], ow[3]);
                *reinterpret_cast<uint4*>(own + (size_t)(kc0 + kk) * planeB) = o;
                if (to_left || to_right) st_async_v4(rem + (uint32_t)(kc0 + kk) * planeB, o, rem_bar);
              }
            };
            if (half == 0) post(std::integral_constant<int, 0>{});
            else post(std::integral_constant<int, 1>{});
          }
          if (mid_valid || in_valid) {
            // one fence for both hand-overs: the local generic-proxy stores before the tensor
            // core's async-proxy reads of the mid stage (the halo pixels from the neighbours
            // arrive as transaction bytes of the same barrier phase), and the residual loads
            // before the TMA refill of the input stage
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
              if (mid_valid) {
                if (warp == 0 && halo_tx) mbar_expect_tx(fullB((int)bst), halo_tx);
                else mbar_arrive(fullB((int)bst));
              }
              if (in_valid) mbar_arrive(emptyA((int)st));
            }
          }
          if (mid_valid && ++bst == (uint32_t)nB) {
            bst = 0;
            bpar ^= 1u;
          }
          if (in_valid) {
#pragma unroll
            for (int kk = 0; kk < KH; ++kk) res[kk] = res_next[kk];
            if (++st == (uint32_t)nA) st = 0;
          }
          slot = slot == 2 ? 0u : slot + 1u;
        }
      }
    } else {
      // ----------------------- epilogue of layer B: TMEM + mid residual -> out (or HEAD)
      for (int sl = 0; sl < 6; ++sl) zero_cols((uint32_t)(3 * C + sl * C));
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      const uint32_t accB_free_t0 = CG2 && !leader ? mapa(accB_free(0), leader_rank) : accB_free(0);
      auto arrive_accB_free = [&](int c) {
        if (CG2 && !leader) mbar_arrive_cluster(accB_free_t0 + 8u * (uint32_t)c);
        else mbar_arrive(accB_free(c));
      };
      if (lane == 0) {
        arrive_accB_free(0);
        arrive_accB_free(1);
      }
      asm volatile("griddepcontrol.wait;" ::: "memory");
      const size_t plane_px = (size_t)geo.H * geo.W;
      float* xch = reinterpret_cast<float*>(smem + L.xch_off) + (size_t)px * 8;
      const int pair_bar = 1 + qd;
      const uint32_t eb_left = has_left ? mapa(emptyB(0), (uint32_t)(rank - 1)) : 0u;
      const uint32_t eb_right = has_right ? mapa(emptyB(0), (uint32_t)(rank + 1)) : 0u;
      PRuns runs;
      runs.init(geo, cid, ncl);
      PRun run;
      uint32_t slot0 = 2, slot1 = 2, par0 = 0, par1 = 0, bst = 0, xpar = 0;
      uint4 res_old[KH], res_mid[KH];
#pragma unroll
      for (int k = 0; k < KH; ++k) res_old[k] = res_mid[k] = make_uint4(0u, 0u, 0u, 0u);
      while (runs.next(geo, run)) {
        int row = run.r + (run.i0 - 2) * d;  // mid row of the step; the finished output row is row - dB
        uint4* orow = reinterpret_cast<uint4*>(out) +
                      (((long long)run.b * (C / 8) + k0) * geo.H * geo.W + (long long)(row - dB) * geo.W + x);
        for (int u = 0; u < run.n + 4; ++u, row += d, orow += (size_t)d * geo.W) {
          const int s = u & 1;
          const bool in_valid = row >= 0 && row < geo.H;
          const bool out_valid = u >= 4 && row - dB < geo.H;
          const bool store = out_valid && x < geo.W;
          wait_bar<false>(accB_full(s), s ? par1 : par0);
          if (s) par1 ^= 1u;
          else par0 ^= 1u;
          tc_fence_after();
          const uint32_t col = (uint32_t)(3 * C) + (uint32_t)s * 3u * C + (s ? slot1 : slot0) * C;
          uint32_t acc[CH];
          if (out_valid) {
            ld_cols(col, acc);
            tc_wait_ld();
          }
          zero_cols(col);
          tc_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) arrive_accB_free(s);
          // HEAD (last pair of the trunk): the epilogue evaluates the detection logit of every pixel
          // - the sum of two fmaf chains, one per channel half, the same chains as head_post.cu,
          // exchanged between the warp pair through shared memory - and stores the activations
          // only where the logit exceeds the threshold: K3 (post_logits_act_kernel) evaluates the
          // other heads there, for the survivors of the 3x3 test.  (All six heads in this
          // epilogue cost 6 x 48 FMAs per pixel and made the HEAD launch 17-29 % slower than a
          // plain one: profiles/conv_pair_r2.md.)
          // The rounded outputs wait for the verdict in shared memory, not in registers: twelve
          // more live registers made the compiler rematerialise addresses inside this loop and
          // the HEAD launch 17 % slower than without the store (profiles/conv_pair_r2.md).
          float hp0 = 0.0f;
          uint4* scr = reinterpret_cast<uint4*>(smem + L.scr_off) + ((warp - kEpiWarps) * 32 + lane);
          auto post = [&](auto HALF) {
            constexpr int kHalf = decltype(HALF)::value;
            if (HEAD && kHalf == 0) hp0 = ha.b[0];
#pragma unroll
            for (int kk = 0; kk < KH; ++kk) {
              constexpr int kc0 = kHalf * KH;
              const uint32_t rw[4] = {res_old[kk].x, res_old[kk].y, res_old[kk].z, res_old[kk].w};
              uint32_t ow[4];
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const int c0 = (kc0 + kk) * 8 + 2 * i;
                float r0, r1;
                unpack2<F16>(rw[i], r0, r1);
                const float v0 = r0 + fmaxf(__uint_as_float(acc[kk * 8 + 2 * i]) + lcB.bias[c0], 0.0f);
                const float v1 = r1 + fmaxf(__uint_as_float(acc[kk * 8 + 2 * i + 1]) + lcB.bias[c0 + 1], 0.0f);
                ow[i] = pack2<F16>(v0, v1);
                if (HEAD) {
                  float a0, a1;
                  unpack2<F16>(ow[i], a0, a1);
                  hp0 = fmaf(a0, ha.w[c0][0], hp0);
                  hp0 = fmaf(a1, ha.w[c0 + 1][0], hp0);
                }
              }
              if (!HEAD) orow[(size_t)kk * plane_px] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
              else scr[kk * 256] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
            }
          };
          if (store) {
            if (half == 0) post(std::integral_constant<int, 0>{});
            else post(std::integral_constant<int, 1>{});
          }
          // residual bookkeeping: the output finished by the next step (other chain) has its
          // centre in the previous step's mid row, the one after that in this step's
#pragma unroll
          for (int kk = 0; kk < KH; ++kk) res_old[kk] = res_mid[kk];
          if (in_valid) {
            const uint4* rp = reinterpret_cast<const uint4*>(smem + (stB((int)bst) - sbase) + (uint32_t)(dB + px) * 16u);
#pragma unroll
            for (int kk = 0; kk < KH; ++kk) res_mid[kk] = rp[(size_t)(k0 + kk) * (planeB / 16u)];
            // the next writers of this stage are the stores of this CTA's and the neighbours' A
            // epilogues, ordered behind these loads by the barrier; the fence keeps the arrive
            // from being issued while the loads are still in flight (conv_umma.cu, kEarly)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
              mbar_arrive(emptyB((int)bst));
              if (has_left) mbar_arrive_cluster(eb_left + 8u * bst);
              if (has_right) mbar_arrive_cluster(eb_right + 8u * bst);
            }
            if (++bst == (uint32_t)nB) bst = 0;
          }
          // (the mid stage is released above, BEFORE the exchange: the barrier below must not delay it)
          if (HEAD && out_valid) {
            float* xb = xch + (xpar ? kTileM * 8 : 0);  // double-buffered by step: a warp may run one barrier ahead
            xpar ^= 1u;
            xb[half] = hp0;
            asm volatile("bar.sync %0, 64;" ::"r"(pair_bar) : "memory");
            const float lg = xb[0] + xb[1];  // (half 0's chain) + (half 1's chain), the same bits in both warps
            if (store) {
              if (half == 0) ha.logit[((size_t)run.b * geo.H + (row - dB)) * geo.W + x] = lg;
              if (lg > ha.lthr) {
#pragma unroll
                for (int kk = 0; kk < KH; ++kk) orow[(size_t)kk * plane_px] = scr[kk * 256];
              }
            }
          }
          if (s) slot1 = slot1 == 2 ? 0u : slot1 + 1u;
          else slot0 = slot0 == 2 ? 0u : slot0 + 1u;
        }
      }
    }
  }

  // ---- teardown: no CTA may leave while a neighbour can still write into it
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 18) {
    tc_fence_after();
    if (CG2)
      asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
    else
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
  }
}

// stages: mid needs 3 (being written / read by the MMAs / waiting for its residual copy); the
// rest of the shared memory goes to the input ring, then to mid
bool pick_pair_stages(int C, int d, bool head, bool cg2, int* nA, int* nB) {
  const uint32_t budget = 227u * 1024u - 1024u;
  static const int pref[][2] = {{4, 4}, {4, 3}, {3, 3}, {3, 2}, {2, 2}};
  for (const auto& p : pref) {
    if (pair_smem(C, d, p[0], p[1], head, cg2).total <= budget) {
      *nA = p[0];
      *nB = p[1];
      return true;
    }
  }
  return false;
}

// cta_group::2 (one M = 256 MMA per CTA pair, B operand split between the two CTAs) needs an
// even number of segments per row.  Measured (profiles/conv_pair_r2.md): the shared-memory
// pipe drops from 95 % to 66 % busy, but layer A's serial loop MMA -> epilogue reads its TMEM
// slot -> next MMA now crosses the SM pair twice per step (multicast commit out, remote
// mbarrier arrive back), so at full clocks the kernel is ~7 % SLOWER than cta_group::1; in the
// sustained, power-capped step it is ~1.6 % FASTER (fewer operand bytes per FLOP).  The
// sustained step is what counts: on by default, SMLM_FUSE_PAIRS_1CTA selects cta_group::1.
bool pair_uses_cg2(int nseg, bool allow) { return allow && nseg % 2 == 0; }

template <int C, bool HEAD, bool F16, bool CG2>
cudaError_t launch_pair_t(const void* in, void* out, PGeo geo, const void* wA, const void* wB, const LayerConst& lcA,
                          const LayerConst& lcB, int nA, int nB, size_t smem, const HeadArgs& ha, int n_sm,
                          cudaStream_t st) {
  static bool attr_done[kMaxDevices] = {};
  static int max_clusters[kMaxDevices][kMaxCluster + 1] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  auto kern = conv_pair_kernel<C, HEAD, F16, CG2>;
  if (!attr_done[dev]) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_done[dev] = true;
  }
  cudaLaunchConfig_t cfg{};
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)geo.nseg;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  if (max_clusters[dev][geo.nseg] == 0) {
    // how many clusters of this size are co-resident (GPC boundaries cost some SMs)
    cfg.gridDim = dim3((unsigned)(n_sm / geo.nseg * geo.nseg));
    int n = 0;
    cudaError_t e = cudaOccupancyMaxActiveClusters(&n, kern, &cfg);
    if (e != cudaSuccess) return e;
    if (n < 1) return cudaErrorInvalidConfiguration;
    max_clusters[dev][geo.nseg] = n;
  }
  // at least ~12 rows per cluster, at most one wave of clusters
  long long want = (geo.total + 11) / 12;
  const int cap = max_clusters[dev][geo.nseg];
  const int ncl = (int)(want < 1 ? 1 : (want > cap ? cap : want));
  cfg.gridDim = dim3((unsigned)(ncl * geo.nseg));
  return cudaLaunchKernelEx(&cfg, kern, (const __nv_bfloat16*)in, (__nv_bfloat16*)out, geo, (const uint8_t*)wA,
                            (const uint8_t*)wB, nA, nB, lcA, lcB, ha);
}

template <int C, bool CG2>
cudaError_t launch_pair_c(bool f16, const void* in, void* out, PGeo geo, const void* wA, const void* wB,
                          const LayerConst& lcA, const LayerConst& lcB, int nA, int nB, size_t smem, const HeadArgs* ha,
                          int n_sm, cudaStream_t st) {
  static const HeadArgs h0{};
  if (f16) {
    if (ha) return launch_pair_t<C, true, true, CG2>(in, out, geo, wA, wB, lcA, lcB, nA, nB, smem, *ha, n_sm, st);
    return launch_pair_t<C, false, true, CG2>(in, out, geo, wA, wB, lcA, lcB, nA, nB, smem, h0, n_sm, st);
  }
  if (ha) return launch_pair_t<C, true, false, CG2>(in, out, geo, wA, wB, lcA, lcB, nA, nB, smem, *ha, n_sm, st);
  return launch_pair_t<C, false, false, CG2>(in, out, geo, wA, wB, lcA, lcB, nA, nB, smem, h0, n_sm, st);
}

}  // namespace

bool conv_pair_supports(int C, int dA, int dB, int W) {
  int nA, nB;
  // TMEM: 9 slots of C columns; cluster = segments of a row
  return C >= 16 && C <= 48 && C % 16 == 0 && dA >= 1 && dB == 2 * dA && dB <= 16 && W >= 1 &&
         (W + kTileM - 1) / kTileM <= kMaxCluster &&
         pick_pair_stages(C, dA, true, false, &nA, &nB);  // (cta_group::2 needs less shared memory)
}

cudaError_t launch_conv_pair(bool f16, const void* in, void* out, ActShape s, int dA, const void* wpackA,
                             const void* wpackB, const LayerConst& lcA, const LayerConst& lcB, const HeadArgs* head,
                             bool allow_cg2, int n_sm, cudaStream_t st, char* err, size_t errlen) {
  if (!conv_pair_supports(s.C, dA, 2 * dA, s.W)) {
    snprintf(err, errlen, "unsupported layer pair");
    return cudaErrorInvalidValue;
  }
  if (s.B <= 0) return cudaSuccess;
  PGeo geo;
  geo.B = s.B;
  geo.H = s.H;
  geo.W = s.W;
  geo.d = dA;
  geo.nseg = (s.W + kTileM - 1) / kTileM;
  geo.Lmax = (s.H + dA - 1) / dA;
  geo.total = (long long)s.B * dA * geo.Lmax;
  int nA = 0, nB = 0;
  const bool cg2 = pair_uses_cg2(geo.nseg, allow_cg2);
  pick_pair_stages(s.C, dA, head != nullptr, cg2, &nA, &nB);
  // One CTA per SM, whatever C: every CTA allocates all 512 TMEM columns with a blocking
  // tcgen05.alloc, so two co-resident CTAs of different clusters, each waiting for cluster peers
  // queued behind the other's allocation, would deadlock.  __launch_bounds__(608, 1) does not
  // forbid a second CTA; the small-C instantiations need little shared memory and few registers.
  // Asking for more than half of an SM's 228 KB does (and makes the cluster-occupancy figure
  // cached per cluster size in launch_pair_t independent of d and of the stage counts).
  const size_t smem = std::max<size_t>(pair_smem(s.C, dA, nA, nB, head != nullptr, cg2).total + 1024, 116 * 1024);
#define SMLM_PAIR_CASE(CC)                                                                                          \
  case CC:                                                                                                          \
    return cg2 ? launch_pair_c<CC, true>(f16, in, out, geo, wpackA, wpackB, lcA, lcB, nA, nB, smem, head, n_sm, st)  \
               : launch_pair_c<CC, false>(f16, in, out, geo, wpackA, wpackB, lcA, lcB, nA, nB, smem, head, n_sm, st);
  switch (s.C) {
    SMLM_PAIR_CASE(16)
    SMLM_PAIR_CASE(32)
    SMLM_PAIR_CASE(48)
  }
#undef SMLM_PAIR_CASE
  return cudaErrorInvalidValue;
}

}  // namespace smlm
