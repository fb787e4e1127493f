// K1: uint16 unpack + offset/gain normalisation + 3x3 stem convolution (IN -> C) (+ReLU),
// fused (BASELINE.json north_star (a); smlm.h: xhat = ((adu - offset)/gain)/norm_scale,
// a0 = act(conv3x3(xhat; W0) + b0), zero padding 1 at the FRAME border).
//
// HBM/L2-write-bound: 2 B/px in, 2C B/px out (bf16).  One thread = four pixels 32 apart, all
// C channels; a warp covers 32 consecutive pixels of a row per store, so each store is one
// dense 512 B run in the chunk-planar layout.  The normalised (TY+2) x (TX+2) input patch is staged in
// shared memory once per block (the divisions happen once per pixel, not once per tap).
// IN = 3 (smlm_net_desc.in_frames): the input channels are the frames f-1, f, f+1 of the
// call, indices clamped to [0, n_total - 1]; taps are accumulated in (channel, ky, kx) order.
#include "chunk_io.cuh"
#include "smlm_internal.cuh"

namespace smlm {
namespace {

constexpr int TX = 128, PX = 4;  // tile = 128 pixels of one row; pixels per thread (x, x+32, x+64, x+96)
constexpr int NW = 4;            // warps per block, one tile each per round

__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
  return ((unsigned long long)__float_as_uint(hi) << 32) | __float_as_uint(lo);
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b,
                                                    unsigned long long c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}

// Persistent blocks: tile t = (view, row, 128-px segment); warp w of block j takes tiles
// (j * NW + w), + gridDim.x * NW, ...  With 5 blocks per SM the tail is one row-tile.
template <typename T, int C, int IN>
__global__ void __launch_bounds__(32 * NW)
    stem_kernel(const uint16_t* __restrict__ frames, int frame_base, ViewSet vs, ActShape s,
                NormParams np, const float* __restrict__ w /*[IN * 9][C]*/,
                const float* __restrict__ bias, int relu, T* __restrict__ act) {
  __shared__ float xs[NW][3 * IN][TX + 2];
  __shared__ __align__(16) float2 ws2[9 * IN][C];  // every weight twice: the broadcast operand of fma.rn.f32x2
  __shared__ __align__(16) float bs[C];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (int i = tid; i < 9 * IN * C; i += 32 * NW) ws2[i / C][i % C] = make_float2(w[i], w[i]);
  for (int i = tid; i < C; i += 32 * NW) bs[i] = bias[i];
  __syncthreads();

  const int nseg = (s.W + TX - 1) / TX;
  const long long ntiles = (long long)s.B * s.H * nseg;
  constexpr int PATCH = 3 * (TX + 2), NLD = (PATCH + 31) / 32;
  for (long long t = (long long)blockIdx.x * NW + warp; t < ntiles; t += (long long)gridDim.x * NW) {
    const int seg = (int)(t % nseg);
    const long long ty = t / nseg;
    const int y = (int)(ty % s.H), b = (int)(ty / s.H);
    const int x0 = seg * TX;
    const View v = view_of(vs, b, s.H, s.W);
    __syncwarp();  // the previous tile's reads of xs[warp] are done
#pragma unroll
    for (int ch = 0; ch < IN; ++ch) {
      int g = v.frame;
      if (IN == 3) {  // temporal context: frames f-1, f, f+1, clamped to the call
        g += ch - 1;
        g = g < 0 ? 0 : (g > vs.n_total - 1 ? vs.n_total - 1 : g);
      }
      const uint16_t* frame = frames + (size_t)(g - frame_base) * vs.Hf * vs.Wf;
      // all loads of the 3 x 130 patch first (independent, one round trip), then the arithmetic
      float adu[NLD], om[NLD], gm[NLD];
      bool ok[NLD];
#pragma unroll
      for (int r = 0; r < NLD; ++r) {
        const int i = lane + r * 32;
        const int ly = i / (TX + 2), lx = i - ly * (TX + 2);
        const int fy = v.wy0 + y + ly - 1, fx = v.wx0 + x0 + lx - 1;  // frame coordinates
        ok[r] = i < PATCH && fy >= 0 && fy < vs.Hf && fx >= 0 && fx < vs.Wf;
        const size_t q = ok[r] ? (size_t)fy * vs.Wf + fx : 0;
        adu[r] = ok[r] ? (float)__ldg(frame + q) : 0.0f;
        om[r] = (ok[r] && np.offset_map) ? __ldg(np.offset_map + q) : np.offset;
        gm[r] = (ok[r] && np.offset_map) ? __ldg(np.gain_map + q) : np.gain;
      }
#pragma unroll
      for (int r = 0; r < NLD; ++r) {
        const int i = lane + r * 32;
        if (i >= PATCH) continue;
        float xn = 0.0f;
        if (ok[r]) xn = ((adu[r] - om[r]) / gm[r]) / np.norm_scale;  // the oracle's operation order (G5)
        xs[warp][ch * 3 + i / (TX + 2)][i % (TX + 2)] = xn;
      }
    }
    __syncwarp();

    // Each thread owns PX = 4 pixels 32 apart in x, held as two pixel pairs: one packed
    // fma.rn.f32x2 (two independent IEEE fp32 FMAs, same bits as fmaf) updates one channel of
    // a pair, which halves the FMA instruction count of this issue-bound loop; every store of
    // the warp is one dense 512-byte run.
    unsigned long long xp[PX / 2][9 * IN];
#pragma unroll
    for (int pp = 0; pp < PX / 2; ++pp)
#pragma unroll
      for (int ky = 0; ky < 3 * IN; ++ky)  // (channel, ky) rows of the patch
#pragma unroll
        for (int kx = 0; kx < 3; ++kx)
          xp[pp][ky * 3 + kx] = pack2(xs[warp][ky][lane + 64 * pp + kx], xs[warp][ky][lane + 64 * pp + 32 + kx]);

#pragma unroll 1
    for (int k = 0; k < C / 8; ++k) {  // not unrolled: keeps the loop body inside the instruction cache
      unsigned long long acc[PX / 2][8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const float bv = bs[k * 8 + c];
#pragma unroll
        for (int pp = 0; pp < PX / 2; ++pp) acc[pp][c] = pack2(bv, bv);
      }
#pragma unroll
      for (int tp = 0; tp < 9 * IN; ++tp)
#pragma unroll
        for (int c = 0; c < 8; c += 2) {
          const ulonglong2 wv = *reinterpret_cast<const ulonglong2*>(&ws2[tp][k * 8 + c]);
#pragma unroll
          for (int pp = 0; pp < PX / 2; ++pp) {
            acc[pp][c] = ffma2(xp[pp][tp], wv.x, acc[pp][c]);
            acc[pp][c + 1] = ffma2(xp[pp][tp], wv.y, acc[pp][c + 1]);
          }
        }
#pragma unroll
      for (int p = 0; p < PX; ++p) {
        const int x = x0 + lane + 32 * p;  // pair pp = p / 2 holds pixels 64 pp (low) and 64 pp + 32 (high)
        if (x >= s.W) continue;
        float v[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const unsigned long long a = acc[p >> 1][c];
          v[c] = __uint_as_float((p & 1) ? (unsigned)(a >> 32) : (unsigned)a);
          if (relu) v[c] = fmaxf(v[c], 0.0f);
        }
        Chunk<T>::store(act, s.chunk_index(b, k, y, x), v);
      }
    }
  }
}

template <typename T, int C, int IN>
cudaError_t launch_tci(const uint16_t* frames, int frame_base, ViewSet vs, ActShape s, NormParams np,
                       const float* w, const float* b, int relu, void* act, cudaStream_t st) {
  static int waves[64] = {};  // resident blocks per device (occupancy is a per-device fact)
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  if (!waves[dev]) {
    int n_sm = 0, per_sm = 0;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, stem_kernel<T, C, IN>, 32 * NW, 0);
    waves[dev] = n_sm * (per_sm > 0 ? per_sm : 1);
  }
  const int blocks_per_wave = waves[dev];
  const long long ntiles = (long long)s.B * s.H * ((s.W + TX - 1) / TX);
  const long long want = (ntiles + NW - 1) / NW;
  const int grid = (int)(want < blocks_per_wave ? want : blocks_per_wave);
  stem_kernel<T, C, IN><<<grid, 32 * NW, 0, st>>>(frames, frame_base, vs, s, np, w, b, relu, (T*)act);
  return cudaGetLastError();
}

template <typename T, int C>
cudaError_t launch_tc(const uint16_t* frames, int frame_base, ViewSet vs, ActShape s, NormParams np,
                      const float* w, const float* b, int relu, void* act, cudaStream_t st) {
  if (vs.in_frames == 3) return launch_tci<T, C, 3>(frames, frame_base, vs, s, np, w, b, relu, act, st);
  return launch_tci<T, C, 1>(frames, frame_base, vs, s, np, w, b, relu, act, st);
}

template <typename T>
cudaError_t launch_t(const uint16_t* frames, int frame_base, ViewSet vs, ActShape s, NormParams np,
                     const float* w, const float* b, int relu, void* act, cudaStream_t st) {
  switch (s.C) {
    case 16: return launch_tc<T, 16>(frames, frame_base, vs, s, np, w, b, relu, act, st);
    case 32: return launch_tc<T, 32>(frames, frame_base, vs, s, np, w, b, relu, act, st);
    case 48: return launch_tc<T, 48>(frames, frame_base, vs, s, np, w, b, relu, act, st);
    case 64: return launch_tc<T, 64>(frames, frame_base, vs, s, np, w, b, relu, act, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

cudaError_t launch_stem(int dt, const uint16_t* frames, int frame_base, ViewSet vs, ActShape s,
                        NormParams np, const float* w_stem, const float* b_stem, int relu,
                        void* act, cudaStream_t st) {
  if (s.B <= 0) return cudaSuccess;
  if (dt == ACT_BF16) return launch_t<__nv_bfloat16>(frames, frame_base, vs, s, np, w_stem, b_stem, relu, act, st);
  if (dt == ACT_F16) return launch_t<__half>(frames, frame_base, vs, s, np, w_stem, b_stem, relu, act, st);
  return launch_t<float>(frames, frame_base, vs, s, np, w_stem, b_stem, relu, act, st);
}

}  // namespace smlm
