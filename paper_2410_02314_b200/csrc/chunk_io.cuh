// 8-channel chunk load/store for the chunk-planar activation layout (smlm_internal.cuh).
// bf16 / fp16: one 16-byte vector per (pixel, chunk); float: two.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace smlm {

template <typename T>
struct Chunk;

template <>
struct Chunk<float> {
  static constexpr int kBytes = 32;
  __device__ static inline void load(const void* base, size_t idx, float v[8]) {
    const float4* p = reinterpret_cast<const float4*>(base) + idx * 2;
    float4 a = p[0], b = p[1];
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
    v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  }
  __device__ static inline void store(void* base, size_t idx, const float v[8]) {
    float4* p = reinterpret_cast<float4*>(base) + idx * 2;
    p[0] = make_float4(v[0], v[1], v[2], v[3]);
    p[1] = make_float4(v[4], v[5], v[6], v[7]);
  }
};

template <>
struct Chunk<__nv_bfloat16> {
  static constexpr int kBytes = 16;
  __device__ static inline void load(const void* base, size_t idx, float v[8]) {
    uint4 q = reinterpret_cast<const uint4*>(base)[idx];
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      v[2 * i] = __uint_as_float(w[i] << 16);
      v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
  __device__ static inline void store(void* base, size_t idx, const float v[8]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      __nv_bfloat162 h = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);  // .x = low half
      w[i] = *reinterpret_cast<uint32_t*>(&h);
    }
    reinterpret_cast<uint4*>(base)[idx] = make_uint4(w[0], w[1], w[2], w[3]);
  }
};

template <>
struct Chunk<__half> {
  static constexpr int kBytes = 16;
  __device__ static inline void load(const void* base, size_t idx, float v[8]) {
    uint4 q = reinterpret_cast<const uint4*>(base)[idx];
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
      v[2 * i] = f.x;
      v[2 * i + 1] = f.y;
    }
  }
  __device__ static inline void store(void* base, size_t idx, const float v[8]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      __half2 h = __floats2half2_rn(v[2 * i], v[2 * i + 1]);  // .x = low half
      w[i] = *reinterpret_cast<uint32_t*>(&h);
    }
    reinterpret_cast<uint4*>(base)[idx] = make_uint4(w[0], w[1], w[2], w[3]);
  }
};

}  // namespace smlm
