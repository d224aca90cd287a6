// geom.cuh -- device helpers: space-filling codes (B2/Q1), leaf/box arithmetic (B6, T1/T3, K1).
//
// Rounding discipline: every squared distance is accumulated with the
// SAME operation sequence  s = fmaf(d, d, s)  in axis order, for points and for boxes.  fp32
// subtraction, fmaf and max are monotone, so for a primitive inside a node's box the node's
// value is <= the primitive's value bit for bit: culling is exactly conservative with
// respect to the fp32 leaf test, and the result equals fp32 brute force.
#pragma once
#include "common.cuh"

namespace arbx {

// order-preserving map float -> uint32 (for atomicMin/atomicMax on floats)
__device__ __forceinline__ uint32_t f2ord(float f) {
  uint32_t u = __float_as_uint(f);
  return u ^ ((u >> 31) ? 0xffffffffu : 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t u) {
  return __uint_as_float(u ^ ((u >> 31) ? 0x80000000u : 0xffffffffu));
}

__host__ __device__ constexpr int code_bits_per_axis(int D) { return 64 / D > 32 ? 32 : 64 / D; }
__host__ __device__ constexpr int qcode_bits_per_axis(int D) { return 32 / D > 16 ? 16 : 32 / D; }

// interleave B bits of each of D quantised coordinates: bit j of axis a -> bit j*D + a
template <int D, int B, typename C>
__device__ __forceinline__ C interleave(const uint32_t (&q)[D]) {
  if constexpr (D == 1) {
    return (C)q[0];
  } else if constexpr (D == 3 && B == 21) {
    C c = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      unsigned long long x = q[a] & 0x1fffffull;
      x = (x | x << 32) & 0x1f00000000ffffull;
      x = (x | x << 16) & 0x1f0000ff0000ffull;
      x = (x | x << 8) & 0x100f00f00f00f00full;
      x = (x | x << 4) & 0x10c30c30c30c30c3ull;
      x = (x | x << 2) & 0x1249249249249249ull;
      c |= (C)(x << a);
    }
    return c;
  } else if constexpr (D == 3 && B == 10) {
    C c = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      uint32_t x = q[a] & 0x3ffu;
      x = (x | x << 16) & 0x030000ffu;
      x = (x | x << 8) & 0x0300f00fu;
      x = (x | x << 4) & 0x030c30c3u;
      x = (x | x << 2) & 0x09249249u;
      c |= (C)(x << a);
    }
    return c;
  } else {
    C c = 0;
#pragma unroll
    for (int j = 0; j < B; ++j)
#pragma unroll
      for (int a = 0; a < D; ++a) c |= (C)((q[a] >> j) & 1u) << (j * D + a);
    return c;
  }
}

// quantise a centre into B bits per axis inside [lo, lo + extent]; scale[a] = 2^B/extent or 0.
// Out-of-range values (query centres outside the scene) saturate to the nearest cell.
template <int D, int B>
__device__ __forceinline__ void quantise(const float (&c)[D], const float* lo, const float* scale,
                                         uint32_t (&q)[D]) {
  constexpr uint32_t QMAX = B >= 32 ? 0xffffffffu : ((1u << (B & 31)) - 1u);
#pragma unroll
  for (int a = 0; a < D; ++a) q[a] = min(__float2uint_rz((c[a] - lo[a]) * scale[a]), QMAX);
}

// centre used for the space-filling code of a primitive/query row of `kind`
template <int D, int KIND>
__device__ __forceinline__ void centre_of(const float* v, float (&c)[D]) {
#pragma unroll
  for (int a = 0; a < D; ++a) c[a] = KIND == KIND_BOX ? 0.5f * v[a] + 0.5f * v[D + a] : v[a];
}

// AABB of a primitive row; spheres are rounded outward so the box really contains them
template <int D, int KIND>
__device__ __forceinline__ void box_of(const float* v, float (&lo)[D], float (&hi)[D]) {
#pragma unroll
  for (int a = 0; a < D; ++a) {
    if constexpr (KIND == KIND_POINT) { lo[a] = v[a]; hi[a] = v[a]; }
    else if constexpr (KIND == KIND_BOX) { lo[a] = v[a]; hi[a] = v[D + a]; }
    else { lo[a] = __fsub_rd(v[a], v[D]); hi[a] = __fadd_ru(v[a], v[D]); }
  }
}

// squared distance point-point / point-box with the shared accumulation order
template <int D>
__device__ __forceinline__ float dist2_pp(const float* x, const float* y) {
  float s = 0.f;
#pragma unroll
  for (int a = 0; a < D; ++a) { float d = x[a] - y[a]; s = fmaf(d, d, s); }
  return s;
}
template <int D>
__device__ __forceinline__ float dist2_pb(const float* x, const float* lo, const float* hi) {
  float s = 0.f;
#pragma unroll
  for (int a = 0; a < D; ++a) {
    float d = fmaxf(0.f, fmaxf(lo[a] - x[a], x[a] - hi[a]));
    s = fmaf(d, d, s);
  }
  return s;
}

}  // namespace arbx
