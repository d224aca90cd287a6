// build.cu -- build steps B1 (scene bounds), B2 (space-filling codes), B4 (leaf emission),
// B5+B6 (bottom-up hierarchy fused with bounding-volume refit).  SURVEY.md §8(a).
// PAPER.md:L293 (64-bit Morton codes), L294 (bottom-up hierarchy construction fused with
// bounding volumes, after Apetrei 2014), L309 (16-byte point leaves).
#include <algorithm>

#include "geom.cuh"

namespace arbx {
namespace {

constexpr int BT = 256;   // threads per block of the streaming build kernels

inline int grid_for(int64_t n, int threads, int max_blocks) {
  int64_t b = (n + threads - 1) / threads;
  return (int)std::max<int64_t>(1, std::min<int64_t>(b, max_blocks));
}

// ---- B1: scene bounds ------------------------------------------------------------------------
// enc[0..D) = ordered-uint min of lo, enc[D..2D) = ordered-uint max of hi
__global__ void bounds_init_kernel(uint32_t* enc, int D) {
  int a = threadIdx.x;
  if (a < D) enc[a] = 0xffffffffu;
  else if (a < 2 * D) enc[a] = 0u;
}

template <int D, int PK>
__global__ void __launch_bounds__(BT) bounds_kernel(const float* __restrict__ prims, int64_t n,
                                                    uint32_t* __restrict__ enc) {
  constexpr int W = prim_width(PK, D);
  float lo[D], hi[D];
#pragma unroll
  for (int a = 0; a < D; ++a) { lo[a] = INFINITY; hi[a] = -INFINITY; }
  for (int64_t i = (int64_t)blockIdx.x * BT + threadIdx.x; i < n; i += (int64_t)gridDim.x * BT) {
    float v[W];
#pragma unroll
    for (int e = 0; e < W; ++e) v[e] = __ldg(prims + i * W + e);
    float bl[D], bh[D];
    box_of<D, PK>(v, bl, bh);
#pragma unroll
    for (int a = 0; a < D; ++a) { lo[a] = fminf(lo[a], bl[a]); hi[a] = fmaxf(hi[a], bh[a]); }
  }
#pragma unroll
  for (int a = 0; a < D; ++a)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(~0u, lo[a], o));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(~0u, hi[a], o));
    }
  __shared__ float s_lo[BT / 32][D], s_hi[BT / 32][D];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0)
#pragma unroll
    for (int a = 0; a < D; ++a) { s_lo[w][a] = lo[a]; s_hi[w][a] = hi[a]; }
  __syncthreads();
  if (threadIdx.x < D) {
    const int a = threadIdx.x;
    float l = s_lo[0][a], h = s_hi[0][a];
    for (int i = 1; i < BT / 32; ++i) { l = fminf(l, s_lo[i][a]); h = fmaxf(h, s_hi[i][a]); }
    atomicMin(enc + a, f2ord(l));
    atomicMax(enc + D + a, f2ord(h));
  }
}

// decode the ordered-uint bounds into floats: bounds = lo[D], hi[D]
__global__ void bounds_decode_kernel(const uint32_t* enc, float* bounds, int D) {
  int a = threadIdx.x;
  if (a < 2 * D) bounds[a] = ord2f(enc[a]);
}

// ---- B2: 64-bit space-filling codes of primitive centres -------------------------------------
template <int D, int PK>
__global__ void __launch_bounds__(BT) codes_kernel(const float* __restrict__ prims, int64_t n,
                                                   const float* __restrict__ bounds,
                                                   unsigned long long* __restrict__ codes) {
  constexpr int W = prim_width(PK, D);
  constexpr int B = code_bits_per_axis(D);
  float lo[D], scale[D];
#pragma unroll
  for (int a = 0; a < D; ++a) {
    lo[a] = bounds[a];
    float ext = bounds[D + a] - lo[a];
    scale[a] = ext > 0.f ? exp2f((float)B) / ext : 0.f;
  }
  for (int64_t i = (int64_t)blockIdx.x * BT + threadIdx.x; i < n; i += (int64_t)gridDim.x * BT) {
    float v[W], c[D];
#pragma unroll
    for (int e = 0; e < W; ++e) v[e] = __ldg(prims + i * W + e);
    centre_of<D, PK>(v, c);
    uint32_t q[D];
    quantise<D, B>(c, lo, scale, q);
    codes[i] = interleave<D, B, unsigned long long>(q);
  }
}

// ---- B4: leaves in sorted order ---------------------------------------------------------------
template <int D, int PK>
__global__ void __launch_bounds__(BT) leaves_kernel(const float* __restrict__ prims,
                                                    const uint32_t* __restrict__ perm, int64_t n,
                                                    float* __restrict__ leaves) {
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
  const int64_t j = (int64_t)blockIdx.x * BT + threadIdx.x;
  if (j >= n) return;
  const uint32_t i = perm[j];
  float v[LW];
#pragma unroll
  for (int e = 0; e < W; ++e) v[e] = __ldg(prims + (int64_t)i * W + e);
  v[W] = __uint_as_float(i);
#pragma unroll
  for (int e = W + 1; e < LW; ++e) v[e] = 0.f;
  float4* out = reinterpret_cast<float4*>(leaves + j * LW);
#pragma unroll
  for (int e = 0; e < LW / 4; ++e) out[e] = make_float4(v[4 * e], v[4 * e + 1], v[4 * e + 2], v[4 * e + 3]);
}

// ---- B5+B6: bottom-up hierarchy with fused refit ------------------------------------------------
// Adjacent-leaf metric: XOR of the two codes; equal codes fall back to the XOR of the sorted
// positions (SURVEY.md reading A16), ordered below every non-zero code XOR.
struct Delta { unsigned long long x; uint32_t ix; };
__device__ __forceinline__ Delta delta_at(const unsigned long long* __restrict__ codes, int i) {
  Delta d;
  d.x = __ldg(codes + i) ^ __ldg(codes + i + 1);
  d.ix = (uint32_t)i ^ (uint32_t)(i + 1);
  return d;
}
__device__ __forceinline__ bool delta_less(const Delta& a, const Delta& b) {
  return a.x != b.x ? a.x < b.x : a.ix < b.ix;
}

template <int D, int PK>
__global__ void __launch_bounds__(BT) hierarchy_kernel(const unsigned long long* __restrict__ codes,
                                                       float* __restrict__ leaves, float* __restrict__ nodes,
                                                       int* __restrict__ flags, int n, int leaf_max,
                                                       int32_t* __restrict__ root) {
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
  constexpr int NW = node_width(D);
  const int i = blockIdx.x * BT + threadIdx.x;
  if (i >= n) return;
  int l = i, r = i;
  int32_t ref = ~i;
  float lo[D], hi[D];
  {
    float v[W];
    const float* lf = leaves + (int64_t)i * LW;
#pragma unroll
    for (int e = 0; e < W; ++e) v[e] = lf[e];
    box_of<D, PK>(v, lo, hi);
  }
  uint32_t* leaf_idx = reinterpret_cast<uint32_t*>(leaves);
  for (;;) {
    if (l == 0 && r == n - 1) {   // root
      *root = ref;
      if (ref < 0) leaf_idx[(int64_t)r * LW + W] |= LEAF_END;
      return;
    }
    // the parent splits either right after r (we are its left child) or right before l
    bool left_child;
    if (l == 0) left_child = true;
    else if (r == n - 1) left_child = false;
    else left_child = delta_less(delta_at(codes, r), delta_at(codes, l - 1));
    const int p = left_child ? r : l - 1;
    float* node = nodes + (int64_t)p * NW;
    const int slot = left_child ? 0 : 1;
#pragma unroll
    for (int a = 0; a < D; ++a) {
      __stcg(node + slot * 2 * D + a, lo[a]);
      __stcg(node + slot * 2 * D + D + a, hi[a]);
    }
    __stcg(reinterpret_cast<int*>(node) + 4 * D + slot, ref);
    __threadfence();
    const int other = atomicExch(flags + p, left_child ? l : r);
    if (other == -1) return;     // first to arrive: the sibling's thread carries on
    __threadfence();
    // second to arrive: `other` is the far end of the sibling's range
    const int sib = 1 - slot;
#pragma unroll
    for (int a = 0; a < D; ++a) {
      lo[a] = fminf(lo[a], __ldcg(node + sib * 2 * D + a));
      hi[a] = fmaxf(hi[a], __ldcg(node + sib * 2 * D + D + a));
    }
    if (left_child) r = other; else l = other;
    __stcg(reinterpret_cast<int*>(node) + 4 * D + 2, l);
    __stcg(reinterpret_cast<int*>(node) + 4 * D + 3, r);
    if (r - l + 1 <= leaf_max) {
      ref = ~l;                  // collapsed subtree: a leaf range, node p stays unused
    } else {
      ref = p;
      if (p - l + 1 <= leaf_max) leaf_idx[(int64_t)p * LW + W] |= LEAF_END;
      if (r - p <= leaf_max) leaf_idx[(int64_t)r * LW + W] |= LEAF_END;
    }
  }
}

template <int D, int PK>
arbx_status build_typed(const float* prims, int64_t n, cudaStream_t s, Index* ix, int sms) {
  constexpr int LW = leaf_width(PK, D);
  constexpr int NW = node_width(D);
  Scratch<uint32_t> enc, perm;
  Scratch<int> flags;
  ARBX_TRY(enc.alloc(2 * D, s));
  const int sgrid = grid_for(n, BT, sms * 8);
  {
    ProfScope ps(K_BOUNDS, s);
    bounds_init_kernel<<<1, 32, 0, s>>>(enc.p, D);
    ARBX_LAUNCH_CHECK();
    bounds_kernel<D, PK><<<sgrid, BT, 0, s>>>(prims, n, enc.p);
    ARBX_LAUNCH_CHECK();
    bounds_decode_kernel<<<1, 32, 0, s>>>(enc.p, ix->bounds, D);
    ARBX_LAUNCH_CHECK();
  }

  ARBX_TRY(scratch_alloc((void**)&ix->codes, (size_t)n * sizeof(unsigned long long), s));
  {
    ProfScope ps(K_CODES, s);
    codes_kernel<D, PK><<<sgrid, BT, 0, s>>>(prims, n, ix->bounds, ix->codes);
    ARBX_LAUNCH_CHECK();
  }
  ARBX_TRY(perm.alloc((size_t)n, s));
  ARBX_TRY(radix_sort_u64(ix->codes, perm.p, true, n, D * code_bits_per_axis(D), s));

  ARBX_TRY(scratch_alloc((void**)&ix->leaves, (size_t)n * LW * sizeof(float), s));
  const int fgrid = (int)((n + BT - 1) / BT);
  {
    ProfScope ps(K_LEAVES, s);
    leaves_kernel<D, PK><<<fgrid, BT, 0, s>>>(prims, perm.p, n, ix->leaves);
    ARBX_LAUNCH_CHECK();
  }

  const size_t nn = n > 1 ? (size_t)(n - 1) : 1;
  ARBX_TRY(scratch_alloc((void**)&ix->nodes, nn * NW * sizeof(float), s));
  ARBX_TRY(flags.alloc(nn, s));
  ProfScope ps(K_HIERARCHY, s);
  ARBX_CUDA(cudaMemsetAsync(flags.p, 0xff, nn * sizeof(int), s));
  hierarchy_kernel<D, PK><<<fgrid, BT, 0, s>>>(ix->codes, ix->leaves, ix->nodes, flags.p, (int)n,
                                               ix->leaf_max, ix->root);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

template <int D>
arbx_status build_dim(const float* prims, int64_t n, int kind, cudaStream_t s, Index* ix, int sms) {
  switch (kind) {
    case KIND_POINT: return build_typed<D, KIND_POINT>(prims, n, s, ix, sms);
    case KIND_BOX: return build_typed<D, KIND_BOX>(prims, n, s, ix, sms);
    default: return build_typed<D, KIND_SPHERE>(prims, n, s, ix, sms);
  }
}

__global__ void empty_bounds_kernel(float* bounds, int D) {
  int a = threadIdx.x;
  if (a < D) bounds[a] = INFINITY;
  else if (a < 2 * D) bounds[a] = -INFINITY;
}

}  // namespace

arbx_status build_index(const float* prims, int64_t n, int dim, int kind, cudaStream_t s, Index* ix) {
  ix->n = n; ix->dim = dim; ix->kind = kind;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  ARBX_TRY(scratch_alloc((void**)&ix->bounds, 2 * ARBX_MAX_DIM * sizeof(float), s));
  ARBX_TRY(scratch_alloc((void**)&ix->root, sizeof(int32_t), s));
  if (n == 0) {
    empty_bounds_kernel<<<1, 32, 0, s>>>(ix->bounds, dim);
    ARBX_LAUNCH_CHECK();
    return ARBX_OK;
  }
  switch (dim) {
#define ARBX_CASE(DD) case DD: return build_dim<DD>(prims, n, kind, s, ix, sms);
    ARBX_CASE(1) ARBX_CASE(2) ARBX_CASE(3) ARBX_CASE(4) ARBX_CASE(5)
    ARBX_CASE(6) ARBX_CASE(7) ARBX_CASE(8) ARBX_CASE(9) ARBX_CASE(10)
#undef ARBX_CASE
  }
  return ARBX_ERR_INVALID_ARG;
}

}  // namespace arbx
