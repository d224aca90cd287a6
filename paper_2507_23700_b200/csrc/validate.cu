// validate.cu -- structural self-check of the tree (test hook, SURVEY.md §8(c-5) pin P9).
// Not on the hot path.  Checks, on the device:
//   V0 the build raised no fault flag;
//   V1 the codes of the leaves (recomputed from the leaf records) are non-decreasing;
//   V2 the leaf indices are a permutation of [0,n);
//   V3 every real internal node (range larger than leaf_max) has children whose ranges
//      partition its own range at its split position, and each stored child box equals the
//      union of that child's contents bit for bit (min/max are exact);
//   V4 every real node except the root is referenced exactly once, every leaf lies in exactly
//      one leaf range, the root covers [0,n).
#include "geom.cuh"

namespace arbx {
namespace {

__device__ __forceinline__ void fail(unsigned long long* v) { atomicAdd(v, 1ull); }

// V1: the codes are not kept after the build; they are recomputed here from the leaf records
// (the same geometry, the same quantisation) and must be non-decreasing along the leaves.
template <int D, int PK>
__device__ unsigned long long leaf_code(const float* leaves, int j, const float* bounds, int drop) {
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
  constexpr int B = code_bits_per_axis(D);
  float v[W], c[D], lo[D], scale[D];
  for (int e = 0; e < W; ++e) v[e] = leaves[(int64_t)j * LW + e];
  for (int a = 0; a < D; ++a) {
    lo[a] = bounds[a];
    const float ext = bounds[D + a] - lo[a];
    scale[a] = ext > 0.f ? exp2f((float)B) / ext : 0.f;
  }
  centre_of<D, PK>(v, c);
  uint32_t q[D];
  quantise<D, B>(c, lo, scale, q);
  return interleave<D, B, unsigned long long>(q) >> drop;
}
template <int D, int PK>
__global__ void v_codes_kernel(const float* leaves, const float* bounds, int n, int drop, unsigned long long* viol) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i + 1 < n && leaf_code<D, PK>(leaves, i, bounds, drop) > leaf_code<D, PK>(leaves, i + 1, bounds, drop)) fail(viol);
}
__global__ void v_fault_kernel(const int32_t* root, unsigned long long* viol) {
  if (root[1] != 0) fail(viol);   // V0: the build raised a fault flag (parked-subtree list overflow)
}

__global__ void v_perm_kernel(const float* leaves, int LW, int W, int n, int* seen,
                              unsigned long long* viol) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  uint32_t idx = __float_as_uint(leaves[(int64_t)j * LW + W]) & ~LEAF_END;
  if (idx >= (uint32_t)n) { fail(viol); return; }
  atomicAdd(seen + idx, 1);
}

__global__ void v_ones_kernel(const int* a, int n, unsigned long long* viol) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n && a[j] != 1) fail(viol);
}

template <int D, int PK>
__device__ void leaf_range_box(const float* leaves, int first, int last_expected, int n, float (&lo)[D],
                               float (&hi)[D], int* cover, unsigned long long* viol) {
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
#pragma unroll
  for (int a = 0; a < D; ++a) { lo[a] = INFINITY; hi[a] = -INFINITY; }
  int j = first;
  for (;; ++j) {
    if (j >= n) { fail(viol); return; }
    float v[W], bl[D], bh[D];
    for (int e = 0; e < W; ++e) v[e] = leaves[(int64_t)j * LW + e];
    box_of<D, PK>(v, bl, bh);
    for (int a = 0; a < D; ++a) { lo[a] = fminf(lo[a], bl[a]); hi[a] = fmaxf(hi[a], bh[a]); }
    atomicAdd(cover + j, 1);
    if (__float_as_uint(leaves[(int64_t)j * LW + W]) & LEAF_END) break;
  }
  if (j != last_expected) fail(viol);
}

template <int D, int PK>
__device__ void check_child(const float* leaves, const float* nodes, int32_t ref, int cl, int cr, int n,
                            int leaf_max, const float* slo, const float* shi, int* refcnt, int* cover,
                            unsigned long long* viol) {
  constexpr int NW = node_width(D);
  float lo[D], hi[D];
  if (ref < 0) {
    if (~ref != cl || cr - cl + 1 > leaf_max) fail(viol);
    leaf_range_box<D, PK>(leaves, ~ref, cr, n, lo, hi, cover, viol);
  } else {
    if (ref >= n - 1) { fail(viol); return; }
    const float* c = nodes + (int64_t)ref * NW;
    const int* ci = reinterpret_cast<const int*>(c) + 4 * D;
    if (ci[2] != cl || ci[3] != cr || cr - cl + 1 <= leaf_max || ref < cl || ref >= cr) fail(viol);
    atomicAdd(refcnt + ref, 1);
    for (int a = 0; a < D; ++a) {
      lo[a] = fminf(c[a], c[2 * D + a]);
      hi[a] = fmaxf(c[D + a], c[3 * D + a]);
    }
  }
  for (int a = 0; a < D; ++a)
    if (__float_as_uint(lo[a]) != __float_as_uint(slo[a]) || __float_as_uint(hi[a]) != __float_as_uint(shi[a]))
      fail(viol);
}

template <int D, int PK>
__global__ void v_nodes_kernel(const float* leaves, const float* nodes, int n, int leaf_max, int* refcnt,
                               int* cover, int* real, unsigned long long* viol) {
  constexpr int NW = node_width(D);
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n - 1) return;
  const float* nd = nodes + (int64_t)p * NW;
  const int* ni = reinterpret_cast<const int*>(nd) + 4 * D;
  // a split inside a leaf range has no node (its slot is never written): leaf p does not carry
  // the end-of-range mark
  if (!(__float_as_uint(leaves[(int64_t)p * leaf_width(PK, D) + prim_width(PK, D)]) & LEAF_END)) return;
  const int l = ni[2], r = ni[3];
  if (l < 0 || r >= n || l > p || r <= p) { fail(viol); return; }
  if (r - l + 1 <= leaf_max) { fail(viol); return; }   // leaf ranges are maximal
  real[p] = 1;
  check_child<D, PK>(leaves, nodes, ni[0], l, p, n, leaf_max, nd, nd + D, refcnt, cover, viol);
  check_child<D, PK>(leaves, nodes, ni[1], p + 1, r, n, leaf_max, nd + 2 * D, nd + 3 * D, refcnt, cover, viol);
}

template <int D, int PK>
__global__ void v_root_kernel(const float* leaves, const float* nodes, const float* bounds,
                              const int32_t* root, int n, int leaf_max, int* refcnt, int* cover,
                              unsigned long long* viol) {
  constexpr int NW = node_width(D);
  if (blockIdx.x || threadIdx.x) return;
  int32_t ref = *root;
  float lo[D], hi[D];
  if (ref < 0) {
    if (~ref != 0 || n > leaf_max) fail(viol);
    leaf_range_box<D, PK>(leaves, 0, n - 1, n, lo, hi, cover, viol);
  } else {
    if (ref >= n - 1) { fail(viol); return; }
    const float* c = nodes + (int64_t)ref * NW;
    const int* ci = reinterpret_cast<const int*>(c) + 4 * D;
    if (ci[2] != 0 || ci[3] != n - 1) fail(viol);
    atomicAdd(refcnt + ref, 1);
    for (int a = 0; a < D; ++a) {
      lo[a] = fminf(c[a], c[2 * D + a]);
      hi[a] = fmaxf(c[D + a], c[3 * D + a]);
    }
  }
  // root box == scene bounds (B1), bit for bit
  for (int a = 0; a < D; ++a)
    if (__float_as_uint(lo[a]) != __float_as_uint(bounds[a]) ||
        __float_as_uint(hi[a]) != __float_as_uint(bounds[D + a]))
      fail(viol);
}

__global__ void v_refs_kernel(const int* refcnt, const int* real, int n1, unsigned long long* viol) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n1 && refcnt[p] != real[p]) fail(viol);
}

template <int D, int PK>
arbx_status validate_typed(const Index* ix, unsigned long long* viol, cudaStream_t s) {
  const int n = (int)ix->n;
  const int T = 256, g = (n + T - 1) / T;
  Scratch<int> seen, cover, refcnt, real;
  ARBX_TRY(seen.alloc(n, s)); ARBX_TRY(cover.alloc(n, s));
  ARBX_TRY(refcnt.alloc(n, s)); ARBX_TRY(real.alloc(n, s));
  ARBX_CUDA(cudaMemsetAsync(seen.p, 0, sizeof(int) * n, s));
  ARBX_CUDA(cudaMemsetAsync(cover.p, 0, sizeof(int) * n, s));
  ARBX_CUDA(cudaMemsetAsync(refcnt.p, 0, sizeof(int) * n, s));
  ARBX_CUDA(cudaMemsetAsync(real.p, 0, sizeof(int) * n, s));
  v_fault_kernel<<<1, 1, 0, s>>>(ix->root, viol); ARBX_LAUNCH_CHECK();
  if (!ix->brute) v_codes_kernel<D, PK><<<g, T, 0, s>>>(ix->leaves, ix->bounds, n, D * (code_bits_per_axis(D) - ix->code_bits), viol); ARBX_LAUNCH_CHECK();
  v_perm_kernel<<<g, T, 0, s>>>(ix->leaves, leaf_width(PK, D), prim_width(PK, D), n, seen.p, viol); ARBX_LAUNCH_CHECK();
  v_ones_kernel<<<g, T, 0, s>>>(seen.p, n, viol); ARBX_LAUNCH_CHECK();
  if (n > 1) { v_nodes_kernel<D, PK><<<g, T, 0, s>>>(ix->leaves, ix->nodes, n, ix->leaf_max, refcnt.p, cover.p, real.p, viol); ARBX_LAUNCH_CHECK(); }
  v_root_kernel<D, PK><<<1, 32, 0, s>>>(ix->leaves, ix->nodes, ix->bounds, ix->root, n, ix->leaf_max, refcnt.p, cover.p, viol); ARBX_LAUNCH_CHECK();
  v_ones_kernel<<<g, T, 0, s>>>(cover.p, n, viol); ARBX_LAUNCH_CHECK();
  if (n > 1) { v_refs_kernel<<<g, T, 0, s>>>(refcnt.p, real.p, n - 1, viol); ARBX_LAUNCH_CHECK(); }
  return ARBX_OK;
}

template <int D>
arbx_status validate_dim(const Index* ix, unsigned long long* viol, cudaStream_t s) {
  switch (ix->kind) {
    case KIND_POINT: return validate_typed<D, KIND_POINT>(ix, viol, s);
    case KIND_BOX: return validate_typed<D, KIND_BOX>(ix, viol, s);
    default: return validate_typed<D, KIND_SPHERE>(ix, viol, s);
  }
}

}  // namespace

arbx_status validate_index(const Index* ix, int64_t* violations_host, cudaStream_t s) {
  *violations_host = 0;
  if (ix->n == 0) return ARBX_OK;
  Scratch<unsigned long long> viol;
  ARBX_TRY(viol.alloc(1, s));
  ARBX_CUDA(cudaMemsetAsync(viol.p, 0, sizeof(unsigned long long), s));
  arbx_status st = ARBX_ERR_INVALID_ARG;
  switch (ix->dim) {
#define ARBX_CASE(DD) case DD: st = validate_dim<DD>(ix, viol.p, s); break;
    ARBX_CASE(1) ARBX_CASE(2) ARBX_CASE(3) ARBX_CASE(4) ARBX_CASE(5)
    ARBX_CASE(6) ARBX_CASE(7) ARBX_CASE(8) ARBX_CASE(9) ARBX_CASE(10)
#undef ARBX_CASE
  }
  ARBX_TRY(st);
  unsigned long long h = 0;
  ARBX_CUDA(cudaMemcpyAsync(&h, viol.p, sizeof(h), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaStreamSynchronize(s));
  *violations_host = (int64_t)h;
  return ARBX_OK;
}

}  // namespace arbx
