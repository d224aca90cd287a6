// f64.cu -- fp64 coordinates ("different data dimensions
// (1-10) and floating point precisions").
//
// Design: fp64 REFINEMENT over the fp32 tree.  Every fp64 primitive gets its bounding box
// rounded OUTWARD to fp32 (lo down, hi up); the ordinary build (build.cu) makes a BOX tree over
// those boxes; the fp64 rows are kept beside it in leaf order.  A query is answered by walking
// the fp32 tree with the query's own outward-rounded fp32 box (spatial) or with lower bounds of
// the fp64 box distance (kNN) -- both can only over-approximate -- and by evaluating the EXACT
// predicate / distance in fp64 on the fp64 rows at the leaves.  So results are those of an fp64
// brute force; the fp32 tree only prunes.  One query per lane, dimension and kinds are run-time
// values (one translation unit, no per-dimension instantiation): this path is about the
// numbers, not about speed.
#include <algorithm>

#include "common.cuh"

namespace arbx {
namespace {

constexpr int FT = 128;   // threads per block

__host__ __device__ inline int pw64(int kind, int D) { return kind == KIND_POINT ? D : kind == KIND_BOX ? 2 * D : D + 1; }

// ---- build side ------------------------------------------------------------------------------------
// fp32 box of every fp64 primitive, rounded outward
__global__ void f64_boxes_kernel(const double* __restrict__ prims, int64_t n, int D, int kind,
                                 float* __restrict__ boxes) {
  const int64_t i = (int64_t)blockIdx.x * FT + threadIdx.x;
  if (i >= n) return;
  const double* p = prims + i * pw64(kind, D);
  for (int a = 0; a < D; ++a) {
    double lo, hi;
    if (kind == KIND_POINT) { lo = p[a]; hi = p[a]; }
    else if (kind == KIND_BOX) { lo = p[a]; hi = p[D + a]; }
    else { lo = __dsub_rd(p[a], p[D]); hi = __dadd_ru(p[a], p[D]); }
    boxes[i * 2 * D + a] = __double2float_rd(lo);
    boxes[i * 2 * D + D + a] = __double2float_ru(hi);
  }
}

// fp64 rows in leaf order: rows64[j] = prims[index of sorted leaf j]
__global__ void f64_gather_kernel(const double* __restrict__ prims, const float* __restrict__ leaves, int64_t n,
                                  int D, int kind, int LW, double* __restrict__ rows64) {
  const int64_t j = (int64_t)blockIdx.x * FT + threadIdx.x;
  if (j >= n) return;
  const uint32_t idx = __float_as_uint(leaves[j * LW + 2 * D]) & ~LEAF_END;
  const int W = pw64(kind, D);
  for (int e = 0; e < W; ++e) rows64[j * W + e] = prims[(int64_t)idx * W + e];
}

// ---- query side -------------------------------------------------------------------------------------
// fp32 box of every fp64 query, rounded outward (also the rows the query sort is computed from)
__global__ void f64_qboxes_kernel(const double* __restrict__ queries, int64_t nq, int D, int qkind,
                                  float* __restrict__ qboxes) {
  const int64_t i = (int64_t)blockIdx.x * FT + threadIdx.x;
  if (i >= nq) return;
  const double* q = queries + i * pw64(qkind, D);
  for (int a = 0; a < D; ++a) {
    double lo, hi;
    if (qkind == KIND_POINT) { lo = q[a]; hi = q[a]; }
    else if (qkind == KIND_BOX) { lo = q[a]; hi = q[D + a]; }
    else { const double r = fmax(q[D], 0.0); lo = __dsub_rd(q[a], r); hi = __dadd_ru(q[a], r); }
    qboxes[i * 2 * D + a] = __double2float_rd(lo);
    qboxes[i * 2 * D + D + a] = __double2float_ru(hi);
  }
}

__device__ inline double d2_pp(const double* x, const double* y, int D) {
  double s = 0.0;
  for (int a = 0; a < D; ++a) { const double d = x[a] - y[a]; s = fma(d, d, s); }
  return s;
}
__device__ inline double d2_pb(const double* x, const double* lo, const double* hi, int D) {
  double s = 0.0;
  for (int a = 0; a < D; ++a) { const double d = fmax(0.0, fmax(lo[a] - x[a], x[a] - hi[a])); s = fma(d, d, s); }
  return s;
}

// the predicate table of SURVEY.md §8(c-1) in fp64, all sets closed
__device__ inline bool pred64(const double* q, int qk, const double* p, int pk, int D) {
  if (qk == KIND_SPHERE) {
    const double r = q[D];
    if (r < 0.0) return false;
    if (pk == KIND_POINT) return d2_pp(p, q, D) <= r * r;
    if (pk == KIND_BOX) return d2_pb(q, p, p + D, D) <= r * r;
    const double rr = r + p[D];
    return d2_pp(p, q, D) <= rr * rr;
  }
  if (qk == KIND_BOX) {
    if (pk == KIND_POINT) { for (int a = 0; a < D; ++a) if (!(q[a] <= p[a] && p[a] <= q[D + a])) return false; return true; }
    if (pk == KIND_BOX) { for (int a = 0; a < D; ++a) if (!(p[a] <= q[D + a] && q[a] <= p[D + a])) return false; return true; }
    return d2_pb(p, q, q + D, D) <= p[D] * p[D];
  }
  if (pk == KIND_POINT) { for (int a = 0; a < D; ++a) if (!(p[a] == q[a])) return false; return true; }
  if (pk == KIND_BOX) { for (int a = 0; a < D; ++a) if (!(p[a] <= q[a] && q[a] <= p[D + a])) return false; return true; }
  return d2_pp(q, p, D) <= p[D] * p[D];
}

__device__ inline bool overlap32(const float* qlo, const float* qhi, const float* lo, const float* hi, int D) {
  for (int a = 0; a < D; ++a) if (!(lo[a] <= qhi[a] && qlo[a] <= hi[a])) return false;
  return true;
}

// One query per lane over the fp32 BOX tree.  fill == 0: counts[q] = matches.  fill == 1:
// indices[offsets[q] ...] = matches.
__global__ void __launch_bounds__(FT) f64_spatial_kernel(const float* __restrict__ nodes, const float* __restrict__ leaves,
                                                         const double* __restrict__ rows64, const int32_t* __restrict__ root,
                                                         int D, int pkind, const double* __restrict__ queries,
                                                         const float* __restrict__ qboxes, const uint32_t* __restrict__ qorder,
                                                         int64_t nq, int qkind, int32_t* __restrict__ counts,
                                                         const int32_t* __restrict__ offsets, int32_t* __restrict__ indices,
                                                         int fill) {
  const int64_t t = (int64_t)blockIdx.x * FT + threadIdx.x;
  if (t >= nq) return;
  const int64_t qi = qorder ? (int64_t)qorder[t] : t;
  const int NW = 4 * (D + 1), LW = (2 * D + 1 + 3) / 4 * 4, PW = pw64(pkind, D);
  double q[2 * ARBX_MAX_DIM];
  float qlo[ARBX_MAX_DIM], qhi[ARBX_MAX_DIM];
  const int QW = pw64(qkind, D);
  for (int e = 0; e < QW; ++e) q[e] = queries[qi * QW + e];
  for (int a = 0; a < D; ++a) { qlo[a] = qboxes[qi * 2 * D + a]; qhi[a] = qboxes[qi * 2 * D + D + a]; }
  int32_t* out = fill ? indices + offsets[qi] : nullptr;
  int cnt = 0;
  if (!(qkind == KIND_SPHERE && q[D] < 0.0)) {
    int32_t stack[STACK_DEPTH];
    int sp = 0;
    constexpr int32_t DONE = INT32_MIN;
    int32_t ref = *root;
    while (ref != DONE) {
      if (ref >= 0) {
        const float* nd = nodes + (int64_t)ref * NW;
        const bool h0 = overlap32(qlo, qhi, nd, nd + D, D);
        const bool h1 = overlap32(qlo, qhi, nd + 2 * D, nd + 3 * D, D);
        const int32_t c0 = __float_as_int(nd[4 * D]), c1 = __float_as_int(nd[4 * D + 1]);
        if (h0) { ref = c0; if (h1) stack[sp++] = c1; }
        else if (h1) ref = c1;
        else ref = sp > 0 ? stack[--sp] : DONE;
        continue;
      }
      for (int64_t j = ~ref;; ++j) {
        const float* lf = leaves + j * LW;
        const uint32_t tag = __float_as_uint(lf[2 * D]);
        if (overlap32(qlo, qhi, lf, lf + D, D) && pred64(q, qkind, rows64 + j * PW, pkind, D)) {
          if (fill) out[cnt] = (int32_t)(tag & ~LEAF_END);
          ++cnt;
        }
        if (tag & LEAF_END) break;
      }
      ref = sp > 0 ? stack[--sp] : DONE;
    }
  }
  if (!fill) counts[qi] = cnt;
}

// kNN: distance (not squared) from the query point to the stored fp64 geometry
__device__ inline double knn_dist64(const double* y, const double* p, int pk, int D) {
  if (pk == KIND_POINT) return sqrt(d2_pp(p, y, D));
  if (pk == KIND_BOX) return sqrt(d2_pb(y, p, p + D, D));
  return fmax(0.0, sqrt(d2_pp(p, y, D)) - p[D]);
}
// lower bound of the distance from y to anything inside the fp32 box [lo,hi] (the box contains
// the primitive's exact box; the factor leaves room for the roundings of the fp64 arithmetic)
__device__ inline double box_bound64(const double* y, const float* lo, const float* hi, int D) {
  double s = 0.0;
  for (int a = 0; a < D; ++a) { const double d = fmax(0.0, fmax((double)lo[a] - y[a], y[a] - (double)hi[a])); s = fma(d, d, s); }
  return sqrt(s) * (1.0 - 1e-12);
}

// binary max-heap of (distance, index) in local memory
struct Heap64 {
  double d[ARBX_K_MAX];
  int32_t i[ARBX_K_MAX];
  int k, m;
  __device__ void init(int k_) { k = k_; m = 0; }
  __device__ double worst() const { return m < k ? INFINITY : d[0]; }
  __device__ void sift_down(int pos, int size, double t, int32_t idx) {
    for (;;) {
      int c = 2 * pos + 1;
      if (c >= size) break;
      if (c + 1 < size && d[c + 1] > d[c]) ++c;
      if (d[c] <= t) break;
      d[pos] = d[c]; i[pos] = i[c];
      pos = c;
    }
    d[pos] = t; i[pos] = idx;
  }
  __device__ void push(double t, int32_t idx) {
    if (m < k) {
      int pos = m++;
      while (pos > 0) {
        const int par = (pos - 1) >> 1;
        if (d[par] >= t) break;
        d[pos] = d[par]; i[pos] = i[par];
        pos = par;
      }
      d[pos] = t; i[pos] = idx;
    } else {
      sift_down(0, k, t, idx);
    }
  }
};

__global__ void __launch_bounds__(FT) f64_knn_kernel(const float* __restrict__ nodes, const float* __restrict__ leaves,
                                                     const double* __restrict__ rows64, const int32_t* __restrict__ root,
                                                     int D, int pkind, const double* __restrict__ qpoints,
                                                     const uint32_t* __restrict__ qorder, int64_t nq, int k,
                                                     int32_t* __restrict__ indices, double* __restrict__ distances) {
  const int64_t t = (int64_t)blockIdx.x * FT + threadIdx.x;
  if (t >= nq) return;
  const int64_t qi = qorder ? (int64_t)qorder[t] : t;
  const int NW = 4 * (D + 1), LW = (2 * D + 1 + 3) / 4 * 4, PW = pw64(pkind, D);
  double y[ARBX_MAX_DIM];
  for (int a = 0; a < D; ++a) y[a] = qpoints[qi * D + a];
  Heap64 heap;
  heap.init(k);
  int32_t sref[STACK_DEPTH];
  double sbound[STACK_DEPTH];
  int sp = 0;
  constexpr int32_t DONE = INT32_MIN;
  int32_t ref = *root;
  while (ref != DONE) {
    if (ref >= 0) {
      const float* nd = nodes + (int64_t)ref * NW;
      double b0 = box_bound64(y, nd, nd + D, D), b1 = box_bound64(y, nd + 2 * D, nd + 3 * D, D);
      int32_t c0 = __float_as_int(nd[4 * D]), c1 = __float_as_int(nd[4 * D + 1]);
      if (b1 < b0) { const double tb = b0; b0 = b1; b1 = tb; const int32_t tc = c0; c0 = c1; c1 = tc; }
      const double w = heap.worst();
      if (b0 < w) {
        ref = c0;
        if (b1 < w) { sref[sp] = c1; sbound[sp] = b1; ++sp; }
        continue;
      }
    } else {
      for (int64_t j = ~ref;; ++j) {
        const float* lf = leaves + j * LW;
        const uint32_t tag = __float_as_uint(lf[2 * D]);
        const double key = knn_dist64(y, rows64 + j * PW, pkind, D);
        if (key < heap.worst()) heap.push(key, (int32_t)(tag & ~LEAF_END));
        if (tag & LEAF_END) break;
      }
    }
    ref = DONE;
    while (sp > 0) {
      --sp;
      if (sbound[sp] < heap.worst()) { ref = sref[sp]; break; }
    }
  }
  // heap sort: largest to the back, then rows ascending; padding when fewer than k primitives
  for (int size = heap.m; size > 1; --size) {
    const double td = heap.d[size - 1]; const int32_t ti = heap.i[size - 1];
    heap.d[size - 1] = heap.d[0]; heap.i[size - 1] = heap.i[0];
    heap.sift_down(0, size - 1, td, ti);
  }
  for (int s = 0; s < k; ++s) {
    indices[qi * k + s] = s < heap.m ? heap.i[s] : -1;
    if (distances) distances[qi * k + s] = s < heap.m ? heap.d[s] : INFINITY;
  }
}

}  // namespace

// ---- host entry points (called from api.cu) --------------------------------------------------------
arbx_status f64_build(const double* prims, int64_t n, int dim, int kind, cudaStream_t s, Index* ix) {
  Scratch<float> boxes;
  ARBX_TRY(boxes.alloc((size_t)std::max<int64_t>(n, 1) * 2 * dim, s));
  const unsigned grid = (unsigned)((n + FT - 1) / FT);
  if (n > 0) {
    f64_boxes_kernel<<<grid, FT, 0, s>>>(prims, n, dim, kind, boxes.p);
    ARBX_LAUNCH_CHECK();
  }
  ARBX_TRY(build_index(boxes.p, n, dim, KIND_BOX, s, ix));
  ix->f64 = true;
  ix->kind64 = kind;
  if (n == 0) return ARBX_OK;
  ARBX_TRY(scratch_alloc((void**)&ix->rows64, (size_t)n * pw64(kind, dim) * sizeof(double), s));
  f64_gather_kernel<<<grid, FT, 0, s>>>(prims, ix->leaves, n, dim, kind, leaf_width(KIND_BOX, dim), ix->rows64);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

arbx_status f64_qboxes(const double* queries, int64_t nq, int dim, int qkind, float* qboxes, cudaStream_t s) {
  f64_qboxes_kernel<<<(unsigned)((nq + FT - 1) / FT), FT, 0, s>>>(queries, nq, dim, qkind, qboxes);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

arbx_status f64_spatial(const Index* ix, const double* queries, const float* qboxes, const uint32_t* qorder, int64_t nq,
                        int qkind, int32_t* counts, const int32_t* offsets, int32_t* indices, int fill, cudaStream_t s) {
  ProfScope ps(fill ? K_SPATIAL_FILL : K_SPATIAL_COUNT, s);
  f64_spatial_kernel<<<(unsigned)((nq + FT - 1) / FT), FT, 0, s>>>(ix->nodes, ix->leaves, ix->rows64, ix->root, ix->dim,
                                                                   ix->kind64, queries, qboxes, qorder, nq, qkind, counts,
                                                                   offsets, indices, fill);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

arbx_status f64_knn(const Index* ix, const double* qpoints, const uint32_t* qorder, int64_t nq, int k, int32_t* indices,
                    double* distances, cudaStream_t s) {
  ProfScope ps(K_KNN, s);
  f64_knn_kernel<<<(unsigned)((nq + FT - 1) / FT), FT, 0, s>>>(ix->nodes, ix->leaves, ix->rows64, ix->root, ix->dim,
                                                               ix->kind64, qpoints, qorder, nq, k, indices, distances);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

}  // namespace arbx
