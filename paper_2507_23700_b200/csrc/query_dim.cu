// query_dim.cu -- compiled once per dimension (-DARBX_DIM=1..10): query steps Q1 (query codes),
// T1/T3 (spatial traversal: count / fill) and K1/K2 (kNN traversal + emit).  SURVEY.md §8(a).
// PAPER.md:L69 (radius / nearest predicates), L79 (nearest = distance to the stored geometry),
// L104-115 (callback / storage queries), L295 + L307 (traversal, sorted queries), L303 (count).
//
// Also the traversal forms of the NEXT items: capped count / capped fill (early exit), the
// self-join (SELF: half traversal over the index's own leaves) and the DBSCAN edge callback
// (MODE 3).
//
// The 32 queries of a warp are neighbours on the space-filling curve (qorder).  Spatial
// queries pick, per warp, a warp-cooperative packet traversal (coherent queries) or one
// independent traversal per lane; kNN runs one traversal per lane.
#include <algorithm>
#include <cstdlib>
#include <cstdint>
#include <type_traits>

#include "geom.cuh"

#ifndef ARBX_DIM
#error "compile with -DARBX_DIM=<1..10>"
#endif

namespace arbx {
namespace {

constexpr int D = ARBX_DIM;
constexpr int QT = 64;    // threads per block of the traversal kernels (64 measured ~1% faster than 128)

// ---- Q1: 32-bit space-filling code of each query centre inside the scene bounds --------------
template <int QK>
__global__ void __launch_bounds__(256) qcode_kernel(const float* __restrict__ queries, int64_t nq,
                                                    const float* __restrict__ bounds,
                                                    uint32_t* __restrict__ codes, int drop) {
  constexpr int QW = prim_width(QK, D);
  constexpr int B = qcode_bits_per_axis(D);
  float lo[D], scale[D];
#pragma unroll
  for (int a = 0; a < D; ++a) {
    lo[a] = bounds[a];
    float ext = bounds[D + a] - lo[a];
    scale[a] = ext > 0.f ? exp2f((float)B) / ext : 0.f;
  }
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < nq; i += (int64_t)gridDim.x * 256) {
    float v[QW], c[D];
#pragma unroll
    for (int e = 0; e < QW; ++e) v[e] = __ldg(queries + i * QW + e);
    centre_of<D, QK>(v, c);
    uint32_t q[D];
    quantise<D, B>(c, lo, scale, q);
    codes[i] = interleave<D, B, uint32_t>(q) >> drop;
  }
}

// ---- node / leaf access ------------------------------------------------------------------------
struct Node { float v[4 * D]; int32_t c0, c1; };

__device__ __forceinline__ void load_node(const float4* __restrict__ nodes, int32_t ref, Node& nd) {
  const float4* p = nodes + (int64_t)ref * (D + 1);
#pragma unroll
  for (int e = 0; e < D; ++e) {
    float4 t = __ldg(p + e);
    nd.v[4 * e] = t.x; nd.v[4 * e + 1] = t.y; nd.v[4 * e + 2] = t.z; nd.v[4 * e + 3] = t.w;
  }
  float4 t = __ldg(p + D);
  nd.c0 = __float_as_int(t.x);
  nd.c1 = __float_as_int(t.y);
}

template <int PK>
struct Leaf { float v[prim_width(PK, D)]; uint32_t idx; };

template <int PK>
__device__ __forceinline__ void load_leaf(const float4* __restrict__ leaves, int j, Leaf<PK>& lf) {
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
  float t[LW];
  const float4* p = leaves + (int64_t)j * (LW / 4);
#pragma unroll
  for (int e = 0; e < LW / 4; ++e) {
    float4 x = __ldg(p + e);
    t[4 * e] = x.x; t[4 * e + 1] = x.y; t[4 * e + 2] = x.z; t[4 * e + 3] = x.w;
  }
#pragma unroll
  for (int e = 0; e < W; ++e) lf.v[e] = t[e];
  lf.idx = __float_as_uint(t[W]);
}

// ---- spatial predicates (closed sets) ---------------------------------
template <int QK>
struct Query {
  float v[prim_width(QK, D)];
  float r2;   // SPHERE: r*r
};

template <int QK>
__device__ __forceinline__ bool hits_box(const Query<QK>& q, const float* lo, const float* hi) {
  if constexpr (QK == KIND_SPHERE) {
    return dist2_pb<D>(q.v, lo, hi) <= q.r2;
  } else if constexpr (QK == KIND_BOX) {
    bool ok = true;
#pragma unroll
    for (int a = 0; a < D; ++a) ok = ok && lo[a] <= q.v[D + a] && q.v[a] <= hi[a];
    return ok;
  } else {
    bool ok = true;
#pragma unroll
    for (int a = 0; a < D; ++a) ok = ok && lo[a] <= q.v[a] && q.v[a] <= hi[a];
    return ok;
  }
}

template <int QK, int PK>
__device__ __forceinline__ bool hits_prim(const Query<QK>& q, const float* p) {
  if constexpr (PK == KIND_BOX) {
    return hits_box<QK>(q, p, p + D);
  } else if constexpr (PK == KIND_POINT) {
    if constexpr (QK == KIND_SPHERE) {
      return dist2_pp<D>(p, q.v) <= q.r2;
    } else if constexpr (QK == KIND_BOX) {
      bool ok = true;
#pragma unroll
      for (int a = 0; a < D; ++a) ok = ok && q.v[a] <= p[a] && p[a] <= q.v[D + a];
      return ok;
    } else {
      bool ok = true;
#pragma unroll
      for (int a = 0; a < D; ++a) ok = ok && p[a] == q.v[a];
      return ok;
    }
  } else {   // SPHERE primitive (c, R)
    const float R = p[D];
    if constexpr (QK == KIND_SPHERE) {
      const float rr = q.v[D] + R;
      return dist2_pp<D>(p, q.v) <= rr * rr;
    } else if constexpr (QK == KIND_BOX) {
      return dist2_pb<D>(p, q.v, q.v + D) <= R * R;
    } else {
      return dist2_pp<D>(q.v, p) <= R * R;
    }
  }
}

// ---- T1 / T3: spatial traversal ------------------------------------------------------------------
// Warp-cooperative ("packet") traversal.  A warp owns 32 queries that are neighbours on the
// space-filling curve and walks the tree ONCE for all of them: every lane tests its own query
// against the two child boxes of the current node, the warp descends where ANY lane hits.
// All lanes fetch the same node / leaf record, so a fetch is one broadcast L1 transaction
// instead of 32 divergent ones, control flow is uniform, and the stack is one short array
// per warp in shared memory.  The leaf test is per lane and exact, so the result is the same
// set as one-query-per-thread traversal.
// ---- DBSCAN edge callback (MODE 3): lock-free union-find over the core points ------------------
// uf[i] = i at start for core points, -1 for the others.  Core-core edges are united (the
// larger root is hooked under the smaller with atomicCAS, finds use path halving); a non-core
// point next to a core point remembers ONE such core point as -2 - core (first writer wins).
#ifndef ARBX_UF_HELPERS
#define ARBX_UF_HELPERS
__device__ __forceinline__ int32_t uf_find(int32_t* uf, int32_t x) {
  for (;;) {
    const int32_t p = ((volatile int32_t*)uf)[x];
    if (p == x) return x;
    const int32_t gp = ((volatile int32_t*)uf)[p];
    if (gp != p) uf[x] = gp;     // path halving; roots only ever decrease, so a stale write is harmless
    x = p;
  }
}
__device__ __forceinline__ void uf_union(int32_t* uf, int32_t a, int32_t b) {
  for (;;) {
    a = uf_find(uf, a);
    b = uf_find(uf, b);
    if (a == b) return;
    if (a < b) { const int32_t t = a; a = b; b = t; }       // hook the larger root a under b
    if (atomicCAS(uf + a, a, b) == a) return;
  }
}
__device__ __forceinline__ void dbscan_edge(int32_t* uf, const int32_t* counts, int min_pts, int32_t i, int32_t j) {
  const bool ci = counts[i] >= min_pts, cj = counts[j] >= min_pts;
  if (ci && cj) uf_union(uf, i, j);
  else if (ci) atomicCAS(uf + j, -1, -2 - i);
  else if (cj) atomicCAS(uf + i, -1, -2 - j);
}
#endif

struct NodeX { float v[4 * D]; int32_t c0, c1, l, r; };

__device__ __forceinline__ void load_node_x(const float4* __restrict__ nodes, int32_t ref, NodeX& nd) {
  const float4* p = nodes + (int64_t)ref * (D + 1);
#pragma unroll
  for (int e = 0; e < D; ++e) {
    float4 t = __ldg(p + e);
    nd.v[4 * e] = t.x; nd.v[4 * e + 1] = t.y; nd.v[4 * e + 2] = t.z; nd.v[4 * e + 3] = t.w;
  }
  float4 t = __ldg(p + D);
  nd.c0 = __float_as_int(t.x); nd.c1 = __float_as_int(t.y);
  nd.l = __float_as_int(t.z); nd.r = __float_as_int(t.w);
}

// SELF (self-join, queries = the index's own primitives in tree order): query number `tpos` is
// the leaf at sorted position tpos; only primitives at LATER positions are reported, so every
// unordered pair appears once, and subtrees that end at or before tpos are skipped.
template <int PK, int QK, int MODE, bool SELF>
__device__ __forceinline__ int thread_traverse(const float4* __restrict__ nodes, const float4* __restrict__ leaves,
                                               const int32_t* __restrict__ root, const Query<QK>& q,
                                               int32_t* __restrict__ out, int limit, int stop, int tpos,
                                               const int32_t* __restrict__ counts, int min_pts, int32_t qi) {
  constexpr bool FILL = MODE == 1 || MODE == 2;
  // Node work and leaf work are separated: a lane that reaches a leaf range does not stop and
  // wait for the other lanes (measured on C5: the node loop then runs at 5 of 32 lanes), it
  // queues the range and keeps walking nodes until its stack is empty or its queue is full;
  // then all lanes scan their queued ranges together.
  constexpr int LQ = 32;
  int cnt = 0;
  int32_t stack[STACK_DEPTH];
  int32_t lq[LQ];
  int sp = 0, nl = 0;
  constexpr int32_t DONE = INT32_MIN;
  int32_t ref = __ldg(root);
  for (;;) {
    while (ref != DONE && nl < LQ) {
      if (ref < 0) {
        lq[nl++] = ref;
        ref = sp > 0 ? stack[--sp] : DONE;
        continue;
      }
      NodeX nd;
      load_node_x(nodes, ref, nd);
      bool h0 = hits_box<QK>(q, nd.v, nd.v + D);
      bool h1 = hits_box<QK>(q, nd.v + 2 * D, nd.v + 3 * D);
      if constexpr (SELF) { h0 = h0 && ref > tpos; h1 = h1 && nd.r > tpos; }   // child ranges [l,ref], [ref+1,r]
      if (h0) {
        ref = nd.c0;
        if (h1) stack[sp++] = nd.c1;
      } else if (h1) {
        ref = nd.c1;
      } else {
        ref = sp > 0 ? stack[--sp] : DONE;
      }
    }
    for (int e = 0; e < nl; ++e) {
      int j = ~lq[e];
      for (;; ++j) {
        Leaf<PK> lf;
        load_leaf<PK>(leaves, j, lf);
        if ((!SELF || j > tpos) && hits_prim<QK, PK>(q, lf.v)) {
          if constexpr (FILL) { if (cnt < limit) out[cnt] = (int32_t)(lf.idx & ~LEAF_END); }
          if constexpr (MODE == 3) dbscan_edge(out, counts, min_pts, qi, (int32_t)(lf.idx & ~LEAF_END));
          ++cnt;
          if (cnt >= stop) return cnt;   // capped query: early exit
        }
        if (lf.idx & LEAF_END) break;
      }
    }
    nl = 0;
    if (ref == DONE) break;
  }
  return cnt;
}

// Are the 32 queries of this warp close together compared with their own reach?  Per axis:
// spread of the query centres <= alpha * (largest query extent).  Coherent warps take the
// packet path, the others traverse independently (one query per lane).  Warp-uniform result.
template <int QK>
__device__ __forceinline__ bool warp_coherent(const Query<QK>& q, bool valid, float alpha) {
  if constexpr (QK == KIND_POINT) {
    return false;
  } else {
    bool ok = true;
#pragma unroll
    for (int a = 0; a < D; ++a) {
      const float c = QK == KIND_BOX ? 0.5f * q.v[a] + 0.5f * q.v[D + a] : q.v[a];
      const float ext = QK == KIND_BOX ? q.v[D + a] - q.v[a] : 2.f * q.v[D];
      float lo = valid ? c : INFINITY, hi = valid ? c : -INFINITY, e = valid ? ext : 0.f;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(~0u, lo, o));
        hi = fmaxf(hi, __shfl_xor_sync(~0u, hi, o));
        e = fmaxf(e, __shfl_xor_sync(~0u, e, o));
      }
      ok = ok && (hi - lo <= alpha * e);
    }
    return ok;
  }
}

// Joint region of the (coherent) queries of a warp: the box [lo,hi] of the query centres /
// query boxes and the largest radius.  joint_hits_prim is true whenever ANY lane's exact
// hits_prim can be true (same monotone fp32 operation sequences), so it is used to discard
// the primitives of a leaf range 32 at a time, one per lane, before the exact per-lane tests.
template <int QK>
struct Joint { float lo[D], hi[D]; float r, r2; };

template <int QK>
__device__ __forceinline__ void joint_of_warp(const Query<QK>& q, bool alive, Joint<QK>& J) {
#pragma unroll
  for (int a = 0; a < D; ++a) {
    float lo = alive ? q.v[a] : INFINITY;
    float hi = alive ? (QK == KIND_BOX ? q.v[D + a] : q.v[a]) : -INFINITY;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = fminf(lo, __shfl_xor_sync(~0u, lo, o));
      hi = fmaxf(hi, __shfl_xor_sync(~0u, hi, o));
    }
    J.lo[a] = lo; J.hi[a] = hi;
  }
  J.r = 0.f; J.r2 = 0.f;
  if constexpr (QK == KIND_SPHERE) {
    float r = alive ? q.v[D] : 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r = fmaxf(r, __shfl_xor_sync(~0u, r, o));
    J.r = r; J.r2 = r * r;
  }
}

template <int D_>
__device__ __forceinline__ float dist2_bb(const float* alo, const float* ahi, const float* blo, const float* bhi) {
  float s = 0.f;
#pragma unroll
  for (int a = 0; a < D_; ++a) {
    float d = fmaxf(0.f, fmaxf(alo[a] - bhi[a], blo[a] - ahi[a]));
    s = fmaf(d, d, s);
  }
  return s;
}

template <int QK, int PK>
__device__ __forceinline__ bool joint_hits_prim(const Joint<QK>& J, const float* p) {
  if constexpr (QK == KIND_SPHERE) {
    if constexpr (PK == KIND_POINT) return dist2_pb<D>(p, J.lo, J.hi) <= J.r2;
    else if constexpr (PK == KIND_BOX) return dist2_bb<D>(p, p + D, J.lo, J.hi) <= J.r2;
    else { const float rr = J.r + p[D]; return dist2_pb<D>(p, J.lo, J.hi) <= rr * rr; }
  } else {   // BOX queries: J is the union box
    if constexpr (PK == KIND_SPHERE) {
      return dist2_pb<D>(p, J.lo, J.hi) <= p[D] * p[D];
    } else {
      bool ok = true;
#pragma unroll
      for (int a = 0; a < D; ++a) ok = ok && p[a] <= J.hi[a] && J.lo[a] <= (PK == KIND_BOX ? p[D + a] : p[a]);
      return ok;
    }
  }
}

template <int QK>
__device__ __forceinline__ bool joint_hits_box(const Joint<QK>& J, const float* lo, const float* hi) {
  if constexpr (QK == KIND_SPHERE) {
    return dist2_bb<D>(lo, hi, J.lo, J.hi) <= J.r2;
  } else {
    bool ok = true;
#pragma unroll
    for (int a = 0; a < D; ++a) ok = ok && lo[a] <= J.hi[a] && J.lo[a] <= hi[a];
    return ok;
  }
}

// MODE 0: count.  MODE 1: fill the CSR slices (offsets known); with cap > 0 the queries whose
// count is <= cap are skipped (their rows were stored by MODE 2 and are copied by
// compact_rows).  MODE 2: count AND store the first `cap` hits of query q in rows[q*cap ..].
template <int PK, int QK, int MODE, bool SELF>
__global__ void __launch_bounds__(QT) spatial_kernel(const float4* __restrict__ nodes,
                                                     const float4* __restrict__ leaves,
                                                     const int32_t* __restrict__ root, int n,
                                                     const float* __restrict__ queries,
                                                     const uint32_t* __restrict__ qorder, int64_t nq,
                                                     int32_t* __restrict__ counts,
                                                     const int32_t* __restrict__ offsets,
                                                     int32_t* __restrict__ indices, int cap,
                                                     int* __restrict__ overflow, uint32_t* __restrict__ ovf_list,
                                                     int stop_fill, int mode, float alpha) {
  constexpr bool FILL = MODE == 1 || MODE == 2;     // hits are written to rows / CSR slices
  constexpr int QW = prim_width(QK, D);
  constexpr int PQ_CAP = 320;   // packet work list (node ids) per warp
  __shared__ int32_t s_stack[QT / 32][PQ_CAP];
  int32_t* stack = s_stack[threadIdx.x >> 5];
  const int64_t t = (int64_t)blockIdx.x * QT + threadIdx.x;
  const bool valid = t < nq;
  const int64_t qi = valid ? (qorder ? (int64_t)qorder[t] : t) : 0;
  bool alive = valid;
  if constexpr (MODE == 1) {   // rows that were stored are copied, not traversed again
    if (cap > 0) {
      alive = alive && counts[qi] > cap;
      if (!__any_sync(~0u, alive)) return;
    }
  }
  Query<QK> q;
#pragma unroll
  for (int e = 0; e < QW; ++e) q.v[e] = __ldg(queries + qi * QW + e);
  if constexpr (QK == KIND_SPHERE) {
    q.r2 = q.v[D] * q.v[D];
    alive = alive && q.v[D] >= 0.f;      // negative radius matches nothing (reading A21)
  }
  int64_t base64 = 0;   // where this query's hits go in `indices` (MODE 1: CSR slice, MODE 2: row q*cap)
  int limit = INT32_MAX;
  bool capped = false;   // this lane stops after `limit` hits (capped count / capped fill)
  if constexpr (MODE == 1) {
    base64 = valid ? offsets[qi] : 0;
    if (stop_fill) {     // capped storage query: write exactly the counted number of hits
      limit = valid ? counts[qi] : 0;
      alive = alive && limit > 0;
      capped = true;
      if (!__any_sync(~0u, alive)) return;
    }
  }
  if constexpr (MODE == 2) { base64 = qi * cap; limit = cap; }
  if constexpr (MODE == 0) { if (cap > 0) { limit = cap; capped = true; } }   // arbx_query_count_upto
  // mode 0: per-warp choice; 1: always one query per lane; 2: always packet
  if (mode == 1 || (mode == 0 && !warp_coherent<QK>(q, valid, alpha))) {
    int c = 0;
    if (alive) c = thread_traverse<PK, QK, MODE, SELF>(nodes, leaves, root, q,
                                                       MODE == 3 ? indices : FILL ? indices + base64 : nullptr, limit,
                                                       capped ? limit : INT32_MAX, (int)t, counts, cap, (int32_t)qi);
    if constexpr (MODE == 0 || MODE == 2) {
      if (valid) counts[qi] = c;
      if constexpr (MODE == 2) { if (c > cap) ovf_list[atomicAdd(overflow, 1)] = (uint32_t)qi; }
    }
    return;
  }
  // FILL: hits are staged per lane in shared memory (FS slots, column `lane` of a padded
  // [FS][33] array) and flushed row by row with all lanes writing one query's pending hits as
  // one contiguous run, instead of one scattered 4-byte store per hit.
  constexpr int FS = 16;
  __shared__ int32_t s_stage[FILL ? QT / 32 : 1][FILL ? FS * 33 : 1];
  int32_t* stage = s_stage[FILL ? (threadIdx.x >> 5) : 0];
  const int lane = threadIdx.x & 31;
  int64_t base = base64;   // FILL: position in `indices` of this query's next unflushed hit
  int cnt = 0, pend = 0;

  auto flush = [&](uint32_t who) {   // who: lanes whose pending hits are written out (warp-uniform)
    __syncwarp();
    while (who) {
      const int L = __ffs(who) - 1;
      who &= who - 1;
      const int m = __shfl_sync(~0u, pend, L);
      const int64_t b = __shfl_sync(~0u, base, L);
      if (lane < m) indices[b + lane] = stage[lane * 33 + L];
      if (lane == L) { base += pend; pend = 0; }
    }
    __syncwarp();
  };

  // Leaf ranges: lane j first tests primitive j against the warp's JOINT region (one
  // coalesced load, 32 primitives at a time); only the survivors are broadcast to all lanes
  // for the exact per-lane test.
  Joint<QK> J;
  joint_of_warp<QK>(q, alive, J);
  auto leaf_range = [&](int first, int m) {   // m is warp-uniform
    for (int j0 = 0; j0 < m; j0 += 32) {
      bool in = false;
      if (j0 + lane < m) {
        Leaf<PK> mine;
        load_leaf<PK>(leaves, first + j0 + lane, mine);
        in = joint_hits_prim<QK, PK>(J, mine.v);
      }
      uint32_t todo = __ballot_sync(~0u, in);
      while (todo) {
        const int b = __ffs(todo) - 1;
        todo &= todo - 1;
        Leaf<PK> lf;
        load_leaf<PK>(leaves, first + j0 + b, lf);
        const bool hit = alive && (!SELF || first + j0 + b > (int)t) && hits_prim<QK, PK>(q, lf.v);
        if constexpr (FILL) {
          const uint32_t full = __ballot_sync(~0u, pend == FS);
          if (full) flush(full);
          if (hit) {
            if (cnt < limit) { stage[pend * 33 + lane] = (int32_t)(lf.idx & ~LEAF_END); ++pend; }
            ++cnt;
          }
        } else if constexpr (MODE == 3) {
          if (hit) dbscan_edge(indices, counts, cap, (int32_t)qi, (int32_t)(lf.idx & ~LEAF_END));
        } else {
          cnt += hit ? 1 : 0;
        }
      }
    }
    if (capped && cnt >= limit) alive = false;   // capped query: this lane has seen enough
  };

  // Node work is spread over the lanes: the warp keeps a work list of node ids in shared
  // memory, pops up to 32 of them, and lane i tests the two child boxes of node i against the
  // JOINT region.  Hit leaf-range children are scanned on the spot (warp-uniform loop over the
  // ballot), hit internal children are compacted back onto the list.  When the list runs
  // close to its capacity the warp pops one node at a time, which bounds growth by the tree depth.
  if (__any_sync(~0u, alive)) {
    const int32_t rootref = __ldg(root);
    if (rootref < 0) {
      leaf_range(0, n);
    } else {
      const uint32_t lt = (1u << lane) - 1u;
      // Upper tree: while only ONE child of the current node can hold a match, and it is an
      // internal node, there is nothing to spread over the lanes: the warp steps down that
      // single path (every lane does the same two box tests on a broadcast node) and the work
      // list starts below it.
      int32_t top = rootref;
      for (;;) {
        NodeX nd;
        load_node_x(nodes, top, nd);
        bool h0 = joint_hits_box<QK>(J, nd.v, nd.v + D);
        bool h1 = joint_hits_box<QK>(J, nd.v + 2 * D, nd.v + 3 * D);
        if constexpr (SELF) {
          const int tmin = (int)(t - lane);
          h0 = h0 && top > tmin; h1 = h1 && nd.r > tmin;
        }
        if (h0 && !h1 && nd.c0 >= 0) top = nd.c0;
        else if (h1 && !h0 && nd.c1 >= 0) top = nd.c1;
        else break;
      }
      int nlist = 1;
      stack[0] = top;
      __syncwarp();
      while (nlist > 0) {
        const int take = nlist > PQ_CAP - STACK_DEPTH - 64 ? 1 : min(32, nlist);
        nlist -= take;
        const int32_t my = lane < take ? stack[nlist + lane] : -1;
        __syncwarp();
        NodeX nd;
        bool in0 = false, in1 = false, lf0 = false, lf1 = false;
        if (my >= 0) {
          load_node_x(nodes, my, nd);
          bool h0 = joint_hits_box<QK>(J, nd.v, nd.v + D);
          bool h1 = joint_hits_box<QK>(J, nd.v + 2 * D, nd.v + 3 * D);
          if constexpr (SELF) {   // the warp's smallest query position is its first lane's
            const int tmin = (int)(t - lane);
            h0 = h0 && my > tmin; h1 = h1 && nd.r > tmin;
          }
          in0 = h0 && nd.c0 >= 0; lf0 = h0 && nd.c0 < 0;
          in1 = h1 && nd.c1 >= 0; lf1 = h1 && nd.c1 < 0;
        }
        uint32_t m0 = __ballot_sync(~0u, lf0), m1 = __ballot_sync(~0u, lf1);
        while (m0) {
          const int b = __ffs(m0) - 1;
          m0 &= m0 - 1;
          const int l = __shfl_sync(~0u, nd.l, b), p = __shfl_sync(~0u, my, b);
          leaf_range(l, p - l + 1);
        }
        while (m1) {
          const int b = __ffs(m1) - 1;
          m1 &= m1 - 1;
          const int r = __shfl_sync(~0u, nd.r, b), p = __shfl_sync(~0u, my, b);
          leaf_range(p + 1, r - p);
        }
        if (capped && !__any_sync(~0u, alive)) break;
        const uint32_t b0 = __ballot_sync(~0u, in0), b1 = __ballot_sync(~0u, in1);
        if (in0) stack[nlist + __popc(b0 & lt)] = nd.c0;
        if (in1) stack[nlist + __popc(b0) + __popc(b1 & lt)] = nd.c1;
        nlist += __popc(b0) + __popc(b1);
        __syncwarp();
      }
    }
  }
  if constexpr (FILL) flush(__ballot_sync(~0u, pend > 0));
  if constexpr (MODE == 0 || MODE == 2) {
    if (valid) counts[qi] = MODE == 0 ? min(cnt, limit) : cnt;
    if constexpr (MODE == 2) { if (cnt > cap) ovf_list[atomicAdd(overflow, 1)] = (uint32_t)qi; }   // valid: cnt > 0
  }
}

// Fill pass for the queries whose row overflowed the stored `cap` hits (list `qlist`, built by
// MODE 2): ONE WARP PER QUERY.  These are the long rows (hundreds of hits), and a lane walking
// such a row alone is pure latency (measured: C5 1.3 ms, C4 0.35 ms for a few thousand queries).
// Here lane i tests the child boxes of node i of a shared-memory work list against the query
// itself, the primitives of a hit leaf range are tested one per lane, and the hits of a step
// leave as one ballot-compacted run into the query's CSR slice.
template <int PK, int QK>
__global__ void __launch_bounds__(QT) spatial_heavy_kernel(const float4* __restrict__ nodes,
                                                           const float4* __restrict__ leaves,
                                                           const int32_t* __restrict__ root, int n,
                                                           const float* __restrict__ queries,
                                                           const uint32_t* __restrict__ qlist, int64_t nlistq,
                                                           const int32_t* __restrict__ offsets,
                                                           int32_t* __restrict__ indices) {
  constexpr int QW = prim_width(QK, D);
  constexpr int PQ_CAP = 320;
  __shared__ int32_t s_stack[QT / 32][PQ_CAP];
  int32_t* stack = s_stack[threadIdx.x >> 5];
  const int lane = threadIdx.x & 31;
  const int64_t wq = ((int64_t)blockIdx.x * QT + threadIdx.x) >> 5;
  if (wq >= nlistq) return;
  const int64_t qi = qlist[wq];
  Query<QK> q;
#pragma unroll
  for (int e = 0; e < QW; ++e) q.v[e] = __ldg(queries + qi * QW + e);
  if constexpr (QK == KIND_SPHERE) q.r2 = q.v[D] * q.v[D];
  int64_t base = offsets[qi];
  const uint32_t lt = (1u << lane) - 1u;
  auto leaf_range = [&](int first, int m) {   // m is warp-uniform
    for (int j0 = 0; j0 < m; j0 += 32) {
      bool hit = false;
      uint32_t idx = 0;
      if (j0 + lane < m) {
        Leaf<PK> lf;
        load_leaf<PK>(leaves, first + j0 + lane, lf);
        hit = hits_prim<QK, PK>(q, lf.v);
        idx = lf.idx & ~LEAF_END;
      }
      const uint32_t bal = __ballot_sync(~0u, hit);
      if (hit) indices[base + __popc(bal & lt)] = (int32_t)idx;
      base += __popc(bal);
    }
  };
  const int32_t rootref = __ldg(root);
  if (rootref < 0) { leaf_range(0, n); return; }
  int nlist = 1;
  stack[0] = rootref;
  __syncwarp();
  while (nlist > 0) {
    const int take = nlist > PQ_CAP - STACK_DEPTH - 64 ? 1 : min(32, nlist);
    nlist -= take;
    const int32_t my = lane < take ? stack[nlist + lane] : -1;
    __syncwarp();
    NodeX nd;
    bool in0 = false, in1 = false, lf0 = false, lf1 = false;
    if (my >= 0) {
      load_node_x(nodes, my, nd);
      const bool h0 = hits_box<QK>(q, nd.v, nd.v + D);
      const bool h1 = hits_box<QK>(q, nd.v + 2 * D, nd.v + 3 * D);
      in0 = h0 && nd.c0 >= 0; lf0 = h0 && nd.c0 < 0;
      in1 = h1 && nd.c1 >= 0; lf1 = h1 && nd.c1 < 0;
    }
    uint32_t m0 = __ballot_sync(~0u, lf0), m1 = __ballot_sync(~0u, lf1);
    while (m0) {
      const int b = __ffs(m0) - 1;
      m0 &= m0 - 1;
      const int l = __shfl_sync(~0u, nd.l, b), p = __shfl_sync(~0u, my, b);
      leaf_range(l, p - l + 1);
    }
    while (m1) {
      const int b = __ffs(m1) - 1;
      m1 &= m1 - 1;
      const int r = __shfl_sync(~0u, nd.r, b), p = __shfl_sync(~0u, my, b);
      leaf_range(p + 1, r - p);
    }
    const uint32_t b0 = __ballot_sync(~0u, in0), b1 = __ballot_sync(~0u, in1);
    if (in0) stack[nlist + __popc(b0 & lt)] = nd.c0;
    if (in1) stack[nlist + __popc(b0) + __popc(b1 & lt)] = nd.c1;
    nlist += __popc(b0) + __popc(b1);
    __syncwarp();
  }
}

// ---- K1 / K2: k nearest neighbours ------------------------------------------------------------------
// Heap key: squared distance for POINT/BOX primitives, distance for SPHERE primitives
// (max(0,||y-c||-R) is not monotone in the squared centre distance alone).
template <int PK>
__device__ __forceinline__ float knn_key(const float* y, const float* p) {
  if constexpr (PK == KIND_POINT) return dist2_pp<D>(p, y);
  else if constexpr (PK == KIND_BOX) return dist2_pb<D>(y, p, p + D);
  else return fmaxf(0.f, sqrtf(dist2_pp<D>(p, y)) - p[D]);
}
template <int PK>
__device__ __forceinline__ float knn_bound(const float* y, const float* lo, const float* hi) {
  const float d2 = dist2_pb<D>(y, lo, hi);
  if constexpr (PK == KIND_SPHERE) return sqrtf(d2);
  else return d2;
}

// Best-k container, KB > 0: ascending sorted array in registers (all indices static).  Slots
// [0, KB-k) hold -inf sentinels so that the k-th best is always slot KB-1.
template <int KB>
struct RegHeap {
  float d[KB];
  int32_t i[KB];
  __device__ __forceinline__ void init(int k) {
#pragma unroll
    for (int s = 0; s < KB; ++s) { d[s] = s < KB - k ? -INFINITY : INFINITY; i[s] = -1; }
  }
  __device__ __forceinline__ float worst() const { return d[KB - 1]; }
  __device__ __forceinline__ void push(float t, int32_t idx) {   // requires t < worst()
    if constexpr (KB >= 16) {
      constexpr int H = KB / 2;
      if (t >= d[H - 1]) {      // lands in the upper half: the lower half is untouched
        d[KB - 1] = t; i[KB - 1] = idx;
#pragma unroll
        for (int s = KB - 1; s > H; --s) {
          const bool sw = d[s] < d[s - 1];
          const float td = d[s]; const int32_t ti = i[s];
          d[s] = sw ? d[s - 1] : td; i[s] = sw ? i[s - 1] : ti;
          d[s - 1] = sw ? td : d[s - 1]; i[s - 1] = sw ? ti : i[s - 1];
        }
        return;
      }
#pragma unroll
      for (int s = KB - 1; s >= H; --s) { d[s] = d[s - 1]; i[s] = i[s - 1]; }   // upper half moves up by one
      d[H - 1] = t; i[H - 1] = idx;
#pragma unroll
      for (int s = H - 1; s > 0; --s) {
        const bool sw = d[s] < d[s - 1];
        const float td = d[s]; const int32_t ti = i[s];
        d[s] = sw ? d[s - 1] : td; i[s] = sw ? i[s - 1] : ti;
        d[s - 1] = sw ? td : d[s - 1]; i[s - 1] = sw ? ti : i[s - 1];
      }
      return;
    }
    d[KB - 1] = t; i[KB - 1] = idx;
#pragma unroll
    for (int s = KB - 1; s > 0; --s) {
      const bool sw = d[s] < d[s - 1];
      const float td = d[s]; const int32_t ti = i[s];
      d[s] = sw ? d[s - 1] : td; i[s] = sw ? i[s - 1] : ti;
      d[s - 1] = sw ? td : d[s - 1]; i[s - 1] = sw ? ti : i[s - 1];
    }
  }
  // the same insertion as one straight compare-exchange chain: when the whole warp executes it
  // (packet kNN) the two branches of push() would both run
  __device__ __forceinline__ void push_uniform(float t, int32_t idx) {   // requires t < worst()
    d[KB - 1] = t; i[KB - 1] = idx;
#pragma unroll
    for (int s = KB - 1; s > 0; --s) {
      const bool sw = d[s] < d[s - 1];
      const float td = d[s]; const int32_t ti = i[s];
      d[s] = sw ? d[s - 1] : td; i[s] = sw ? i[s - 1] : ti;
      d[s - 1] = sw ? td : d[s - 1]; i[s - 1] = sw ? ti : i[s - 1];
    }
  }
  template <class F>
  __device__ __forceinline__ void emit(int k, F&& f) {
#pragma unroll
    for (int s = 0; s < KB; ++s)
      if (s >= KB - k) f(s - (KB - k), d[s], i[s]);
  }
  // k == KB and KB % 4 == 0: the row is 16-byte aligned, write it with 128-bit stores
  static constexpr bool kVec = KB % 4 == 0;
  static constexpr int kSlots = KB;
  __device__ __forceinline__ void emit_vec(int32_t* oi, float* od, bool take_sqrt) {
#pragma unroll
    for (int s = 0; s < KB / 4; ++s) {
      reinterpret_cast<int4*>(oi)[s] = make_int4(i[4 * s], i[4 * s + 1], i[4 * s + 2], i[4 * s + 3]);
      if (od) {
        float4 v = make_float4(d[4 * s], d[4 * s + 1], d[4 * s + 2], d[4 * s + 3]);
        if (take_sqrt) { v.x = sqrtf(v.x); v.y = sqrtf(v.y); v.z = sqrtf(v.z); v.w = sqrtf(v.w); }
        reinterpret_cast<float4*>(od)[s] = v;
      }
    }
  }
};

// k > 32: binary max-heap in local memory, heap-sorted at the end
struct LocalHeap {
  float d[ARBX_K_MAX];
  int32_t i[ARBX_K_MAX];
  int k, m;
  __device__ __forceinline__ void init(int k_) { k = k_; m = 0; }
  __device__ __forceinline__ float worst() const { return k == 0 ? -INFINITY : m < k ? INFINITY : d[0]; }
  __device__ __forceinline__ void sift_down(int pos, int size, float t, int32_t idx) {
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
  __device__ __forceinline__ void push(float t, int32_t idx) {
    if (m < k) {
      int pos = m++;
      while (pos > 0) {
        int par = (pos - 1) >> 1;
        if (d[par] >= t) break;
        d[pos] = d[par]; i[pos] = i[par];
        pos = par;
      }
      d[pos] = t; i[pos] = idx;
    } else {
      sift_down(0, k, t, idx);
    }
  }
  static constexpr bool kVec = false;
  static constexpr int kSlots = 0;
  __device__ __forceinline__ void emit_vec(int32_t*, float*, bool) {}
  template <class F>
  __device__ __forceinline__ void emit(int kk, F&& f) {
    for (int size = m; size > 1; --size) {   // heap sort: largest to the back
      const float t = d[size - 1]; const int32_t idx = i[size - 1];
      d[size - 1] = d[0]; i[size - 1] = i[0];
      sift_down(0, size - 1, t, idx);
    }
    for (int s = 0; s < kk; ++s) f(s, s < m ? d[s] : INFINITY, s < m ? i[s] : -1);
  }
};

// ---- packet kNN (coherent warps) ---------------------------------------------------------------------
// The 32 query points of a warp are neighbours on the curve.  When they lie close together
// compared with their k-th neighbour distance, the warp walks the tree ONCE for all of them:
//   1. seed bound: the warp descends from the root towards the centre c* of its query points to
//      the smallest subtree with >= k primitives, computes the distances from c* to (at most 64
//      of) those primitives, one or two per lane, and takes an upper bound d* of the k-th
//      smallest of them with a 16-step radix select over ballots.  By the triangle inequality
//      lane's k-th neighbour distance is <= d* + ||y - c*||: a VALID initial bound per lane.
//   2. lanes-over-nodes traversal with the joint region (box J of the query points, radius
//      Rj = largest current per-lane bound): lane i tests the two child boxes of node i of a
//      shared-memory work list; primitives of hit leaf ranges are first filtered against
//      (J, Rj), one primitive per lane, and only the survivors are broadcast for the exact
//      per-lane distance and best-k insertion.  Every lane's bound shrinks to its current
//      k-th distance as its best-k set fills, and Rj with it.
//   3. rows are staged in shared memory and written as whole 32-byte sectors.
// Node and leaf tests are shared by the 32 queries; what stays per lane is one exact distance
// per surviving primitive and the insertions.  Warps that are not coherent (spread of the
// query points > alpha * d*) are flagged and answered by knn_thread_kernel.  The joint tests
// use the same monotone fp32 operation sequences as the exact ones, so the packet result is
// the same set as the per-lane traversal's.
template <int PK>
__device__ __forceinline__ float knn_key_joint_box(const float* lo, const float* hi, const float* jlo, const float* jhi) {
  const float d2 = dist2_bb<D>(lo, hi, jlo, jhi);
  if constexpr (PK == KIND_SPHERE) return sqrtf(d2);
  else return d2;
}
template <int PK>
__device__ __forceinline__ float knn_key_joint_prim(const float* p, const float* jlo, const float* jhi) {
  if constexpr (PK == KIND_POINT) return dist2_pb<D>(p, jlo, jhi);
  else if constexpr (PK == KIND_BOX) return dist2_bb<D>(p, p + D, jlo, jhi);
  else return fmaxf(0.f, sqrtf(dist2_pb<D>(p, jlo, jhi)) - p[D]);
}

#ifdef ARBX_STATS
__device__ unsigned long long g_knn_stats[8];   // packet warps, fallback warps, node pops, leaf ranges, prims filtered, survivors, push rounds, lane pushes
#define KSTAT(i, v) do { const unsigned long long v__ = (unsigned long long)(v); if (lane == 0) atomicAdd(&g_knn_stats[i], v__); } while (0)
#else
#define KSTAT(i, v) do { } while (0)
#endif

template <int PK, int KB>
__global__ void __launch_bounds__(QT) knn_packet_kernel(const float4* __restrict__ nodes,
                                                        const float4* __restrict__ leaves,
                                                        const int32_t* __restrict__ root, int n,
                                                        const float* __restrict__ qpoints,
                                                        const uint32_t* __restrict__ qorder, int64_t nq,
                                                        const int32_t* __restrict__ kq, int kmax,
                                                        int32_t* __restrict__ indices,
                                                        float* __restrict__ distances,
                                                        uint32_t* __restrict__ wlist, uint32_t* __restrict__ wcount,
                                                        float alpha, int force) {
  using Heap = RegHeap<KB>;
  constexpr int PQ_CAP = 320;                       // node work list per warp
  constexpr int RCAP = 96;                          // candidate leaf ranges per warp (3 per lane)
  constexpr int KBP = KB | 1;                       // odd row pitch: conflict-free staging
  constexpr int STAGE = 32 * KBP;
  // the node work list is dead once the leaf ranges are collected: the row staging reuses it
  __shared__ int32_t s_work[QT / 32][(PQ_CAP > 2 * STAGE ? PQ_CAP : 2 * STAGE)];
  __shared__ int32_t s_path[QT / 32][STACK_DEPTH];
  __shared__ int32_t s_rfirst[QT / 32][RCAP];
  __shared__ int32_t s_rcount[QT / 32][RCAP];
  __shared__ float s_rdist[QT / 32][RCAP];
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int32_t* stack = s_work[w];
  const int64_t t = (int64_t)blockIdx.x * QT + threadIdx.x;
  const int64_t wfirst = t - lane;
  if (wfirst >= nq) return;
  const bool valid = t < nq;
  // lanes past the end of the batch repeat the warp's first query: they do not change the joint region
  const int64_t qi = qorder ? (int64_t)qorder[valid ? t : wfirst] : (valid ? t : wfirst);
  float y[D];
#pragma unroll
  for (int a = 0; a < D; ++a) y[a] = __ldg(qpoints + qi * D + a);
  int k = kq ? min(max(__ldg(kq + qi), 0), kmax) : kmax;
  if (!valid) k = 0;
  int kw = k;   // the warp's largest k: D_k is monotone in k, so its bound serves every lane
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) kw = max(kw, __shfl_xor_sync(~0u, kw, o));

  // joint box of the query points and its centre
  float jlo[D], jhi[D], cs[D];
#pragma unroll
  for (int a = 0; a < D; ++a) {
    float lo = y[a], hi = y[a];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = fminf(lo, __shfl_xor_sync(~0u, lo, o));
      hi = fmaxf(hi, __shfl_xor_sync(~0u, hi, o));
    }
    jlo[a] = lo; jhi[a] = hi; cs[a] = 0.5f * lo + 0.5f * hi;
  }
  const float delta = sqrtf(dist2_pp<D>(y, cs));
  float dmax = delta;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dmax = fmaxf(dmax, __shfl_xor_sync(~0u, dmax, o));

  // 1. seed: warp-uniform descent from the root towards c*, always into the nearer child, down to
  // a leaf range.  The path is kept (node id, bit 30 = went into child 1) for step 2.
  int depth = 0, smid;
  {
    int32_t ref = __ldg(root);
    for (;;) {
      NodeX nd;
      load_node_x(nodes, ref, nd);
      const float d0 = dist2_pb<D>(cs, nd.v, nd.v + D);
      const float d1 = dist2_pb<D>(cs, nd.v + 2 * D, nd.v + 3 * D);
      const bool pick1 = d1 < d0;
      if (lane == 0) s_path[w][depth] = ref | (pick1 ? (1 << 30) : 0);
      ++depth;
      const int32_t child = pick1 ? nd.c1 : nd.c0;
      if (child >= 0 && depth < STACK_DEPTH) { ref = child; continue; }
      smid = pick1 ? (ref + 1 + nd.r) / 2 : (nd.l + ref) / 2;    // middle of the range the descent ended in
      break;
    }
  }
  __syncwarp();
  float bound;   // per-lane initial bound in key space (squared distance; distance for SPHERE primitives)
  {
    // 64 consecutive sorted leaves around the end of the descent (any primitives make a valid bound)
    const int wn = min(n, 64);
    const int wlo = min(max(smid - wn / 2, 0), n - wn);
    uint32_t u0 = 0x7f800000u, u1 = 0x7f800000u;
    if (lane < wn) { Leaf<PK> lf; load_leaf<PK>(leaves, wlo + lane, lf); u0 = __float_as_uint(knn_key<PK>(cs, lf.v)); }
    if (32 + lane < wn) { Leaf<PK> lf; load_leaf<PK>(leaves, wlo + 32 + lane, lf); u1 = __float_as_uint(knn_key<PK>(cs, lf.v)); }
    // upper bound of the kw-th smallest key: radix select on the top 16 bits (keys are >= 0, so
    // their bit patterns order like the values), low bits rounded up
    uint32_t prefix = 0, mask = 0;
    int kk = max(kw, 1);
#pragma unroll
    for (int bit = 30; bit >= 15; --bit) {
      const uint32_t bb = 1u << bit;
      const bool m0 = (u0 & mask) == prefix && !(u0 & bb);
      const bool m1 = (u1 & mask) == prefix && !(u1 & bb);
      const int c = __popc(__ballot_sync(~0u, m0)) + __popc(__ballot_sync(~0u, m1));
      if (c < kk) { kk -= c; prefix |= bb; }
      mask |= bb;
    }
    const float ub = __uint_as_float(prefix | 0x7fffu);
    const float dk = PK == KIND_SPHERE ? ub : sqrtf(ub);
    if (!force && !(dmax <= alpha * dk)) {   // not coherent: one query per lane does it
      if (lane == 0) wlist[atomicAdd(wcount, 1u)] = (uint32_t)(wfirst >> 5);
      KSTAT(1, 1);
      return;
    }
    const float b = (dk + delta) * 1.00002f;   // triangle inequality, with room for the roundings
    bound = PK == KIND_SPHERE ? b : b * b * 1.000002f;
  }
  float thr = k > 0 ? bound : 0.f;            // lane inserts keys < thr = min(bound, k-th best so far)
  float rj = thr;                             // joint radius (key space): largest thr of the warp
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rj = fmaxf(rj, __shfl_xor_sync(~0u, rj, o));

  // 2. candidate leaf ranges: everything whose box comes within rj of the joint box.  The walk
  // starts at the highest node of the seed path whose off-path child can still matter (lane i
  // tests level i: one round instead of one round per level of the upper tree), then runs
  // lanes-over-nodes over a shared-memory work list.
  int nranges = 0;
  {
    int start = depth - 1;
    for (int l0 = 0; l0 < depth - 1; l0 += 32) {
      bool rel = false;
      if (l0 + lane < depth - 1) {
        const int32_t e = s_path[w][l0 + lane];
        NodeX nd;
        load_node_x(nodes, e & ~(1 << 30), nd);
        const bool pick1 = (e >> 30) & 1;
        rel = (pick1 ? knn_key_joint_box<PK>(nd.v, nd.v + D, jlo, jhi)
                     : knn_key_joint_box<PK>(nd.v + 2 * D, nd.v + 3 * D, jlo, jhi)) < rj;
      }
      const uint32_t m = __ballot_sync(~0u, rel);
      if (m) { start = l0 + __ffs(m) - 1; break; }
    }
    const uint32_t lt = (1u << lane) - 1u;
    int nlist = 1;
    if (lane == 0) stack[0] = s_path[w][start] & ~(1 << 30);
    __syncwarp();
    while (nlist > 0) {
      const int take = nlist > PQ_CAP - STACK_DEPTH - 64 ? 1 : min(32, nlist);
      nlist -= take;
      const int32_t my = lane < take ? stack[nlist + lane] : -1;
      __syncwarp();
      KSTAT(2, __popc(__ballot_sync(~0u, my >= 0)));
      NodeX nd;
      float b0 = INFINITY, b1 = INFINITY;
      if (my >= 0) {
        load_node_x(nodes, my, nd);
        b0 = knn_key_joint_box<PK>(nd.v, nd.v + D, jlo, jhi);
        b1 = knn_key_joint_box<PK>(nd.v + 2 * D, nd.v + 3 * D, jlo, jhi);
      }
      const bool h0 = my >= 0 && b0 < rj, h1 = my >= 0 && b1 < rj;
      const bool lf0 = h0 && nd.c0 < 0, lf1 = h1 && nd.c1 < 0;
      const bool in0 = h0 && nd.c0 >= 0, in1 = h1 && nd.c1 >= 0;
      const uint32_t r0 = __ballot_sync(~0u, lf0), r1 = __ballot_sync(~0u, lf1);
      const int nr = __popc(r0) + __popc(r1);
      if (nranges + nr > RCAP) {               // more candidate ranges than the list holds: per-lane kernel
        if (lane == 0) wlist[atomicAdd(wcount, 1u)] = (uint32_t)(wfirst >> 5);
        KSTAT(1, 1);
        return;
      }
      if (lf0) { const int e = nranges + __popc(r0 & lt); s_rfirst[w][e] = nd.l; s_rcount[w][e] = my - nd.l + 1; s_rdist[w][e] = b0; }
      if (lf1) { const int e = nranges + __popc(r0) + __popc(r1 & lt); s_rfirst[w][e] = my + 1; s_rcount[w][e] = nd.r - my; s_rdist[w][e] = b1; }
      nranges += nr;
      const uint32_t q0 = __ballot_sync(~0u, in0), q1 = __ballot_sync(~0u, in1);
      if (in0) stack[nlist + __popc(q0 & lt)] = nd.c0;
      if (in1) stack[nlist + __popc(q0) + __popc(q1 & lt)] = nd.c1;
      nlist += __popc(q0) + __popc(q1);
      __syncwarp();
    }
  }
  KSTAT(0, 1);

  // 3. the ranges nearest-first; every lane's bound shrinks to its current k-th distance as its
  // best-k set fills, the joint radius with it, and the walk ends when the nearest unvisited
  // range lies beyond the joint radius
  Heap heap;
  heap.init(k);
  {
    float rd[RCAP / 32];
#pragma unroll
    for (int j = 0; j < RCAP / 32; ++j) rd[j] = j * 32 + lane < nranges ? s_rdist[w][j * 32 + lane] : INFINITY;
    for (;;) {
      float best = rd[0];
      int bi = lane;
#pragma unroll
      for (int j = 1; j < RCAP / 32; ++j)
        if (rd[j] < best) { best = rd[j]; bi = j * 32 + lane; }
      // warp argmin with redux.sync: box distances are >= 0 (or +inf), so their bit patterns
      // order like the values; among equal minima the lowest lane's range is taken
      {
        const uint32_t bb = __float_as_uint(best);
        const uint32_t mb = __reduce_min_sync(~0u, bb);
        const int src = __ffs(__ballot_sync(~0u, bb == mb)) - 1;
        bi = __shfl_sync(~0u, bi, src);
        best = __uint_as_float(mb);
      }
      if (!(best < rj)) break;
#pragma unroll
      for (int j = 0; j < RCAP / 32; ++j)
        if (bi == j * 32 + lane) rd[j] = INFINITY;
      const int first = s_rfirst[w][bi], m = s_rcount[w][bi];
      KSTAT(3, 1); KSTAT(4, m);
      for (int j0 = 0; j0 < m; j0 += 32) {
        bool in = false;
        if (j0 + lane < m) {
          Leaf<PK> mine;
          load_leaf<PK>(leaves, first + j0 + lane, mine);
          in = knn_key_joint_prim<PK>(mine.v, jlo, jhi) < rj;
        }
        uint32_t todo = __ballot_sync(~0u, in);
        KSTAT(5, __popc(todo));
        while (todo) {
          const int b = __ffs(todo) - 1;
          todo &= todo - 1;
          Leaf<PK> lf;
          load_leaf<PK>(leaves, first + j0 + b, lf);
          const float key = knn_key<PK>(y, lf.v);
#ifdef ARBX_STATS
          { const uint32_t pm = __ballot_sync(~0u, key < thr); KSTAT(6, pm != 0); KSTAT(7, __popc(pm)); }
#endif
          if (key < thr) {
            heap.push_uniform(key, (int32_t)(lf.idx & ~LEAF_END));
            thr = fminf(thr, heap.worst());
          }
        }
      }
      rj = __uint_as_float(__reduce_max_sync(~0u, __float_as_uint(thr)));   // thr >= 0: bits order like values
    }
  }

  // 4. emit: stage the rows, then write them as runs of whole sectors
  __syncwarp();
  float* sd = reinterpret_cast<float*>(s_work[w]);
  int32_t* si = s_work[w] + STAGE;
  heap.emit(k, [&](int pos, float key, int32_t idx) {
    sd[lane * KBP + pos] = (PK == KIND_SPHERE || idx < 0) ? key : sqrtf(key);
    si[lane * KBP + pos] = idx;
  });
  for (int pos = k; pos < kmax; ++pos) { sd[lane * KBP + pos] = INFINITY; si[lane * KBP + pos] = -1; }
  __syncwarp();
  const int total = (int)min((int64_t)32, nq - wfirst) * kmax;
  auto write_rows = [&](auto kconst) {            // kconst: compile-time row length, or 0 for kmax
    const int kk = decltype(kconst)::value ? decltype(kconst)::value : kmax;
    for (int e0 = 0; e0 < total; e0 += 32) {      // warp-uniform trip count: the shuffle needs every lane
      const int e = min(e0 + lane, total - 1);
      const int row = e / kk, slot = e - row * kk;
      const int64_t q = __shfl_sync(~0u, qi, row);
      if (e0 + lane < total) {
        indices[q * kk + slot] = si[row * KBP + slot];
        if (distances) distances[q * kk + slot] = sd[row * KBP + slot];
      }
    }
  };
  if (kmax == KB) write_rows(std::integral_constant<int, KB>{});
  else write_rows(std::integral_constant<int, 0>{});
}

// ---- one query per thread (independent traversal) --------------------------------------------------
// Kept beside the packet kernels: when the 32 queries of a warp are NOT spatially coherent
// (high dimension, strongly clustered data) the packet visits the union of 32 unrelated
// paths and independent traversal wins.  Spatial kernels choose per warp (warp_coherent).
template <int PK, class Heap>
__device__ __forceinline__ void knn_thread_query(const int64_t t, const float4* __restrict__ nodes,
                                                 const float4* __restrict__ leaves,
                                                 const int32_t* __restrict__ root,
                                                 const float* __restrict__ qpoints,
                                                 const uint32_t* __restrict__ qorder,
                                                 const int32_t* __restrict__ kq, int kmax,
                                                 int64_t n, int32_t* __restrict__ indices,
                                                 float* __restrict__ distances, int vec_ok) {
  const int64_t qi = qorder ? (int64_t)qorder[t] : t;
  float y[D];
#pragma unroll
  for (int a = 0; a < D; ++a) y[a] = __ldg(qpoints + qi * D + a);
  const int k = kq ? min(max(__ldg(kq + qi), 0), kmax) : kmax;
  Heap heap;
  heap.init(k);
  if (n > 0) {
    int32_t sref[STACK_DEPTH];
    float sbound[STACK_DEPTH];
    int sp = 0;
    constexpr int32_t DONE = INT32_MIN;
    auto pop = [&]() -> int32_t {
      while (sp > 0) {
        --sp;
        if (sbound[sp] < heap.worst()) return sref[sp];
      }
      return DONE;
    };
    int32_t ref = __ldg(root);
    // "while-while" loop: all lanes first descend through internal nodes until each holds a
    // leaf range (or is done), then the leaf scans run together -- less divergence than
    // mixing node steps and leaf scans in one loop body.
    for (;;) {
      while (ref >= 0) {
        Node nd;
        load_node(nodes, ref, nd);
        float b0 = knn_bound<PK>(y, nd.v, nd.v + D);
        float b1 = knn_bound<PK>(y, nd.v + 2 * D, nd.v + 3 * D);
        int32_t c0 = nd.c0, c1 = nd.c1;
        if (b1 < b0) { float tb = b0; b0 = b1; b1 = tb; int32_t tc = c0; c0 = c1; c1 = tc; }
        const float w = heap.worst();
        if (b0 < w) {
          ref = c0;
          if (b1 < w) { sref[sp] = c1; sbound[sp] = b1; ++sp; }
        } else {
          ref = pop();
        }
      }
      if (ref == DONE) break;
      int j = ~ref;
      for (;; ++j) {
        Leaf<PK> lf;
        load_leaf<PK>(leaves, j, lf);
        const float key = knn_key<PK>(y, lf.v);
        if (key < heap.worst()) heap.push(key, (int32_t)(lf.idx & ~LEAF_END));
        if (lf.idx & LEAF_END) break;
      }
      ref = pop();
    }
  }
  int32_t* oi = indices + qi * kmax;
  float* od = distances ? distances + qi * kmax : nullptr;
  if constexpr (Heap::kVec) {
    // rows of exactly kSlots entries on 16-byte aligned outputs: 128-bit stores
    // (sqrt(+inf) = +inf keeps the padding of short rows (n < k) intact)
    if (vec_ok && k == Heap::kSlots) { heap.emit_vec(oi, od, PK != KIND_SPHERE); return; }
  }
  heap.emit(k, [&](int s, float key, int32_t idx) {
    oi[s] = idx;
    if (od) od[s] = (PK == KIND_SPHERE || idx < 0) ? key : sqrtf(key);
  });
  for (int s = k; s < kmax; ++s) {      // per-query k: the rest of the row is padding
    oi[s] = -1;
    if (od) od[s] = INFINITY;
  }
}

template <int PK, class Heap>
__global__ void __launch_bounds__(QT) knn_thread_kernel(const float4* __restrict__ nodes,
                                                 const float4* __restrict__ leaves,
                                                 const int32_t* __restrict__ root,
                                                 const float* __restrict__ qpoints,
                                                 const uint32_t* __restrict__ qorder, int64_t nq,
                                                 const int32_t* __restrict__ kq, int kmax,
                                                 int64_t n, int32_t* __restrict__ indices,
                                                 float* __restrict__ distances, int vec_ok) {
  const int64_t t = (int64_t)blockIdx.x * QT + threadIdx.x;
  if (t < nq) knn_thread_query<PK, Heap>(t, nodes, leaves, root, qpoints, qorder, kq, kmax, n, indices, distances, vec_ok);
}

// The warps the packet kernel handed over (list `wlist` of warp numbers, `*wcount` entries): a
// fixed grid walks the list, so every resident warp has work for the whole launch (a launch
// over all warps with an early exit ran at 34 % active warps).
template <int PK, class Heap>
__global__ void __launch_bounds__(QT) knn_thread_list_kernel(const float4* __restrict__ nodes,
                                                 const float4* __restrict__ leaves,
                                                 const int32_t* __restrict__ root,
                                                 const float* __restrict__ qpoints,
                                                 const uint32_t* __restrict__ qorder, int64_t nq,
                                                 const int32_t* __restrict__ kq, int kmax,
                                                 int64_t n, int32_t* __restrict__ indices,
                                                 float* __restrict__ distances, int vec_ok,
                                                 const uint32_t* __restrict__ wlist,
                                                 const uint32_t* __restrict__ wcount) {
  const uint32_t cnt = *wcount;
  for (uint32_t i = blockIdx.x * (QT / 32) + (threadIdx.x >> 5); i < cnt; i += gridDim.x * (QT / 32)) {
    const int64_t t = (int64_t)wlist[i] * 32 + (threadIdx.x & 31);
    if (t < nq) knn_thread_query<PK, Heap>(t, nodes, leaves, root, qpoints, qorder, kq, kmax, n, indices, distances, vec_ok);
  }
}

inline int traversal_mode() { return g_cfg.traversal.load(std::memory_order_relaxed); }

// ---- host dispatch ------------------------------------------------------------------------------------
template <int PK, int QK, bool SELF = false>
arbx_status spatial_launch(const Index* ix, const SpatialArgs& a, cudaStream_t s) {
  const unsigned grid = (unsigned)((a.nq + QT - 1) / QT);
  const float4* nodes = reinterpret_cast<const float4*>(ix->nodes);
  const float4* leaves = reinterpret_cast<const float4*>(ix->leaves);
  ProfScope ps(a.pass == 1 ? K_SPATIAL_FILL : K_SPATIAL_COUNT, s);
  const int mode = traversal_mode();
  // packet threshold (spread of the warp's query centres <= alpha * query extent), measured:
  // 1.5 (spheres) / 2.5 (boxes) up to 3-D, 0.75 above (the joint region gets loose quickly)
  float alpha = D <= 3 ? (QK == KIND_BOX ? 2.5f : 1.5f) : 0.75f;
  if (const float v = g_cfg.packet_alpha.load(std::memory_order_relaxed); v >= 0.f) alpha = v;
  const int n = (int)ix->n;
  if (a.pass == 1 && a.heavy && !SELF) {   // qorder = the list of overflowing queries, one warp each
    const unsigned hgrid = (unsigned)((a.nq * 32 + QT - 1) / QT);
    spatial_heavy_kernel<PK, QK><<<hgrid, QT, 0, s>>>(nodes, leaves, ix->root, n, a.queries, a.qorder, a.nq, a.offsets, a.indices);
  } else if (a.pass == 1)
    spatial_kernel<PK, QK, 1, SELF><<<grid, QT, 0, s>>>(nodes, leaves, ix->root, n, a.queries, a.qorder, a.nq, a.counts, a.offsets, a.indices, a.cap, nullptr, nullptr, a.stop_fill, mode, alpha);
  else if (a.pass == 3) {
    if constexpr (SELF)   // DBSCAN edges: counts = neighbour counts (read), rows = union-find array, cap = min_pts
      spatial_kernel<PK, QK, 3, true><<<grid, QT, 0, s>>>(nodes, leaves, ix->root, n, a.queries, a.qorder, a.nq, a.counts, nullptr, a.rows, a.cap, nullptr, nullptr, 0, mode, alpha);
  } else if (a.pass == 2)
    spatial_kernel<PK, QK, 2, SELF><<<grid, QT, 0, s>>>(nodes, leaves, ix->root, n, a.queries, a.qorder, a.nq, a.counts, nullptr, a.rows, a.cap, a.overflow, a.ovf_list, 0, mode, alpha);
  else
    spatial_kernel<PK, QK, 0, SELF><<<grid, QT, 0, s>>>(nodes, leaves, ix->root, n, a.queries, a.qorder, a.nq, a.counts, nullptr, nullptr, a.cap, nullptr, nullptr, 0, mode, alpha);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

template <int PK>
arbx_status spatial_pk(const Index* ix, const SpatialArgs& a, cudaStream_t s) {
  switch (a.qkind) {
    case KIND_POINT: return spatial_launch<PK, KIND_POINT>(ix, a, s);
    case KIND_BOX: return spatial_launch<PK, KIND_BOX>(ix, a, s);
    default: return spatial_launch<PK, KIND_SPHERE>(ix, a, s);
  }
}

arbx_status spatial_entry(const Index* ix, const SpatialArgs& a, cudaStream_t s) {
  if (a.self) return spatial_launch<KIND_POINT, KIND_SPHERE, true>(ix, a, s);   // api.cu guarantees POINT prims
  switch (ix->kind) {
    case KIND_POINT: return spatial_pk<KIND_POINT>(ix, a, s);
    case KIND_BOX: return spatial_pk<KIND_BOX>(ix, a, s);
    default: return spatial_pk<KIND_SPHERE>(ix, a, s);
  }
}

template <int PK, class Heap>
arbx_status knn_thread_launch(const Index* ix, const KnnArgs& a, const uint32_t* wlist, const uint32_t* wcount, cudaStream_t s) {
  // 128-bit row stores need 16-byte aligned output pointers (rows of 4, 8, 16, 32 entries then stay aligned)
  const int vec_ok = !a.kq && ((reinterpret_cast<uintptr_t>(a.indices) | reinterpret_cast<uintptr_t>(a.distances)) & 15) == 0;
  const float4* nodes = reinterpret_cast<const float4*>(ix->nodes);
  const float4* leaves = reinterpret_cast<const float4*>(ix->leaves);
  if (wlist) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    knn_thread_list_kernel<PK, Heap><<<sms * 16, QT, 0, s>>>(nodes, leaves, ix->root, a.qpoints, a.qorder, a.nq, a.kq, a.k, ix->n,
                                                            a.indices, a.distances, vec_ok, wlist, wcount);
  } else {
    const unsigned grid = (unsigned)((a.nq + QT - 1) / QT);
    knn_thread_kernel<PK, Heap><<<grid, QT, 0, s>>>(nodes, leaves, ix->root, a.qpoints, a.qorder, a.nq, a.kq, a.k, ix->n,
                                                    a.indices, a.distances, vec_ok);
  }
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

// Packet kernel for the coherent warps, per-lane kernel for the rest (listed by the packet kernel).
template <int PK, int KB>
arbx_status knn_launch(const Index* ix, const KnnArgs& a, cudaStream_t s) {
  ProfScope ps(K_KNN, s);
  const int mode = traversal_mode();
  // the packet path needs a real tree and a seed subtree of >= k primitives
  // (a small batch is bound by the latency of one warp's walk, and the packet walk of a warp is the
  //  longer one: C1, 10^4 queries, 0.20 ms with packets against 0.14 ms without)
  const bool packet = mode != 1 && ix->n >= 4 * (int64_t)a.k && ix->n > 4 * (int64_t)ix->leaf_max && ix->n >= 64 &&
                      (a.nq >= 65536 || mode == 2);
  if (!packet) return knn_thread_launch<PK, RegHeap<KB>>(ix, a, nullptr, nullptr, s);
  // measured: above 3-D the warps of the clustered workload (C5) are never coherent and the seed
  // descent is pure overhead (+0.7 ms per 10^7 queries), so packets are off unless asked for
  float alpha = D <= 3 ? 2.0f : 0.f;
  if (const float v = g_cfg.packet_alpha.load(std::memory_order_relaxed); v >= 0.f) alpha = v;
  if (alpha <= 0.f && mode != 2) return knn_thread_launch<PK, RegHeap<KB>>(ix, a, nullptr, nullptr, s);
  const int64_t nwarps = (a.nq + 31) / 32;
  Scratch<uint32_t> wlist;   // [0] = number of listed warps, [1 ..] = their numbers
  ARBX_TRY(wlist.alloc((size_t)nwarps + 1, s));
  ARBX_CUDA(cudaMemsetAsync(wlist.p, 0, sizeof(uint32_t), s));
  const unsigned grid = (unsigned)((a.nq + QT - 1) / QT);
  knn_packet_kernel<PK, KB><<<grid, QT, 0, s>>>(reinterpret_cast<const float4*>(ix->nodes),
                                                reinterpret_cast<const float4*>(ix->leaves), ix->root, (int)ix->n,
                                                a.qpoints, a.qorder, a.nq, a.kq, a.k, a.indices, a.distances,
                                                wlist.p + 1, wlist.p, alpha, mode == 2 ? 1 : 0);
  ARBX_LAUNCH_CHECK();
  // (forced packets still leave the warps with too many candidate ranges to the per-lane kernel)
  return knn_thread_launch<PK, RegHeap<KB>>(ix, a, wlist.p + 1, wlist.p, s);
}

template <int PK>
arbx_status knn_pk(const Index* ix, const KnnArgs& a, cudaStream_t s) {
  const int k = a.k;
  if (k <= 1) return knn_launch<PK, 1>(ix, a, s);
  if (k <= 2) return knn_launch<PK, 2>(ix, a, s);
  if (k <= 4) return knn_launch<PK, 4>(ix, a, s);
  if (k <= 8) return knn_launch<PK, 8>(ix, a, s);
  if (k <= 16) return knn_launch<PK, 16>(ix, a, s);
  if (k <= 32) return knn_launch<PK, 32>(ix, a, s);
  ProfScope ps(K_KNN, s);
  return knn_thread_launch<PK, LocalHeap>(ix, a, nullptr, nullptr, s);
}

arbx_status knn_entry(const Index* ix, const KnnArgs& a, cudaStream_t s) {
  switch (ix->kind) {
    case KIND_POINT: return knn_pk<KIND_POINT>(ix, a, s);
    case KIND_BOX: return knn_pk<KIND_BOX>(ix, a, s);
    default: return knn_pk<KIND_SPHERE>(ix, a, s);
  }
}

arbx_status qcode_entry(const Index* ix, const float* queries, int64_t nq, int qkind, uint32_t* codes,
                        int* key_bits, cudaStream_t s) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((nq + 255) / 256, (int64_t)sms * 8));
  ProfScope ps(K_QCODE, s);
  // the sort key keeps the top `qb` bits per axis of the code (whole 8-bit digit passes)
  constexpr int B = qcode_bits_per_axis(D);
  int qb = B;
  if (const int v = g_cfg.qbits.load(std::memory_order_relaxed); v > 0) qb = std::max(1, std::min(B, v));
  const int drop = D * (B - qb);
  switch (qkind) {
    case KIND_POINT: qcode_kernel<KIND_POINT><<<grid, 256, 0, s>>>(queries, nq, ix->bounds, codes, drop); break;
    case KIND_BOX: qcode_kernel<KIND_BOX><<<grid, 256, 0, s>>>(queries, nq, ix->bounds, codes, drop); break;
    default: qcode_kernel<KIND_SPHERE><<<grid, 256, 0, s>>>(queries, nq, ix->bounds, codes, drop); break;
  }
  ARBX_LAUNCH_CHECK();
  *key_bits = D * qb;
  return ARBX_OK;
}

#ifdef ARBX_STATS
}  // namespace
void knn_stats_read(unsigned long long* out) {   // debug builds only (-DARBX_STATS, dimension ARBX_DIM)
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(out, g_knn_stats, sizeof(g_knn_stats));
  unsigned long long z[8] = {};
  cudaMemcpyToSymbol(g_knn_stats, z, sizeof(z));
}
namespace {
#endif

const DimTable kTable = {spatial_entry, knn_entry, qcode_entry};

}  // namespace

#define ARBX_CAT2(a, b) a##b
#define ARBX_CAT(a, b) ARBX_CAT2(a, b)
const DimTable* ARBX_CAT(dim_table_, ARBX_DIM)() { return &kTable; }

}  // namespace arbx
