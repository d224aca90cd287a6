// api.cu -- the C ABI of include/arbx.h: argument validation, handle ownership, scratch
// management and the order of the hot-path steps:
//   build   : B1 bounds -> B2 codes -> B3 sort -> B4 leaves -> B5+B6 hierarchy/refit
//   count   : Q1 query codes -> Q2 sort -> T1 traversal (count)
//   spatial : Q1 -> Q2 -> T1 -> T2 scan -> [host learns total] -> T3 traversal (fill)
//   knn     : Q1 -> Q2 -> K1 traversal + K2 emit
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <string>
#include <unordered_map>
#include <vector>

#include "common.cuh"

namespace arbx {

std::atomic<long long> g_launches{0};
DebugCfg g_cfg;
static thread_local char t_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(t_err, sizeof(t_err), fmt, ap);
  va_end(ap);
}

// ---- per-kernel timing ---------------------------------------------------------------------
static std::atomic<int> g_prof_on{0};
static std::mutex g_prof_mu;
struct ProfRec { int id; cudaEvent_t a, b; };
static std::vector<ProfRec> g_prof_open, g_prof_done;
static std::vector<cudaEvent_t> g_prof_pool;
static const char* const kKernelNames[K_NUM_] = {
    "B1_bounds", "B2_codes", "B3_sort_hist", "B3_sort_pass", "B4_leaves", "B5B6_hierarchy_refit",
    "Q1_qcodes", "Q2_qsort_hist", "Q2_qsort_pass", "T1_spatial_count", "T2_scan", "T3_spatial_fill",
    "K1K2_knn", "misc"};

bool prof_enabled() { return g_prof_on.load(std::memory_order_relaxed) != 0; }
static cudaEvent_t prof_event() {
  if (!g_prof_pool.empty()) { cudaEvent_t e = g_prof_pool.back(); g_prof_pool.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
void prof_begin(int id, cudaStream_t s) {
  std::lock_guard<std::mutex> g(g_prof_mu);
  ProfRec r{id, prof_event(), prof_event()};
  cudaEventRecord(r.a, s);
  g_prof_open.push_back(r);
}
void prof_end(int id, cudaStream_t s) {
  std::lock_guard<std::mutex> g(g_prof_mu);
  for (size_t i = g_prof_open.size(); i-- > 0;)
    if (g_prof_open[i].id == id) {
      cudaEventRecord(g_prof_open[i].b, s);
      g_prof_done.push_back(g_prof_open[i]);
      g_prof_open.erase(g_prof_open.begin() + i);
      return;
    }
}

// Device memory (the handle's tree and all per-call scratch) comes from a stream-ordered pool
// OWNED BY THE LIBRARY, one per device: the process-wide default pool and PyTorch's caching
// allocator are left alone.  Freed blocks stay cached in the pool up to a bounded release
// threshold (so that the host synchronisation inside the storage query does not hand the
// scratch back to the driver every call); arbx_trim returns the cache to the driver.
static std::once_flag g_pool_once[64];
static cudaMemPool_t g_pool[64];
static std::atomic<long long> g_pool_keep_mb{16384};
static std::atomic<int> g_pool_thr_set[64];

static void pool_apply_threshold(cudaMemPool_t pool) {
  unsigned long long thr = (unsigned long long)g_pool_keep_mb.load() << 20;
  if (cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr) != cudaSuccess) cudaGetLastError();
}

static cudaMemPool_t pool_for(int dev) {
  if (dev < 0 || dev >= 64) return nullptr;
  std::call_once(g_pool_once[dev], [dev] {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool = nullptr;
    if (cudaMemPoolCreate(&pool, &props) == cudaSuccess) {
      pool_apply_threshold(pool);
      g_pool[dev] = pool;
    } else {
      cudaGetLastError();
      g_pool[dev] = nullptr;
    }
  });
  return g_pool[dev];
}

// On top of the pool sits a small caching layer: a freed block is kept, tagged with the stream it
// was freed on, and handed to the next request of (nearly) the same size on that stream -- reuse
// on one stream is ordered by the stream itself.  Measured on B200 / CUDA 12.9: without it the
// 2.56 GB row scratch of the C3 storage query cost 17-290 ms of host time in
// cudaMallocFromPoolAsync on EVERY call (the smaller requests of the calls in between had carved
// up the freed range, so the driver mapped fresh memory each time); with it the call's device
// time is steady.  The cache is bounded by the same "pool_keep_mb"; arbx_trim empties it.
struct CacheBlock { void* p; size_t bytes; int dev; cudaStream_t s; unsigned long long tick; };
static std::mutex g_cache_mu;
static std::vector<CacheBlock> g_cache;
static std::unordered_map<void*, size_t> g_live;
static size_t g_cached_bytes = 0;
static unsigned long long g_cache_tick = 0;

static void cache_evict_locked(size_t keep_bytes) {
  while (g_cached_bytes > keep_bytes && !g_cache.empty()) {
    size_t oldest = 0;
    for (size_t i = 1; i < g_cache.size(); ++i)
      if (g_cache[i].tick < g_cache[oldest].tick) oldest = i;
    const CacheBlock b = g_cache[oldest];
    g_cache[oldest] = g_cache.back();
    g_cache.pop_back();
    g_cached_bytes -= b.bytes;
    if (cudaFreeAsync(b.p, b.s) != cudaSuccess) { cudaGetLastError(); cudaFree(b.p); }
  }
}

arbx_status scratch_alloc(void** p, size_t bytes, cudaStream_t s) {
  int dev = 0;
  cudaGetDevice(&dev);
  cudaMemPool_t pool = pool_for(dev);
  *p = nullptr;
  if (!pool) { set_error("could not create the library's memory pool on device %d", dev); return ARBX_ERR_CUDA; }
  const size_t want = ((bytes ? bytes : 1) + 511) & ~size_t(511);
  {
    std::lock_guard<std::mutex> g(g_cache_mu);
    size_t best = g_cache.size();
    for (size_t i = 0; i < g_cache.size(); ++i) {
      const CacheBlock& b = g_cache[i];
      if (b.dev == dev && b.s == s && b.bytes >= want && b.bytes <= want + want / 8 + 4096 &&
          (best == g_cache.size() || b.bytes < g_cache[best].bytes))
        best = i;
    }
    if (best != g_cache.size()) {
      *p = g_cache[best].p;
      g_live[*p] = g_cache[best].bytes;
      g_cached_bytes -= g_cache[best].bytes;
      g_cache[best] = g_cache.back();
      g_cache.pop_back();
      return ARBX_OK;
    }
  }
  cudaError_t e = cudaMallocFromPoolAsync(p, want, pool, s);
  if (e == cudaErrorMemoryAllocation) {   // make room: drop the cache, then try once more
    cudaGetLastError();
    { std::lock_guard<std::mutex> g(g_cache_mu); cache_evict_locked(0); }
    e = cudaMallocFromPoolAsync(p, want, pool, s);
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    set_error("cudaMallocFromPoolAsync(%zu bytes) failed: %s", bytes, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? ARBX_ERR_OOM : ARBX_ERR_CUDA;
  }
  // measured on B200 / CUDA 12.9: a release threshold set on a pool that has never allocated is
  // not honoured (every synchronisation hands the pool's free memory back), so it is applied
  // again after the pool's first allocation
  if (!g_pool_thr_set[dev].exchange(1)) pool_apply_threshold(pool);
  std::lock_guard<std::mutex> g(g_cache_mu);
  g_live[*p] = want;
  return ARBX_OK;
}
void scratch_free(void* p, cudaStream_t s) {
  if (!p) return;
  int dev = 0;
  cudaGetDevice(&dev);
  std::lock_guard<std::mutex> g(g_cache_mu);
  auto it = g_live.find(p);
  if (it == g_live.end()) { cudaFreeAsync(p, s); return; }
  g_cache.push_back(CacheBlock{p, it->second, dev, s, ++g_cache_tick});
  g_cached_bytes += it->second;
  g_live.erase(it);
  cache_evict_locked((size_t)g_pool_keep_mb.load() << 20);
}

const DimTable* dim_table_1(); const DimTable* dim_table_2(); const DimTable* dim_table_3();
const DimTable* dim_table_4(); const DimTable* dim_table_5(); const DimTable* dim_table_6();
const DimTable* dim_table_7(); const DimTable* dim_table_8(); const DimTable* dim_table_9();
const DimTable* dim_table_10();

const DimTable* dim_table(int dim) {
  switch (dim) {
    case 1: return dim_table_1(); case 2: return dim_table_2(); case 3: return dim_table_3();
    case 4: return dim_table_4(); case 5: return dim_table_5(); case 6: return dim_table_6();
    case 7: return dim_table_7(); case 8: return dim_table_8(); case 9: return dim_table_9();
    case 10: return dim_table_10();
  }
  return nullptr;
}

static void free_index(Index* ix, cudaStream_t s) {
  scratch_free(ix->leaves, s); scratch_free(ix->nodes, s); scratch_free(ix->bounds, s);
  scratch_free(ix->root, s);
  scratch_free(ix->rows64, s);
}

// Q1 + Q2: order in which the queries are traversed (neighbours on the curve share a warp)
struct QueryOrder {
  Scratch<uint32_t> buf[2];
  const uint32_t* p = nullptr;   // order[t] = caller's index of the t-th query on the curve
};
static arbx_status query_order(const Index* ix, const float* queries, int64_t nq, int qkind,
                               QueryOrder& order, cudaStream_t s) {
  if (ix->brute) { order.p = nullptr; return ARBX_OK; }   // every query scans every primitive: order is irrelevant
  Scratch<uint32_t> codes, codes_alt;
  ARBX_TRY(codes.alloc((size_t)nq, s));
  ARBX_TRY(codes_alt.alloc((size_t)nq, s));
  ARBX_TRY(order.buf[0].alloc((size_t)nq, s));
  ARBX_TRY(order.buf[1].alloc((size_t)nq, s));
  int key_bits = 32;
  ARBX_TRY(dim_table(ix->dim)->qcode(ix, queries, nq, qkind, codes.p, &key_bits, s));
  uint32_t *kout = nullptr, *vout = nullptr;
  ARBX_TRY(radix_sort_u32(codes.p, codes_alt.p, order.buf[0].p, order.buf[1].p, true, nq, key_bits, s, &kout, &vout));
  order.p = vout;
  return ARBX_OK;
}

// Experiment (knob "l2_persist"): a persisting-L2 access-policy window over the node array for
// the kernels of one query call.  Node ids are split positions, so the upper levels are NOT
// contiguous: the window can only cover the whole array with hitRatio = carve-out / size.
struct L2Window {
  cudaStream_t s; bool on = false;
  L2Window(const Index* ix, cudaStream_t s_) : s(s_) {
    if (!g_cfg.l2_persist.load(std::memory_order_relaxed) || !ix->nodes || ix->n < 2) return;
    int dev = 0, max_persist = 0, max_window = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev);
    cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev);
    if (max_persist <= 0 || max_window <= 0) return;
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)max_persist);
    const size_t bytes = std::min<size_t>((size_t)(ix->n - 1) * node_width(ix->dim) * sizeof(float), (size_t)max_window);
    cudaStreamAttrValue v = {};
    v.accessPolicyWindow.base_ptr = ix->nodes;
    v.accessPolicyWindow.num_bytes = bytes;
    v.accessPolicyWindow.hitRatio = std::min(1.0f, (float)max_persist / (float)bytes);
    v.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    v.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    on = cudaStreamSetAttribute(s, cudaStreamAttributeAccessPolicyWindow, &v) == cudaSuccess;
    if (!on) cudaGetLastError();
  }
  ~L2Window() {
    if (!on) return;
    cudaStreamAttrValue v = {};
    v.accessPolicyWindow.num_bytes = 0;
    cudaStreamSetAttribute(s, cudaStreamAttributeAccessPolicyWindow, &v);
  }
};

// A fault raised by the (asynchronous) build kernels is reported by the first call on the
// handle that synchronises with the host.
static arbx_status check_build_fault(int32_t flags) {
  if (flags == 0) return ARBX_OK;
  set_error("the build of this handle failed on the device (fault flags 0x%x: parked-subtree list overflow)", flags);
  return ARBX_ERR_CUDA;
}

__global__ void fill_i32_kernel(int32_t* p, int64_t n, int32_t v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}
__global__ void fill_knn_empty_kernel(int32_t* idx, float* dist, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    idx[i] = -1;
    if (dist) dist[i] = INFINITY;
  }
}

// Q3 experiment (knob "gather"): sorted[t] = queries[order[t]] (rows of w floats), and the inverse
// for the counts: counts[order[t]] = sorted_counts[t]
__global__ void gather_rows_kernel(const float* __restrict__ rows, const uint32_t* __restrict__ order, int64_t nq, int w,
                                   float* __restrict__ sorted) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nq * w) return;
  const int64_t t = e / w;
  sorted[e] = rows[(int64_t)order[t] * w + (e - t * w)];
}
__global__ void unpermute_i32_kernel(const int32_t* __restrict__ sorted, const uint32_t* __restrict__ order, int64_t nq,
                                     int32_t* __restrict__ out) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nq) out[order[t]] = sorted[t];
}

// self-join queries: query i = (point i, radius) in the caller's order; order[t] = caller's
// index of the leaf at sorted position t (so no query sort is needed: tree order IS the order)
__global__ void self_queries_kernel(const float* __restrict__ leaves, int64_t n, int D, int LW, float radius,
                                    float* __restrict__ queries, uint32_t* __restrict__ order) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const float* lf = leaves + t * LW;
  const uint32_t idx = __float_as_uint(lf[D]) & ~LEAF_END;
  for (int a = 0; a < D; ++a) queries[(int64_t)idx * (D + 1) + a] = lf[a];
  queries[(int64_t)idx * (D + 1) + D] = radius;
  order[t] = idx;
}

// ---- DBSCAN glue (arbx_dbscan) ------------------------------------------------------------------
__global__ void dbscan_init_kernel(const int32_t* __restrict__ counts, int min_pts, int64_t n, int32_t* __restrict__ uf) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) uf[i] = counts[i] >= min_pts ? (int32_t)i : -1;     // core points start as their own cluster
}
// label = smallest core index of the cluster; a border point takes the cluster of the core point
// it remembered; everything else is noise (-1)
__global__ void dbscan_labels_kernel(const int32_t* __restrict__ uf, int64_t n, int32_t* __restrict__ labels) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t x = uf[i];
  if (x == -1) { labels[i] = -1; return; }
  if (x <= -2) x = -2 - x;                     // border: follow the remembered core point
  else x = (int32_t)i;
  for (int32_t p = uf[x]; p != x; p = uf[x]) x = p;   // the forest is final here: plain root walk
  labels[i] = x;
}

}  // namespace arbx

using namespace arbx;

struct arbx_index_s { Index ix; };

static bool bad_kind(int k) { return k < 0 || k > 2; }
constexpr int64_t kMaxCount = int64_t(1) << 30;

extern "C" {

arbx_status arbx_build(const float* prims, int64_t n, int dim, arbx_kind kind, arbx_stream stream,
                       arbx_handle* out) {
  if (!out || n < 0 || dim < 1 || dim > ARBX_MAX_DIM || bad_kind((int)kind) || (n > 0 && !prims)) {
    set_error("arbx_build: invalid argument (n=%lld dim=%d kind=%d)", (long long)n, dim, (int)kind);
    return ARBX_ERR_INVALID_ARG;
  }
  if (n > kMaxCount) { set_error("arbx_build: n > 2^30 unsupported"); return ARBX_ERR_UNSUPPORTED; }
  cudaStream_t s = (cudaStream_t)stream;
  arbx_index_s* h = new arbx_index_s();
  h->ix.leaf_max = std::max(1, std::min(64, g_cfg.leaf_max.load(std::memory_order_relaxed)));
  arbx_status st = build_index(prims, n, dim, (int)kind, s, &h->ix);
  if (st != ARBX_OK) {
    free_index(&h->ix, s);
    delete h;
    return st;
  }
  *out = h;
  return ARBX_OK;
}

arbx_status arbx_destroy(arbx_handle h, arbx_stream stream) {
  if (!h) return ARBX_OK;
  free_index(&h->ix, (cudaStream_t)stream);
  delete h;
  return ARBX_OK;
}

arbx_status arbx_size(arbx_handle h, int64_t* n) {
  if (!h || !n) { set_error("arbx_size: null argument"); return ARBX_ERR_INVALID_ARG; }
  *n = h->ix.n;
  return ARBX_OK;
}

arbx_status arbx_bounds(arbx_handle h, float* lo_host, float* hi_host, arbx_stream stream) {
  if (!h || !lo_host || !hi_host) { set_error("arbx_bounds: null argument"); return ARBX_ERR_INVALID_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  float tmp[2 * ARBX_MAX_DIM];
  int32_t rootw[2] = {0, 0};
  const int D = h->ix.dim;
  ARBX_CUDA(cudaMemcpyAsync(tmp, h->ix.bounds, 2 * D * sizeof(float), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaMemcpyAsync(rootw, h->ix.root, sizeof(rootw), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaStreamSynchronize(s));
  ARBX_TRY(check_build_fault(rootw[1]));
  for (int a = 0; a < D; ++a) { lo_host[a] = tmp[a]; hi_host[a] = tmp[D + a]; }
  return ARBX_OK;
}

static arbx_status count_impl(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                              int32_t limit, int32_t* counts, arbx_stream stream);

arbx_status arbx_query_count(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                             int32_t* counts, arbx_stream stream) {
  return count_impl(h, queries, nq, qkind, 0, counts, stream);
}

arbx_status arbx_query_count_upto(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                                  int32_t limit, int32_t* counts, arbx_stream stream) {
  if (limit < 1) { set_error("arbx_query_count_upto: limit must be >= 1"); return ARBX_ERR_INVALID_ARG; }
  return count_impl(h, queries, nq, qkind, limit, counts, stream);
}

static arbx_status count_impl(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                              int32_t limit, int32_t* counts, arbx_stream stream) {
  if (!h || nq < 0 || bad_kind((int)qkind) || (nq > 0 && (!queries || !counts))) {
    set_error("arbx_query_count: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  if (h->ix.f64) { set_error("arbx_query_count: the handle was built from fp64 coordinates, use the _f64 calls"); return ARBX_ERR_INVALID_ARG; }
  if (nq > kMaxCount) { set_error("arbx_query_count: nq > 2^30 unsupported"); return ARBX_ERR_UNSUPPORTED; }
  if (nq == 0) return ARBX_OK;
  cudaStream_t s = (cudaStream_t)stream;
  const Index* ix = &h->ix;
  if (ix->n == 0) { ARBX_CUDA(cudaMemsetAsync(counts, 0, (size_t)nq * sizeof(int32_t), s)); return ARBX_OK; }
  QueryOrder order;
  ARBX_TRY(query_order(ix, queries, nq, (int)qkind, order, s));
  SpatialArgs a{queries, nq, (int)qkind, order.p, counts, nullptr, nullptr, nullptr, limit, nullptr, 0};
  L2Window l2(ix, s);
  if (g_cfg.gather.load(std::memory_order_relaxed) && order.p) {
    // Q3 materialised (experiment): sorted copy of the queries, counts written in
    // sorted order, then un-permuted
    const int w = prim_width((int)qkind, ix->dim);
    Scratch<float> sq;
    Scratch<int32_t> sc;
    ARBX_TRY(sq.alloc((size_t)nq * w, s));
    ARBX_TRY(sc.alloc((size_t)nq, s));
    gather_rows_kernel<<<(unsigned)((nq * w + 255) / 256), 256, 0, s>>>(queries, order.p, nq, w, sq.p);
    ARBX_LAUNCH_CHECK();
    a.queries = sq.p; a.qorder = nullptr; a.counts = sc.p;
    ARBX_TRY(dim_table(ix->dim)->spatial(ix, a, s));
    unpermute_i32_kernel<<<(unsigned)((nq + 255) / 256), 256, 0, s>>>(sc.p, order.p, nq, counts);
    ARBX_LAUNCH_CHECK();
    return ARBX_OK;
  }
  return dim_table(ix->dim)->spatial(ix, a, s);
}

static arbx_status spatial_impl(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind, int32_t limit,
                                int32_t* offsets, int32_t* indices, int64_t indices_capacity,
                                int64_t* total_host, arbx_stream stream, float self_radius = -1.f);

arbx_status arbx_query_spatial(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                               int32_t* offsets, int32_t* indices, int64_t indices_capacity,
                               int64_t* total_host, arbx_stream stream) {
  return spatial_impl(h, queries, nq, qkind, 0, offsets, indices, indices_capacity, total_host, stream);
}

arbx_status arbx_query_spatial_upto(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                                    int32_t limit, int32_t* offsets, int32_t* indices,
                                    int64_t indices_capacity, int64_t* total_host, arbx_stream stream) {
  if (limit < 1) { set_error("arbx_query_spatial_upto: limit must be >= 1"); return ARBX_ERR_INVALID_ARG; }
  return spatial_impl(h, queries, nq, qkind, limit, offsets, indices, indices_capacity, total_host, stream);
}

arbx_status arbx_query_pairs(arbx_handle h, float radius, int32_t* offsets, int32_t* indices,
                             int64_t indices_capacity, int64_t* total_host, arbx_stream stream) {
  if (!h || !(radius >= 0.f)) { set_error("arbx_query_pairs: invalid argument"); return ARBX_ERR_INVALID_ARG; }
  if (h->ix.kind != KIND_POINT || h->ix.f64) { set_error("arbx_query_pairs: fp32 POINT primitives only"); return ARBX_ERR_UNSUPPORTED; }
  return spatial_impl(h, nullptr, h->ix.n, ARBX_SPHERE, 0, offsets, indices, indices_capacity, total_host, stream, radius);
}

arbx_status arbx_dbscan(arbx_handle h, float eps, int32_t min_pts, int32_t* labels, arbx_stream stream) {
  if (!h || !(eps >= 0.f) || min_pts < 1 || (h->ix.n > 0 && !labels)) {
    set_error("arbx_dbscan: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  const Index* ix = &h->ix;
  if (ix->kind != KIND_POINT || ix->f64) { set_error("arbx_dbscan: fp32 POINT primitives only"); return ARBX_ERR_UNSUPPORTED; }
  const int64_t n = ix->n;
  if (n == 0) return ARBX_OK;
  cudaStream_t s = (cudaStream_t)stream;
  const unsigned grid = (unsigned)((n + 255) / 256);
  Scratch<float> selfq;
  Scratch<uint32_t> order;   // tree order is the traversal order: no query sort
  Scratch<int32_t> counts, uf;
  ARBX_TRY(selfq.alloc((size_t)n * (ix->dim + 1), s));
  ARBX_TRY(order.alloc((size_t)n, s));
  ARBX_TRY(counts.alloc((size_t)n, s));
  ARBX_TRY(uf.alloc((size_t)n, s));
  self_queries_kernel<<<grid, 256, 0, s>>>(ix->leaves, n, ix->dim, leaf_width(KIND_POINT, ix->dim), eps, selfq.p, order.p);
  ARBX_LAUNCH_CHECK();
  const DimTable* tab = dim_table(ix->dim);
  // 1. core test: capped neighbour count (the point itself included), early exit at min_pts
  SpatialArgs a{selfq.p, n, KIND_SPHERE, order.p, counts.p, nullptr, nullptr, nullptr, min_pts, nullptr, 0};
  ARBX_TRY(tab->spatial(ix, a, s));
  dbscan_init_kernel<<<grid, 256, 0, s>>>(counts.p, min_pts, n, uf.p);
  ARBX_LAUNCH_CHECK();
  // 2. every unordered pair within eps once (half traversal): unite core-core, attach borders
  a.rows = uf.p;
  a.pass = 3;
  a.self = 1;
  ARBX_TRY(tab->spatial(ix, a, s));
  // 3. labels
  dbscan_labels_kernel<<<grid, 256, 0, s>>>(uf.p, n, labels);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

static arbx_status spatial_impl(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind, int32_t limit,
                                int32_t* offsets, int32_t* indices, int64_t indices_capacity,
                                int64_t* total_host, arbx_stream stream, float self_radius) {
  const bool self = self_radius >= 0.f;
  if (self && h) nq = h->ix.n;
  if (!h || nq < 0 || bad_kind((int)qkind) || !offsets || (nq > 0 && !queries && !self) || indices_capacity < 0) {
    set_error("arbx_query_spatial: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  if (h->ix.f64) { set_error("arbx_query_spatial: the handle was built from fp64 coordinates, use the _f64 calls"); return ARBX_ERR_INVALID_ARG; }
  if (nq > kMaxCount) { set_error("arbx_query_spatial: nq > 2^30 unsupported"); return ARBX_ERR_UNSUPPORTED; }
  cudaStream_t s = (cudaStream_t)stream;
  const Index* ix = &h->ix;
  if (total_host) *total_host = 0;
  if (nq == 0 || ix->n == 0) {
    ARBX_CUDA(cudaMemsetAsync(offsets, 0, (size_t)(nq + 1) * sizeof(int32_t), s));
    return ARBX_OK;
  }
  QueryOrder order;
  Scratch<int32_t> counts, rows;
  Scratch<long long> total_dev;   // [0] total, [1] number of queries with more than `cap` matches
  Scratch<float> selfq;
  if (self) {
    ARBX_TRY(selfq.alloc((size_t)nq * (ix->dim + 1), s));
    ARBX_TRY(order.buf[0].alloc((size_t)nq, s));
    self_queries_kernel<<<(unsigned)((nq + 255) / 256), 256, 0, s>>>(ix->leaves, nq, ix->dim, leaf_width(KIND_POINT, ix->dim),
                                                                  self_radius, selfq.p, order.buf[0].p);
    ARBX_LAUNCH_CHECK();
    order.p = order.buf[0].p;
    queries = selfq.p;
  } else {
    ARBX_TRY(query_order(ix, queries, nq, (int)qkind, order, s));
  }
  L2Window l2(ix, s);
  ARBX_TRY(counts.alloc((size_t)nq, s));
  ARBX_TRY(total_dev.alloc(2, s));
  ARBX_CUDA(cudaMemsetAsync(total_dev.p, 0, 2 * sizeof(long long), s));
  const DimTable* tab = dim_table(ix->dim);
  // Single traversal when the caller wants the indices: the count pass also stores the first
  // `cap` matches of every query in a scratch row; after the scan the rows are copied into
  // their CSR slices and only queries with more than cap matches are traversed again.
  int cap = 0;
  if (indices && limit == 0) {
    const long long budget = (long long)g_cfg.store_budget_mb.load(std::memory_order_relaxed) << 20;
    for (int c = 64; c >= 16 && cap == 0; c >>= 1)
      if ((long long)nq * c * 4 <= budget) cap = c;
  }
  SpatialArgs a{queries, nq, (int)qkind, order.p, counts.p, nullptr, nullptr, nullptr, cap,
                reinterpret_cast<int*>(total_dev.p + 1), cap ? 2 : 0};
  // capped storage query: capped count (early exit) -> scan -> fill that stops at each count
  if (limit > 0) a.cap = limit;
  a.self = self ? 1 : 0;
  Scratch<uint32_t> ovf;
  if (cap) {
    ARBX_TRY(rows.alloc((size_t)nq * cap, s));
    ARBX_TRY(ovf.alloc((size_t)nq, s));
    a.rows = rows.p;
    a.ovf_list = ovf.p;
  }
  ARBX_TRY(tab->spatial(ix, a, s));
  ARBX_TRY(exclusive_scan_i32(counts.p, offsets, nq, total_dev.p, s));
  long long host[2] = {0, 0};
  int32_t rootw[2] = {0, 0};
  ARBX_CUDA(cudaMemcpyAsync(host, total_dev.p, sizeof(host), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaMemcpyAsync(rootw, ix->root, sizeof(rootw), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaStreamSynchronize(s));
  ARBX_TRY(check_build_fault(rootw[1]));
  const long long total = host[0];
  const int noverflow = (int)(host[1] & 0xffffffffLL);
  if (total_host) *total_host = total;
  if (total > 0x7fffffffLL) {
    set_error("arbx_query_spatial: total %lld exceeds INT32_MAX", total);
    return ARBX_ERR_OVERFLOW;
  }
  if (!indices) return ARBX_OK;
  if (indices_capacity < total) {
    set_error("arbx_query_spatial: capacity %lld < total %lld", (long long)indices_capacity, total);
    return ARBX_ERR_CAPACITY;
  }
  if (total == 0) return ARBX_OK;
  a.offsets = offsets;
  a.indices = indices;
  a.pass = 1;
  if (limit > 0) { a.cap = 0; a.stop_fill = 1; }
  if (cap) {
    ARBX_TRY(compact_rows(rows.p, cap, counts.p, offsets, indices, nq, s));
    if (noverflow == 0) return ARBX_OK;
    // second traversal for the overflowing queries only, packed into dense warps (their order in
    // the list follows block execution order, so neighbours stay roughly neighbours)
    // (not for the self-join, whose traversal needs the thread index = the query's leaf position)
    if (!self) { a.qorder = ovf.p; a.nq = noverflow; a.heavy = 1; }
  }
  return tab->spatial(ix, a, s);
}

static arbx_status knn_impl(arbx_handle h, const float* qpoints, int64_t nq, const int32_t* kq, int k,
                            int32_t* indices, float* distances, arbx_stream stream, const char* who) {
  if (!h || nq < 0 || k < 1 || (nq > 0 && (!qpoints || !indices))) {
    set_error("%s: invalid argument", who);
    return ARBX_ERR_INVALID_ARG;
  }
  if (h->ix.f64) { set_error("%s: the handle was built from fp64 coordinates, use the _f64 calls", who); return ARBX_ERR_INVALID_ARG; }
  if (k > ARBX_K_MAX) { set_error("%s: k=%d > ARBX_K_MAX=%d", who, k, ARBX_K_MAX); return ARBX_ERR_UNSUPPORTED; }
  if (nq > kMaxCount) { set_error("%s: nq > 2^30 unsupported", who); return ARBX_ERR_UNSUPPORTED; }
  if (nq == 0) return ARBX_OK;
  cudaStream_t s = (cudaStream_t)stream;
  const Index* ix = &h->ix;
  if (ix->n == 0) {
    fill_knn_empty_kernel<<<256, 256, 0, s>>>(indices, distances, nq * k);
    ARBX_LAUNCH_CHECK();
    return ARBX_OK;
  }
  QueryOrder order;
  ARBX_TRY(query_order(ix, qpoints, nq, KIND_POINT, order, s));
  KnnArgs a{qpoints, nq, k, kq, order.p, indices, distances};
  L2Window l2(ix, s);
  return dim_table(ix->dim)->knn(ix, a, s);
}

arbx_status arbx_query_knn(arbx_handle h, const float* qpoints, int64_t nq, int k, int32_t* indices,
                           float* distances, arbx_stream stream) {
  return knn_impl(h, qpoints, nq, nullptr, k, indices, distances, stream, "arbx_query_knn");
}

arbx_status arbx_query_knn_var(arbx_handle h, const float* qpoints, int64_t nq, const int32_t* k_per_query,
                               int kmax, int32_t* indices, float* distances, arbx_stream stream) {
  if (nq > 0 && !k_per_query) { set_error("arbx_query_knn_var: null k_per_query"); return ARBX_ERR_INVALID_ARG; }
  return knn_impl(h, qpoints, nq, k_per_query, kmax, indices, distances, stream, "arbx_query_knn_var");
}

// ---- fp64 coordinates (NEXT-4): exact fp64 leaf tests over the fp32 tree, see f64.cu ----------------
arbx_status arbx_build_f64(const double* prims, int64_t n, int dim, arbx_kind kind, arbx_stream stream,
                           arbx_handle* out) {
  if (!out || n < 0 || dim < 1 || dim > ARBX_MAX_DIM || bad_kind((int)kind) || (n > 0 && !prims)) {
    set_error("arbx_build_f64: invalid argument (n=%lld dim=%d kind=%d)", (long long)n, dim, (int)kind);
    return ARBX_ERR_INVALID_ARG;
  }
  if (n > kMaxCount) { set_error("arbx_build_f64: n > 2^30 unsupported"); return ARBX_ERR_UNSUPPORTED; }
  cudaStream_t s = (cudaStream_t)stream;
  arbx_index_s* h = new arbx_index_s();
  h->ix.leaf_max = std::max(1, std::min(64, g_cfg.leaf_max.load(std::memory_order_relaxed)));
  arbx_status st = f64_build(prims, n, dim, (int)kind, s, &h->ix);
  if (st != ARBX_OK) {
    free_index(&h->ix, s);
    delete h;
    return st;
  }
  *out = h;
  return ARBX_OK;
}

static arbx_status f64_query_prologue(arbx_handle h, const double* queries, int64_t nq, int qkind, const char* who,
                                      Scratch<float>& qboxes, QueryOrder& order, cudaStream_t s) {
  if (!h->ix.f64) { set_error("%s: the handle was built from fp32 coordinates", who); return ARBX_ERR_INVALID_ARG; }
  if (nq > kMaxCount) { set_error("%s: nq > 2^30 unsupported", who); return ARBX_ERR_UNSUPPORTED; }
  ARBX_TRY(qboxes.alloc((size_t)nq * 2 * h->ix.dim, s));
  ARBX_TRY(f64_qboxes(queries, nq, h->ix.dim, qkind, qboxes.p, s));
  return query_order(&h->ix, qboxes.p, nq, KIND_BOX, order, s);   // the curve order of the fp32 boxes
}

arbx_status arbx_query_count_f64(arbx_handle h, const double* queries, int64_t nq, arbx_kind qkind,
                                 int32_t* counts, arbx_stream stream) {
  if (!h || nq < 0 || bad_kind((int)qkind) || (nq > 0 && (!queries || !counts))) {
    set_error("arbx_query_count_f64: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  if (nq == 0) return ARBX_OK;
  cudaStream_t s = (cudaStream_t)stream;
  if (h->ix.f64 && h->ix.n == 0) { ARBX_CUDA(cudaMemsetAsync(counts, 0, (size_t)nq * sizeof(int32_t), s)); return ARBX_OK; }
  Scratch<float> qboxes;
  QueryOrder order;
  ARBX_TRY(f64_query_prologue(h, queries, nq, (int)qkind, "arbx_query_count_f64", qboxes, order, s));
  return f64_spatial(&h->ix, queries, qboxes.p, order.p, nq, (int)qkind, counts, nullptr, nullptr, 0, s);
}

arbx_status arbx_query_spatial_f64(arbx_handle h, const double* queries, int64_t nq, arbx_kind qkind,
                                   int32_t* offsets, int32_t* indices, int64_t indices_capacity,
                                   int64_t* total_host, arbx_stream stream) {
  if (!h || nq < 0 || bad_kind((int)qkind) || !offsets || (nq > 0 && !queries) || indices_capacity < 0) {
    set_error("arbx_query_spatial_f64: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  cudaStream_t s = (cudaStream_t)stream;
  if (total_host) *total_host = 0;
  if (nq == 0 || (h->ix.f64 && h->ix.n == 0)) {
    if (!h->ix.f64) { set_error("arbx_query_spatial_f64: the handle was built from fp32 coordinates"); return ARBX_ERR_INVALID_ARG; }
    ARBX_CUDA(cudaMemsetAsync(offsets, 0, (size_t)(nq + 1) * sizeof(int32_t), s));
    return ARBX_OK;
  }
  Scratch<float> qboxes;
  QueryOrder order;
  ARBX_TRY(f64_query_prologue(h, queries, nq, (int)qkind, "arbx_query_spatial_f64", qboxes, order, s));
  Scratch<int32_t> counts;
  Scratch<long long> total_dev;
  ARBX_TRY(counts.alloc((size_t)nq, s));
  ARBX_TRY(total_dev.alloc(2, s));
  ARBX_CUDA(cudaMemsetAsync(total_dev.p, 0, 2 * sizeof(long long), s));
  ARBX_TRY(f64_spatial(&h->ix, queries, qboxes.p, order.p, nq, (int)qkind, counts.p, nullptr, nullptr, 0, s));
  ARBX_TRY(exclusive_scan_i32(counts.p, offsets, nq, total_dev.p, s));
  long long total = 0;
  int32_t rootw[2] = {0, 0};
  ARBX_CUDA(cudaMemcpyAsync(&total, total_dev.p, sizeof(total), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaMemcpyAsync(rootw, h->ix.root, sizeof(rootw), cudaMemcpyDeviceToHost, s));
  ARBX_CUDA(cudaStreamSynchronize(s));
  ARBX_TRY(check_build_fault(rootw[1]));
  if (total_host) *total_host = total;
  if (total > 0x7fffffffLL) { set_error("arbx_query_spatial_f64: total %lld exceeds INT32_MAX", total); return ARBX_ERR_OVERFLOW; }
  if (!indices) return ARBX_OK;
  if (indices_capacity < total) {
    set_error("arbx_query_spatial_f64: capacity %lld < total %lld", (long long)indices_capacity, total);
    return ARBX_ERR_CAPACITY;
  }
  if (total == 0) return ARBX_OK;
  return f64_spatial(&h->ix, queries, qboxes.p, order.p, nq, (int)qkind, nullptr, offsets, indices, 1, s);
}

__global__ void fill_knn_empty_f64_kernel(int32_t* idx, double* dist, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    idx[i] = -1;
    if (dist) dist[i] = INFINITY;
  }
}

arbx_status arbx_query_knn_f64(arbx_handle h, const double* qpoints, int64_t nq, int k, int32_t* indices,
                               double* distances, arbx_stream stream) {
  if (!h || nq < 0 || k < 1 || (nq > 0 && (!qpoints || !indices))) {
    set_error("arbx_query_knn_f64: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  if (k > ARBX_K_MAX) { set_error("arbx_query_knn_f64: k=%d > ARBX_K_MAX=%d", k, ARBX_K_MAX); return ARBX_ERR_UNSUPPORTED; }
  if (nq == 0) return ARBX_OK;
  cudaStream_t s = (cudaStream_t)stream;
  if (h->ix.f64 && h->ix.n == 0) {
    fill_knn_empty_f64_kernel<<<256, 256, 0, s>>>(indices, distances, nq * k);
    ARBX_LAUNCH_CHECK();
    return ARBX_OK;
  }
  Scratch<float> qboxes;
  QueryOrder order;
  ARBX_TRY(f64_query_prologue(h, qpoints, nq, KIND_POINT, "arbx_query_knn_f64", qboxes, order, s));
  return f64_knn(&h->ix, qpoints, order.p, nq, k, indices, distances, s);
}

// ---- arbx_query_count_noalloc: the count-only query without any allocation -------------------------
// Its scratch (query codes and positions, both ping-pong halves, and the sort's meta words) lives in
// ONE file-scope device array: every GPU that loads the library holds these 17.8 MB until exit.
// In host code the array's name is only a stand-in, not a device address: the address is fetched
// once per device, with that device current, by cudaGetSymbolAddress, and that pointer is what the
// kernels get.
constexpr int64_t kNoAllocMaxQueries = ARBX_NOALLOC_MAX_QUERIES;
constexpr size_t kNoAllocMetaWords = 4 * 256 + 8 + 4 * (size_t)((kNoAllocMaxQueries + 4095) / 4096) * 256;   // 4 passes of 8 bits
constexpr size_t kNoAllocWords = 4 * (size_t)kNoAllocMaxQueries + kNoAllocMetaWords;
static __device__ __align__(256) uint32_t g_noalloc_scratch[kNoAllocWords];

static std::once_flag g_noalloc_once[64];
static uint32_t* g_noalloc_ptr[64];
static cudaError_t g_noalloc_err[64];

static arbx_status noalloc_scratch(uint32_t** out) {
  int dev = 0;
  ARBX_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) { set_error("arbx_query_count_noalloc: device %d out of range", dev); return ARBX_ERR_UNSUPPORTED; }
  std::call_once(g_noalloc_once[dev], [dev] {   // the calling thread has `dev` current
    void* p = nullptr;
    g_noalloc_err[dev] = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    g_noalloc_ptr[dev] = g_noalloc_err[dev] == cudaSuccess ? static_cast<uint32_t*>(p) : nullptr;
  });
  if (!g_noalloc_ptr[dev]) {
    set_error("arbx_query_count_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(g_noalloc_err[dev]));
    return ARBX_ERR_CUDA;
  }
  *out = g_noalloc_ptr[dev];
  return ARBX_OK;
}

arbx_status arbx_query_count_noalloc(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                                     int32_t* counts, arbx_stream stream) {
  if (!h || nq < 0 || bad_kind((int)qkind) || (nq > 0 && (!queries || !counts))) {
    set_error("arbx_query_count_noalloc: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  if (h->ix.f64) { set_error("arbx_query_count_noalloc: fp32 handles only"); return ARBX_ERR_INVALID_ARG; }
  if (nq > kNoAllocMaxQueries) {
    set_error("arbx_query_count_noalloc: nq = %lld exceeds ARBX_NOALLOC_MAX_QUERIES = %lld (the fixed scratch array); "
              "use arbx_query_count or split the batch", (long long)nq, (long long)kNoAllocMaxQueries);
    return ARBX_ERR_UNSUPPORTED;
  }
  if (nq == 0) return ARBX_OK;
  cudaStream_t s = (cudaStream_t)stream;
  const Index* ix = &h->ix;
  if (ix->n == 0) { ARBX_CUDA(cudaMemsetAsync(counts, 0, (size_t)nq * sizeof(int32_t), s)); return ARBX_OK; }
  const uint32_t* order = nullptr;
  if (!ix->brute) {   // Q1 + Q2 in the static scratch (a brute-force index scans everything: no order needed)
    uint32_t* base = nullptr;
    ARBX_TRY(noalloc_scratch(&base));
    uint32_t* codes = base;
    uint32_t* codes_alt = base + kNoAllocMaxQueries;
    uint32_t* ord0 = base + 2 * kNoAllocMaxQueries;
    uint32_t* ord1 = base + 3 * kNoAllocMaxQueries;
    uint32_t* meta = base + 4 * kNoAllocMaxQueries;
    int key_bits = 32;
    ARBX_TRY(dim_table(ix->dim)->qcode(ix, queries, nq, (int)qkind, codes, &key_bits, s));
    uint32_t *kout = nullptr, *vout = nullptr;
    ARBX_TRY(radix_sort_u32_noalloc(codes, codes_alt, ord0, ord1, nq, key_bits, meta, kNoAllocMetaWords, s, &kout, &vout));
    order = vout;
  }
  SpatialArgs a{queries, nq, (int)qkind, order, counts, nullptr, nullptr, nullptr, 0, nullptr, 0};
  return dim_table(ix->dim)->spatial(ix, a, s);
}

arbx_status arbx_sort_pairs(void* keys, uint32_t* values, int64_t n, int key_bytes, int key_bits,
                            arbx_stream stream) {
  if (n < 0 || (n > 0 && !keys) || (key_bytes != 4 && key_bytes != 8) || key_bits < 1 || key_bits > 8 * key_bytes) {
    set_error("arbx_sort_pairs: invalid argument");
    return ARBX_ERR_INVALID_ARG;
  }
  cudaStream_t s = (cudaStream_t)stream;
  if (n == 0) return ARBX_OK;
  Scratch<unsigned char> kalt;
  Scratch<uint32_t> valt;
  ARBX_TRY(kalt.alloc((size_t)n * key_bytes, s));
  if (values) ARBX_TRY(valt.alloc((size_t)n, s));
  void* kout = keys;
  uint32_t* vout = values;
  if (key_bytes == 8) {
    unsigned long long* ko = nullptr;
    ARBX_TRY(radix_sort_u64((unsigned long long*)keys, (unsigned long long*)kalt.p, values, valt.p, false, n, key_bits, s, &ko, &vout));
    kout = ko;
  } else {
    uint32_t* ko = nullptr;
    ARBX_TRY(radix_sort_u32((uint32_t*)keys, (uint32_t*)kalt.p, values, valt.p, false, n, key_bits, s, &ko, &vout));
    kout = ko;
  }
  if (kout != keys) {   // odd number of passes: the result sits in the scratch buffers
    ARBX_CUDA(cudaMemcpyAsync(keys, kout, (size_t)n * key_bytes, cudaMemcpyDeviceToDevice, s));
    if (values) ARBX_CUDA(cudaMemcpyAsync(values, vout, (size_t)n * sizeof(uint32_t), cudaMemcpyDeviceToDevice, s));
  }
  return ARBX_OK;
}

arbx_status arbx_debug_set(const char* key, double value) {
  if (!key) { set_error("arbx_debug_set: null key"); return ARBX_ERR_INVALID_ARG; }
  const std::string k(key);
  const int iv = (int)value;
  if (k == "leaf_max") g_cfg.leaf_max.store(iv);
  else if (k == "store_budget_mb") g_cfg.store_budget_mb.store(iv);
  else if (k == "traversal") g_cfg.traversal.store(iv);
  else if (k == "qbits") g_cfg.qbits.store(iv);
  else if (k == "code_bits") g_cfg.code_bits.store(iv);
  else if (k == "brute_max") g_cfg.brute_max.store(iv);
  else if (k == "l2_persist") g_cfg.l2_persist.store(iv);
  else if (k == "gather") g_cfg.gather.store(iv);
  else if (k == "packet_alpha") g_cfg.packet_alpha.store((float)value);
  else if (k == "pool_keep_mb") {
    g_pool_keep_mb.store((long long)value);
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaMemPool_t pool = pool_for(dev)) pool_apply_threshold(pool);
  } else if (k == "reset") {
    g_cfg.leaf_max.store(16); g_cfg.store_budget_mb.store(4096); g_cfg.traversal.store(0); g_cfg.qbits.store(0);
    g_cfg.code_bits.store(0); g_cfg.brute_max.store(-1); g_cfg.gather.store(0); g_cfg.l2_persist.store(0); g_cfg.packet_alpha.store(-1.f);
  } else {
    set_error("arbx_debug_set: unknown key '%s'", key);
    return ARBX_ERR_INVALID_ARG;
  }
  return ARBX_OK;
}

#ifdef ARBX_STATS
extern "C++" { namespace arbx { void knn_stats_read(unsigned long long* out); } }
extern "C" __attribute__((visibility("default"))) void arbx_debug_knn_stats(unsigned long long* out) { arbx::knn_stats_read(out); }
#endif

arbx_status arbx_trim(int64_t keep_bytes) {
  if (keep_bytes < 0) { set_error("arbx_trim: keep_bytes < 0"); return ARBX_ERR_INVALID_ARG; }
  int dev = 0;
  cudaGetDevice(&dev);
  { std::lock_guard<std::mutex> g(g_cache_mu); cache_evict_locked((size_t)keep_bytes); }
  if (cudaMemPool_t pool = pool_for(dev)) {
    ARBX_CUDA(cudaDeviceSynchronize());   // the evicted blocks are freed in stream order
    ARBX_CUDA(cudaMemPoolTrimTo(pool, (size_t)keep_bytes));
  }
  return ARBX_OK;
}

arbx_status arbx_debug_validate(arbx_handle h, int64_t* violations_host, arbx_stream stream) {
  if (!h || !violations_host) { set_error("arbx_debug_validate: null argument"); return ARBX_ERR_INVALID_ARG; }
  return validate_index(&h->ix, violations_host, (cudaStream_t)stream);
}

int64_t arbx_launch_count(void) { return (int64_t)g_launches.load(); }

arbx_status arbx_profile_enable(int on) {
  g_prof_on.store(on ? 1 : 0);
  return ARBX_OK;
}

int arbx_profile_num_kernels(void) { return K_NUM_; }

const char* arbx_profile_kernel_name(int id) { return id >= 0 && id < K_NUM_ ? kKernelNames[id] : ""; }

arbx_status arbx_profile_read(double* ms_host, int64_t* calls_host, int capacity) {
  if (!ms_host || !calls_host || capacity < K_NUM_) {
    set_error("arbx_profile_read: need capacity >= %d", (int)K_NUM_);
    return ARBX_ERR_INVALID_ARG;
  }
  for (int i = 0; i < capacity; ++i) { ms_host[i] = 0.0; calls_host[i] = 0; }
  std::lock_guard<std::mutex> g(g_prof_mu);
  arbx_status st = ARBX_OK;
  for (const ProfRec& r : g_prof_done) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(r.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.a, r.b);
    if (e != cudaSuccess) { set_error("arbx_profile_read: %s", cudaGetErrorString(e)); st = ARBX_ERR_CUDA; }
    ms_host[r.id] += ms;
    calls_host[r.id] += 1;
    g_prof_pool.push_back(r.a);
    g_prof_pool.push_back(r.b);
  }
  g_prof_done.clear();
  return st;
}

const char* arbx_status_string(arbx_status s) {
  switch (s) {
    case ARBX_OK: return "ARBX_OK";
    case ARBX_ERR_INVALID_ARG: return "ARBX_ERR_INVALID_ARG";
    case ARBX_ERR_UNSUPPORTED: return "ARBX_ERR_UNSUPPORTED";
    case ARBX_ERR_CAPACITY: return "ARBX_ERR_CAPACITY";
    case ARBX_ERR_OVERFLOW: return "ARBX_ERR_OVERFLOW";
    case ARBX_ERR_CUDA: return "ARBX_ERR_CUDA";
    case ARBX_ERR_OOM: return "ARBX_ERR_OOM";
  }
  return "ARBX_ERR_UNKNOWN";
}

const char* arbx_last_error(void) { return t_err; }

}  // extern "C"
