// common.cuh -- shared declarations of the CUDA path (sm_100a).  Internal, not part of the ABI.
//
// Data layout in HBM:
//   leaves : sorted (space-filling-curve order) array, one record per primitive, stride
//            LEAF_W floats (multiple of 4 => every record is 16-byte aligned, LDG.128):
//              POINT  x[D], idx            (D=3: 16 B, the paper's 16-byte leaf)
//              BOX    lo[D], hi[D], idx
//              SPHERE c[D], R, idx
//            idx = position in the caller's array; bit 31 set marks the LAST record of a
//            leaf range (a collapsed subtree of <= leaf_max primitives).
//   nodes  : one record per internal node, id = split position s (between sorted leaves s and
//            s+1), stride 4*(D+1) floats:  lo0[D], hi0[D], lo1[D], hi1[D], c0, c1, l, r.
//            A node stores the boxes of its TWO CHILDREN, so one fetch decides both descents.
//            child ref c >= 0: internal node id; c < 0: leaf range starting at leaf ~c.
//            [l, r] = the node's own range of sorted leaf positions (child 0 covers [l, s],
//            child 1 covers [s+1, r]); the self-join, the packet traversals and the validator
//            read it.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/arbx.h"

namespace arbx {

constexpr int KIND_POINT = 0, KIND_BOX = 1, KIND_SPHERE = 2;
constexpr uint32_t LEAF_END = 0x80000000u;
constexpr int STACK_DEPTH = 96;   // <= 64 code bits + 31 index tie-break bits + 1

__host__ __device__ constexpr int prim_width(int kind, int D) {
  return kind == KIND_POINT ? D : kind == KIND_BOX ? 2 * D : D + 1;
}
__host__ __device__ constexpr int leaf_width(int kind, int D) {
  return (prim_width(kind, D) + 1 + 3) / 4 * 4;
}
__host__ __device__ constexpr int node_width(int D) { return 4 * (D + 1); }

struct Index {
  int64_t n = 0;
  int dim = 0;
  int kind = 0;
  int leaf_max = 1;
  int code_bits = 0;            // bits per axis of the primitive codes the tree was built from
  bool brute = false;           // tiny index: no tree, queries scan the leaves (brute.cu)
  float* leaves = nullptr;      // n * leaf_width floats
  float* nodes = nullptr;       // max(n-1,0) * node_width floats
  float* bounds = nullptr;      // 2*dim floats: lo[dim], hi[dim] of all primitives
  int32_t* root = nullptr;      // 2 ints (device): [0] root child ref, [1] build fault flags
  // fp64 coordinates (f64.cu): the tree is a BOX tree over outward-rounded fp32 boxes; the fp64
  // rows of the caller's kind `kind64` sit beside it in leaf order
  bool f64 = false;
  int kind64 = 0;
  double* rows64 = nullptr;
};
constexpr int BUILD_FAULT_OPEN_OVERFLOW = 1;   // hierarchy: more parked subtrees than open_cap

// Test / experiment knobs, set through arbx_debug_set (never read from the environment).
struct DebugCfg {
  std::atomic<int> leaf_max{16};        // primitives per collapsed leaf range
  std::atomic<int> store_budget_mb{4096};  // scratch rows of the single-traversal storage query
  std::atomic<int> traversal{0};        // 0 per-warp choice, 1 one query per lane, 2 packets
  std::atomic<int> qbits{0};            // query-code bits per axis kept for the query sort (0 = all)
  std::atomic<int> code_bits{0};        // primitive-code bits per axis (0 = adapted to n)
  std::atomic<int> brute_max{-1};       // n <= brute_max builds a brute-force index (-1 = default)
  std::atomic<int> gather{0};           // 1: arbx_query_count materialises the sorted queries (Q3 experiment)
  std::atomic<int> l2_persist{0};       // 1: persisting-L2 window over the node array during queries
  std::atomic<float> packet_alpha{-1.f};   // packet threshold (< 0 = default per kind / dim)
};
extern DebugCfg g_cfg;

// ---- error plumbing ----------------------------------------------------------------------
void set_error(const char* fmt, ...);
extern std::atomic<long long> g_launches;
inline void count_launch(int k = 1) { g_launches.fetch_add(k, std::memory_order_relaxed); }

#define ARBX_CUDA(expr)                                                                  \
  do {                                                                                   \
    cudaError_t e__ = (expr);                                                            \
    if (e__ != cudaSuccess) {                                                            \
      ::arbx::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, \
                        __LINE__);                                                       \
      return e__ == cudaErrorMemoryAllocation ? ARBX_ERR_OOM : ARBX_ERR_CUDA;            \
    }                                                                                    \
  } while (0)

// ---- per-kernel timing (arbx_profile_*): CUDA events on the launching stream ---------------
enum KernelId {
  K_BOUNDS = 0, K_CODES, K_SORT_HIST, K_SORT_PASS, K_LEAVES, K_HIERARCHY, K_QCODE, K_QSORT_HIST,
  K_QSORT_PASS, K_SPATIAL_COUNT, K_SCAN, K_SPATIAL_FILL, K_KNN, K_MISC, K_NUM_
};
bool prof_enabled();
void prof_begin(int id, cudaStream_t s);
void prof_end(int id, cudaStream_t s);
struct ProfScope {   // brackets the launches of one hot-path step with a pair of events
  int id; cudaStream_t s; bool on;
  ProfScope(int id_, cudaStream_t s_) : id(id_), s(s_), on(prof_enabled()) { if (on) prof_begin(id, s); }
  ~ProfScope() { if (on) prof_end(id, s); }
};

#define ARBX_LAUNCH_CHECK()                                                              \
  do {                                                                                   \
    ::arbx::count_launch();                                                              \
    ARBX_CUDA(cudaGetLastError());                                                       \
  } while (0)

#define ARBX_TRY(expr)                        \
  do {                                        \
    arbx_status s__ = (expr);                 \
    if (s__ != ARBX_OK) return s__;           \
  } while (0)

// stream-ordered scratch (never stored in the handle)
arbx_status scratch_alloc(void** p, size_t bytes, cudaStream_t s);
void scratch_free(void* p, cudaStream_t s);

template <class T>
struct Scratch {   // RAII: released in stream order when the call returns
  T* p = nullptr;
  cudaStream_t s = nullptr;
  Scratch() = default;
  Scratch(const Scratch&) = delete;
  Scratch& operator=(const Scratch&) = delete;
  ~Scratch() { if (p) scratch_free(p, s); }
  arbx_status alloc(size_t count, cudaStream_t stream) {
    s = stream;
    return scratch_alloc((void**)&p, (count ? count : 1) * sizeof(T), stream);
  }
  T* release() { T* q = p; p = nullptr; return q; }
};

// ---- internal entry points (one per translation unit) --------------------------------------
// sort.cu: stable LSD radix sort of bits [0,key_bits) with 8-bit digits.  The caller provides
// both ping-pong buffers; *keys_out / *vals_out tell which of them holds the result (no copy
// back after an odd number of passes).  iota_vals: the input values are the positions 0..n-1
// and are not read (saves writing and re-reading an iota).  vals == nullptr sorts keys only.
arbx_status radix_sort_u64(unsigned long long* keys, unsigned long long* keys_alt, uint32_t* vals,
                           uint32_t* vals_alt, bool iota_vals, int64_t n, int key_bits,
                           cudaStream_t s, unsigned long long** keys_out, uint32_t** vals_out);
arbx_status radix_sort_u32(uint32_t* keys, uint32_t* keys_alt, uint32_t* vals, uint32_t* vals_alt,
                           bool iota_vals, int64_t n, int key_bits, cudaStream_t s,
                           uint32_t** keys_out, uint32_t** vals_out);

// sort.cu: the 32-bit query sort (values = positions) on caller-provided buffers only, `meta` included
size_t sort_meta_words(int64_t n, int key_bits);
arbx_status radix_sort_u32_noalloc(uint32_t* keys, uint32_t* keys_alt, uint32_t* vals, uint32_t* vals_alt, int64_t n,
                                   int key_bits, uint32_t* meta, size_t meta_capacity_words, cudaStream_t s,
                                   uint32_t** keys_out, uint32_t** vals_out);

// build.cu
arbx_status build_index(const float* prims, int64_t n, int dim, int kind, cudaStream_t s,
                        Index* ix);
arbx_status validate_index(const Index* ix, int64_t* violations_host, cudaStream_t s);

// query_dN.cu (one TU per dimension), dispatched from query.cu
// One spatial traversal pass.  pass 0: counts[q] = matches (cap > 0: min(matches, cap), with
// early exit).  pass 2: the same, and the first
// `cap` matches of query q are stored in rows[q*cap ..]; *overflow counts the queries with
// more than cap matches and ovf_list names them (so that pass 1 runs on dense warps).  pass 1: fill indices[offsets[q] ..]; with cap > 0 only the queries
// whose counts[q] > cap are traversed (the others are copied from rows by compact_rows).
struct SpatialArgs {
  const float* queries; int64_t nq; int qkind; const uint32_t* qorder;
  int32_t* counts; const int32_t* offsets; int32_t* indices;
  int32_t* rows; int cap; int* overflow; int pass;
  uint32_t* ovf_list = nullptr;   // pass 2: caller's indices of the queries with more than cap matches
  int heavy = 0;       // pass 1 only: qorder lists the overflowing queries; one warp per query
  int stop_fill = 0;   // pass 1 only: query q stops after counts[q] hits (capped storage query)
  int self = 0;        // self-join: query t is the leaf at sorted position t; report later positions only
};
using spatial_fn = arbx_status (*)(const Index*, const SpatialArgs&, cudaStream_t);
// kNN: rows of k entries; kq (optional, device) gives every query its own k_q <= k, the rest of
// its row is padding (-1 / +inf).
struct KnnArgs {
  const float* qpoints; int64_t nq; int k; const int32_t* kq; const uint32_t* qorder;
  int32_t* indices; float* distances;
};
using knn_fn = arbx_status (*)(const Index*, const KnnArgs&, cudaStream_t);
using qcode_fn = arbx_status (*)(const Index*, const float* queries, int64_t nq, int qkind_or_point,
                                 uint32_t* codes, int* key_bits, cudaStream_t);
struct DimTable { spatial_fn spatial; knn_fn knn; qcode_fn qcode; };
const DimTable* dim_table(int dim);

// f64.cu: fp64 coordinates as exact fp64 leaf tests over the fp32 tree
arbx_status f64_build(const double* prims, int64_t n, int dim, int kind, cudaStream_t s, Index* ix);
arbx_status f64_qboxes(const double* queries, int64_t nq, int dim, int qkind, float* qboxes, cudaStream_t s);
arbx_status f64_spatial(const Index* ix, const double* queries, const float* qboxes, const uint32_t* qorder, int64_t nq,
                        int qkind, int32_t* counts, const int32_t* offsets, int32_t* indices, int fill, cudaStream_t s);
arbx_status f64_knn(const Index* ix, const double* qpoints, const uint32_t* qorder, int64_t nq, int k, int32_t* indices,
                    double* distances, cudaStream_t s);

// scan.cu: offsets[0..nq] = exclusive scan of counts[0..nq); *total (device, int64) = sum
arbx_status exclusive_scan_i32(const int32_t* counts, int32_t* offsets, int64_t nq,
                               long long* total_dev, cudaStream_t s);
// scan.cu: indices[offsets[q] + j] = rows[q*cap + j] for j < counts[q], for every q with counts[q] <= cap
arbx_status compact_rows(const int32_t* rows, int cap, const int32_t* counts, const int32_t* offsets,
                         int32_t* indices, int64_t nq, cudaStream_t s);

}  // namespace arbx
