/* arbx.h -- C ABI of the B200-native (sm_100a) linear-BVH build + batched search library.
 *
 * The operations are those of arXiv 2507.23700 ("The ArborX library: version 2.0"),
 * cited below as PAPER.md:Lnn (line of /root/reference/PAPER.md) + section:
 *   - an index is built over user primitives (§2.2 "BVH ... constructor");
 *   - spatial queries return, per query, the primitives that satisfy it, as
 *     `indices` + `offsets` (CSR) (§2.1.1; L112-115, §2.2 query overload 3);
 *   - the same search with a pure callback stores nothing; our instance of it counts
 *     (§2.2 query overload 1; L303 Table 1 "Query (count)");
 *   - nearest queries return the k closest primitives, distance measured to the stored
 *     geometry ("fine" search, §2.1.2);
 *   - every call takes an execution space = CUDA stream.
 *
 * Conventions
 *   Pointers marked DEVICE must be device memory accessible from the current CUDA device;
 *   pointers marked HOST are ordinary host memory.  The caller owns every buffer it passes;
 *   the library never returns device memory.  The handle owns the tree and a private copy
 *   of the geometry ("behave like a container"): `prims` may be released once
 *   the build has completed on `stream`.  The tree and all per-call scratch come from a
 *   stream-ordered memory pool that the library creates for itself on each device (the
 *   process's default pool and the caller's allocator are not touched); scratch is released
 *   before the call returns (in stream order) and stays cached in that pool up to 16 GiB
 *   (arbx_trim hands the cache back to the driver).  Nothing per-query is stored in the
 *   handle, so several queries may run concurrently on one handle from different streams
 *   (PAPER.md:L77, L128).
 *   Using a handle on another stream than the one it was built on requires the caller to
 *   order that stream after the build (event or synchronize).
 *
 *   Layout (row-major fp32):   POINT : dim floats            (coordinates)
 *                              BOX   : 2*dim floats          (lo[dim] then hi[dim])
 *                              SPHERE: dim+1 floats          (centre[dim] then radius)
 *   1 <= dim <= 10.   0 <= n <= 2^30.   0 <= nq <= 2^30.
 *
 *   All geometric tests are CLOSED (touching counts), Euclidean, no self-exclusion.
 *   NaN/Inf coordinates and inverted boxes are not validated (results undefined).
 *   A SPHERE query with negative radius matches nothing.
 *
 *   Errors: every entry point returns an arbx_status; nothing throws or aborts.
 *   arbx_last_error() gives a thread-local human-readable detail for the last failure.
 */
#ifndef ARBX_H_
#define ARBX_H_

#include <stdint.h>

#if defined(__GNUC__)
#define ARBX_API __attribute__((visibility("default")))
#else
#define ARBX_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct arbx_index_s* arbx_handle;   /* opaque; owns the device tree */
typedef void* arbx_stream;                  /* a cudaStream_t (NULL = legacy default stream) */

typedef enum { ARBX_POINT = 0, ARBX_BOX = 1, ARBX_SPHERE = 2 } arbx_kind;

typedef enum {
  ARBX_OK = 0,
  ARBX_ERR_INVALID_ARG = 1, /* null pointer with non-zero count, dim/kind/k out of range, n<0 */
  ARBX_ERR_UNSUPPORTED = 2, /* n or nq > 2^30, k > ARBX_K_MAX                                 */
  ARBX_ERR_CAPACITY = 3,    /* indices_capacity < total (offsets and *total_host are valid)   */
  ARBX_ERR_OVERFLOW = 4,    /* total > INT32_MAX: int32 offsets cannot hold it                */
  ARBX_ERR_CUDA = 5,        /* a CUDA runtime call failed (detail in arbx_last_error)         */
  ARBX_ERR_OOM = 6          /* device allocation failed                                       */
} arbx_status;

#define ARBX_MAX_DIM 10
#define ARBX_K_MAX 256      /* k <= 32 runs on the register heap, 32 < k <= 256 on a local-memory heap */

/* Build the index (PAPER.md:L101-103 constructor; internals L293-295: space-filling codes,
 * sort, bottom-up hierarchy with bounding volumes).  Asynchronous on `stream` except for
 * allocation.  prims: DEVICE, n rows in the layout of `kind`.  n == 0 gives a valid empty
 * handle (PAPER.md:L120 empty()).  *out is written only on ARBX_OK.                        */
ARBX_API arbx_status arbx_build(const float* prims, int64_t n, int dim, arbx_kind kind,
                       arbx_stream stream, arbx_handle* out);

/* Release the handle's device memory in stream order on `stream`. NULL is accepted.        */
ARBX_API arbx_status arbx_destroy(arbx_handle h, arbx_stream stream);

/* PAPER.md:L119 size().  HOST out pointer; no synchronisation.                              */
ARBX_API arbx_status arbx_size(arbx_handle h, int64_t* n);

/* PAPER.md:L121 bounds(): bounding box of all primitives.  lo_host/hi_host: HOST, dim floats
 * each.  Synchronises `stream`.  For an empty index lo=+inf, hi=-inf.                        */
ARBX_API arbx_status arbx_bounds(arbx_handle h, float* lo_host, float* hi_host, arbx_stream stream);

/* Count-only search = the pure-callback query whose callback increments a counter
 * (PAPER.md:L104-106, L131, L303).  qkind SPHERE = radius search (centre, r) (PAPER.md:L69
 * "a pair of a query point and a radius"); BOX = box intersection; POINT =
 * primitives containing the point.  queries: DEVICE, nq rows in the layout
 * of qkind with the handle's dim.  counts: DEVICE int32[nq], counts[q] = number of
 * primitives matching query q (caller's query order).  Asynchronous on `stream`.            */
ARBX_API arbx_status arbx_query_count(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                             int32_t* counts, arbx_stream stream);

/* Capped count = the pure-callback query whose callback stops a query's traversal once it
 * has seen `limit` matches (PAPER.md:L174 CallbackTreeTraversalControl::early_exit; L180-209
 * the CountUpToN example; L306).  counts[q] = min(matches of query q, limit), limit >= 1.
 * Reading A20: the paper's example post-increments and therefore stores
 * min(total, n+1); this call returns min(total, limit).  Other arguments as arbx_query_count. */
ARBX_API arbx_status arbx_query_count_upto(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                                  int32_t limit, int32_t* counts, arbx_stream stream);

/* Storage search (PAPER.md:L69 v1 "indices and offsets"; L112-115 overload 3).
 * offsets: DEVICE int32[nq+1]; offsets[0]=0, offsets[q+1]-offsets[q] = matches of query q,
 * offsets[nq] = total.  indices: DEVICE int32[indices_capacity] or NULL; the slice
 * [offsets[q], offsets[q+1]) holds the positions, in the caller's prims array, of the
 * primitives matching query q, in unspecified order.  total_host: HOST int64, may be NULL.
 * The call enqueues count + scan, synchronises `stream` ONCE to learn the total, then:
 *   indices == NULL               -> returns ARBX_OK (offsets and *total_host valid);
 *   total > INT32_MAX             -> ARBX_ERR_OVERFLOW (*total_host valid, offsets not);
 *   indices_capacity < total      -> ARBX_ERR_CAPACITY (offsets and *total_host valid);
 *   otherwise enqueues the fill pass and returns without a second synchronisation.          */
ARBX_API arbx_status arbx_query_spatial(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                               int32_t* offsets, int32_t* indices, int64_t indices_capacity,
                               int64_t* total_host, arbx_stream stream);

/* Capped storage search: as arbx_query_spatial, but every query keeps at most `limit`
 * (>= 1) of its matches and stops its traversal there (PAPER.md:L174 early_exit from a
 * callback that stores).  offsets[q+1]-offsets[q] = min(matches of q, limit); WHICH matches
 * are kept is unspecified (traversal order).  Same capacity protocol and errors.            */
ARBX_API arbx_status arbx_query_spatial_upto(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                                    int32_t limit, int32_t* offsets, int32_t* indices,
                                    int64_t indices_capacity, int64_t* total_host, arbx_stream stream);

/* Self-join / pair search over the index's own POINT primitives ("special
 * traversal algorithm when searching for pairs of objects"): every unordered
 * pair {i,j}, i != j, with ||x_i - x_j|| <= radius (closed) is reported EXACTLY ONCE, either as
 * j in row i or as i in row j (which of the two is unspecified).  offsets: DEVICE int32[n+1],
 * rows in the caller's primitive order; indices / capacity / total_host / errors as in
 * arbx_query_spatial.  Half traversal: a query only visits subtrees after its own leaf.
 * ARBX_ERR_UNSUPPORTED for BOX / SPHERE primitives.                                           */
ARBX_API arbx_status arbx_query_pairs(arbx_handle h, float radius, int32_t* offsets, int32_t* indices,
                             int64_t indices_capacity, int64_t* total_host, arbx_stream stream);

/* DBSCAN over the index's own POINT primitives (PAPER.md:L251-257 FDBSCAN: density clustering
 * on the search index; L274-277 dbscan(space, points, eps, minPts) -> labels, -1 = noise;
 * SURVEY.md NEXT-3).  A point is a CORE point iff at least min_pts primitives (itself included)
 * lie within eps (closed).  Core points within eps of each other share a cluster; a non-core
 * point within eps of a core point is a BORDER point of (any) one such cluster; all other
 * points are noise.  labels: DEVICE int32[n]; labels[i] = the smallest caller index of a core
 * point of i's cluster, or -1 for noise.  Asynchronous on `stream`.  POINT primitives only.   */
ARBX_API arbx_status arbx_dbscan(arbx_handle h, float eps, int32_t min_pts, int32_t* labels, arbx_stream stream);

/* k nearest primitives to each query point ("a pair of a query point and a
 * number of neighbors"; L79 distance to the stored geometry: point ||x-y||, box point-box
 * distance (0 inside), sphere max(0,||y-c||-R)).  qpoints: DEVICE nq*dim.  One k per call,
 * 1 <= k <= ARBX_K_MAX.  indices: DEVICE int32[nq*k]; distances: DEVICE fp32[nq*k] or NULL;
 * both need only their natural 4-byte alignment.
 * Row q holds min(k,n) neighbours by ascending Euclidean distance (not squared); ties in
 * unspecified order; when n < k the row is padded with index -1 / distance +inf.
 * Asynchronous on `stream`.                                                                 */
ARBX_API arbx_status arbx_query_knn(arbx_handle h, const float* qpoints, int64_t nq, int k,
                           int32_t* indices, float* distances, arbx_stream stream);

/* As arbx_query_knn with one k per query (a nearest query IS "a pair of a query
 * point and a number of neighbors").  k_per_query: DEVICE int32[nq], values clamped to
 * [0, kmax]; 1 <= kmax <= ARBX_K_MAX.  indices / distances: rows of kmax entries; row q holds
 * min(k_q, n) neighbours in ascending distance, then padding (index -1 / distance +inf).
 * Asynchronous on `stream`.                                                                  */
ARBX_API arbx_status arbx_query_knn_var(arbx_handle h, const float* qpoints, int64_t nq,
                               const int32_t* k_per_query, int kmax, int32_t* indices,
                               float* distances, arbx_stream stream);

/* fp64 coordinates (the library "supports different data dimensions (1-10) and
 * floating point precisions").  Same layouts and semantics as the fp32
 * calls with `double` rows; kNN distances are fp64.  The results are those of the fp64
 * predicates / distances evaluated on the caller's fp64 numbers: the index is a tree over the
 * primitives' bounding boxes rounded OUTWARD to fp32, which only prunes; every reported match or
 * neighbour is decided by the exact fp64 test at the leaves.  A handle from arbx_build_f64 is
 * queried with the _f64 calls only (and an fp32 handle with the fp32 calls only): the other
 * family returns ARBX_ERR_INVALID_ARG.  arbx_size / arbx_destroy / arbx_debug_validate work on
 * both; arbx_bounds of an fp64 handle gives the fp32 outward-rounded bounds; arbx_query_pairs,
 * arbx_dbscan, the capped calls and arbx_query_knn_var are fp32 only.  Errors, capacity protocol,
 * streams and padding as in the fp32 calls.                                                    */
ARBX_API arbx_status arbx_build_f64(const double* prims, int64_t n, int dim, arbx_kind kind,
                           arbx_stream stream, arbx_handle* out);
ARBX_API arbx_status arbx_query_count_f64(arbx_handle h, const double* queries, int64_t nq, arbx_kind qkind,
                                 int32_t* counts, arbx_stream stream);
ARBX_API arbx_status arbx_query_spatial_f64(arbx_handle h, const double* queries, int64_t nq, arbx_kind qkind,
                                   int32_t* offsets, int32_t* indices, int64_t indices_capacity,
                                   int64_t* total_host, arbx_stream stream);
ARBX_API arbx_status arbx_query_knn_f64(arbx_handle h, const double* qpoints, int64_t nq, int k,
                               int32_t* indices, double* distances, arbx_stream stream);

/* arbx_query_count for callers that must not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same count-only search, same arguments,
 * same results, but it calls no cudaMalloc / cudaFree / pool routine.  Its scratch (query codes,
 * the sorted order, the sort's bookkeeping: 17.8 MB) is ONE fixed array inside the library, held by
 * every GPU that loads the library until the process exits.  Limits and rules:
 *   - nq <= ARBX_NOALLOC_MAX_QUERIES, otherwise ARBX_ERR_UNSUPPORTED (split the batch or use
 *     arbx_query_count); fp32 handles only;
 *   - every call on a device shares that one array: calls that overlap on the GPU (different
 *     streams, or the same handle from two threads) RACE -- order them on one stream or with events;
 *   - the array keeps the last call's contents; the call clears what it needs on `stream`.
 * Asynchronous on `stream`.                                                                    */
#define ARBX_NOALLOC_MAX_QUERIES (1 << 20)
ARBX_API arbx_status arbx_query_count_noalloc(arbx_handle h, const float* queries, int64_t nq, arbx_kind qkind,
                                     int32_t* counts, arbx_stream stream);

/* Return the library's cached device memory on the current device to the driver, keeping at
 * most keep_bytes (0 = everything not in use).  Does not touch live handles.                 */
ARBX_API arbx_status arbx_trim(int64_t keep_bytes);

/* Test / experiment hook: sets one internal knob for the whole process (the library reads no
 * environment variable).  Keys: "leaf_max" (primitives per collapsed leaf range, 1..64,
 * default 16; applies to later builds), "code_bits" (space-filling-code bits per axis, 0 =
 * adapted to n), "brute_max" (n at or below which arbx_build makes a brute-force index, -1 =
 * default), "store_budget_mb" (scratch rows of the single-traversal storage query; 0 forces
 * count -> scan -> fill), "traversal" (0 = per-warp choice, 1 = one query per lane, 2 =
 * warp packets), "packet_alpha" (packet threshold, < 0 = default), "qbits" (query-code bits
 * per axis used by the query sort, 0 = all), "l2_persist" (1 = persisting-L2 window over the
 * node array during queries), "gather" (1 = arbx_query_count copies the queries into sorted order
 * first and un-permutes the counts), "pool_keep_mb" (release threshold of the memory pool),
 * "reset" (all knobs back to their defaults).  Results never depend on these knobs; they
 * choose between equivalent paths.  ARBX_ERR_INVALID_ARG for an unknown key.                 */
ARBX_API arbx_status arbx_debug_set(const char* key, double value);

/* Stable LSD radix sort of (key, value) pairs, exposed for tests of build step B3
 * ("Sorting in both construction and search").  keys: DEVICE, sorted in place
 * on bits [0, key_bits) -- bits at or above key_bits do not influence the order; values:
 * DEVICE uint32[n] or NULL (then only keys are sorted).  key_bytes is 4 or 8.  Asynchronous
 * on `stream`.                                                                              */
ARBX_API arbx_status arbx_sort_pairs(void* keys, uint32_t* values, int64_t n, int key_bytes, int key_bits,
                            arbx_stream stream);

/* Structural self-check of the tree (test hook for SURVEY.md §8(c-5) pin P9): verifies on
 * the device that the build raised no fault, the space-filling codes of the leaves
 * (recomputed from the leaf records) are non-decreasing, the leaf permutation is a permutation,
 * every node is reachable exactly once from the root, every stored child box equals the
 * union of that child's contents bit for bit.  *violations_host (HOST) = number of failed
 * checks (0 = valid).  Synchronises `stream`.                                               */
ARBX_API arbx_status arbx_debug_validate(arbx_handle h, int64_t* violations_host, arbx_stream stream);

/* Number of kernels this library has launched in the calling process (for bench.py's
 * gpu_launches claim).                                                                      */
ARBX_API int64_t arbx_launch_count(void);

/* Per-step device timing, for the roofline figures of bench.py.  While
 * enabled, every hot-path step (one entry of arbx_profile_kernel_name: "B3_sort_pass",
 * "T1_spatial_count", "K1K2_knn", ...) is bracketed by a pair of CUDA events recorded on the
 * stream it is launched on.  arbx_profile_read waits for the recorded events, adds up the
 * elapsed milliseconds and the number of bracketed steps per kernel id into the HOST arrays
 * ms_host / calls_host (capacity >= arbx_profile_num_kernels()) and clears the record.      */
ARBX_API arbx_status arbx_profile_enable(int on);
ARBX_API int arbx_profile_num_kernels(void);
ARBX_API const char* arbx_profile_kernel_name(int id);
ARBX_API arbx_status arbx_profile_read(double* ms_host, int64_t* calls_host, int capacity);

ARBX_API const char* arbx_status_string(arbx_status s);
ARBX_API const char* arbx_last_error(void);          /* thread-local detail of the last failure */

#ifdef __cplusplus
}
#endif
#endif /* ARBX_H_ */
