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
                                                   unsigned long long* __restrict__ codes, int drop) {
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
    codes[i] = interleave<D, B, unsigned long long>(q) >> drop;   // keep the top bits of every axis
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

// Brute-force index ("new brute-force search structure"): the primitives in the
// caller's order form ONE leaf range [0, n), root = ~0; the traversal kernels then scan every
// primitive for every query, and no codes, sort or hierarchy are needed.
template <int D, int PK>
__global__ void __launch_bounds__(BT) brute_leaves_kernel(const float* __restrict__ prims, int64_t n,
                                                          float* __restrict__ leaves, int32_t* __restrict__ root) {
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
  const int64_t j = (int64_t)blockIdx.x * BT + threadIdx.x;
  if (j == 0) root[0] = ~0;
  if (j >= n) return;
  float v[LW];
#pragma unroll
  for (int e = 0; e < W; ++e) v[e] = __ldg(prims + j * W + e);
  v[W] = __uint_as_float((uint32_t)j | (j == n - 1 ? LEAF_END : 0u));
#pragma unroll
  for (int e = W + 1; e < LW; ++e) v[e] = 0.f;
  float4* out = reinterpret_cast<float4*>(leaves + j * LW);
#pragma unroll
  for (int e = 0; e < LW / 4; ++e) out[e] = make_float4(v[4 * e], v[4 * e + 1], v[4 * e + 2], v[4 * e + 3]);
}

// ---- B5+B6: bottom-up hierarchy with fused refit ------------------------------------------------
// The tree is the binary radix tree of the sorted codes (Karras 2012): internal node p sits at
// the split between sorted leaves p and p+1, and a subtree covering [l,r] hangs under split r
// or split l-1, whichever separates codes that share the LONGER prefix.  Only the position of
// the highest differing bit matters for that comparison (two splits with the same highest bit
// always have a higher one between them, so they never bound the same range), so every split j
// is reduced to one byte:
//   level(j) = 32 + (1 + index of the top set bit of code[j]^code[j+1])      distinct codes
//            =      (1 + index of the top set bit of j^(j+1))                equal codes (A16:
//              duplicates are split by sorted position, which yields a balanced subtree)
//            = 255  for j = -1 and j = n-1 (the ends of the array).
// Emission is bottom-up (Apetrei 2014): every leaf climbs; at each node the first
// child to arrive leaves its box and stops, the second merges both boxes and carries on.
// B200 design: a block owns a chunk of HB consecutive leaves and does every merge whose node
// range lies inside the chunk through SHARED memory (flag + sibling box, __threadfence_block
// only).  A node is chunk-local iff its level is below the running maximum on both sides inside
// the chunk (prefix / suffix maxima of the level bytes), a property both children evaluate
// identically.  Only the O(log HB) subtrees per chunk that stick out continue through global
// atomics + __threadfence, so the long dependent chain of global round trips disappears.
template <int D> struct HierCfg { static constexpr int HB = D <= 5 ? 512 : 256; };

__device__ __forceinline__ int split_level(const unsigned long long* __restrict__ codes, int j, int n) {
  if (j < 0 || j >= n - 1) return 255;
  const unsigned long long x = __ldg(codes + j) ^ __ldg(codes + j + 1);
  return x ? 32 + 64 - __clzll((long long)x) : 32 - __clz(j ^ (j + 1));
}

// inclusive running maximum over the block, thread order
template <int HB>
__device__ __forceinline__ int block_running_max(int v, int* s_w) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(~0u, v, o);
    if (lane >= o) v = max(v, y);
  }
  if (lane == 31) s_w[w] = v;
  __syncthreads();
  int base = 0;
  for (int i = 0; i < w; ++i) base = max(base, s_w[i]);
  __syncthreads();
  return max(v, base);
}

template <int D, int PK>
__global__ void __launch_bounds__(HierCfg<D>::HB)
hierarchy_kernel(const unsigned long long* __restrict__ codes, float* __restrict__ leaves,
                 float* __restrict__ nodes, int n, int leaf_max, int32_t* __restrict__ root,
                 int* __restrict__ open_count, int* __restrict__ open_lrf, float* __restrict__ open_box,
                 int open_cap) {
  constexpr int HB = HierCfg<D>::HB;
  constexpr int W = prim_width(PK, D);
  constexpr int LW = leaf_width(PK, D);
  constexpr int NW = node_width(D);
  // s_lvl[t] = level of split c0-1+t, t = 0..HB;  s_pre[t] = max s_lvl[0..t];  s_suf[t] = max s_lvl[t..HB]
  constexpr int HALO = 64;   // >= the largest leaf_max
  __shared__ uint8_t s_lx[HALO + HB + 1 + HALO], s_pre[HB + 1], s_suf[HB + 1];
  uint8_t* const s_lvl = s_lx + HALO;   // s_lvl[t], -HALO <= t <= HB + HALO
  __shared__ int s_w[HB / 32];
  __shared__ int s_flag[HB];
  __shared__ float s_box[2][HB][2 * D];
  const int tid = threadIdx.x;
  const int c0 = blockIdx.x * HB;
  const int i = c0 + tid;
  {
    const int lv = split_level(codes, c0 - 1 + tid, n);
    s_lvl[tid] = (uint8_t)lv;
    s_flag[tid] = -1;
    const int pm = block_running_max<HB>(lv, s_w);
    s_pre[tid] = (uint8_t)pm;
    if (tid == 0) s_lvl[HB] = (uint8_t)split_level(codes, c0 - 1 + HB, n);
    __syncthreads();
    // suffix maxima: thread t handles element HB - t (elements HB..1)
    const int lr = s_lvl[HB - tid];
    const int sm = block_running_max<HB>(lr, s_w);
    s_suf[HB - tid] = (uint8_t)sm;
    // levels of the leaf_max splits on either side of the chunk, for the range classification
    if (tid < HALO) { if (tid < leaf_max) s_lvl[-1 - tid] = (uint8_t)split_level(codes, c0 - 2 - tid, n); }
    else if (tid < 2 * HALO) { const int d = tid - HALO; if (d < leaf_max) s_lvl[HB + 1 + d] = (uint8_t)split_level(codes, c0 + HB + d, n); }
  }
  __syncthreads();

  // Leaf ranges first, from the level bytes alone (no atomics, no boxes).  Split j is the top
  // of a subtree [l_j, r_j] bounded by the nearest higher level on each side; it is a leaf-
  // range BOUNDARY iff that subtree holds more than leaf_max primitives.  Every thread
  // classifies one split with two short scans; then the thread of each range's first leaf
  // scans the range for its box and starts the climb there.  The merges below leaf-range
  // level (the bulk of all merges) never happen.
  auto lvl = [&](int j) -> int {   // level of split j, -1 <= j <= n-1
    const int t = j - (c0 - 1);
    return (t >= 0 && t <= HB) ? (int)s_lvl[t] : split_level(codes, j, n);
  };
  auto is_boundary = [&](int j) -> bool {
    const int L = lvl(j);
    if (L == 255) return true;
    int da = 1, db = 1;          // steps to the nearest higher level on the left / right
    while (da <= leaf_max && lvl(j - da) < L) ++da;
    while (da + db <= leaf_max && lvl(j + db) < L) ++db;
    return da + db > leaf_max;   // subtree size = da + db
  };
  // the same test for a split of this chunk (0 <= t <= HB), from shared memory only and with a
  // warp-uniform trip count: nearest level >= L within leaf_max steps on each side
  auto is_boundary_local = [&](int t) -> bool {
    const int L = s_lvl[t];
    if (L == 255) return true;
    int da = leaf_max + 1, db = leaf_max + 1;
    for (int d = leaf_max; d >= 1; --d) {
      if (s_lvl[t - d] >= L) da = d;
      if (s_lvl[t + d] >= L) db = d;
    }
    return da + db > leaf_max;
  };
  __shared__ uint8_t s_bnd[HB + 1];
  s_bnd[tid] = is_boundary_local(tid) ? 1 : 0;
  if (tid == 0) s_bnd[HB] = is_boundary_local(HB) ? 1 : 0;
  __syncthreads();
  // Every thread loads the box of its own leaf (one coalesced load per thread, all in flight at
  // once) so that the few range leaders below read shared memory instead of walking global
  // memory one leaf at a time.
  constexpr bool STAGE_LEAF = sizeof(float) * 2 * D * HB <= 12288;
  __shared__ float s_leaf[STAGE_LEAF ? HB : 1][2 * D];
  if constexpr (STAGE_LEAF) {
    if (i < n) {
      float v[W], bl[D], bh[D];
      const float* lf = leaves + (int64_t)i * LW;
#pragma unroll
      for (int e = 0; e < W; ++e) v[e] = lf[e];
      box_of<D, PK>(v, bl, bh);
#pragma unroll
      for (int a = 0; a < D; ++a) { s_leaf[tid][a] = bl[a]; s_leaf[tid][D + a] = bh[a]; }
    }
  }
  // The first leaves of the ranges (about one thread in twelve) are packed into the block's
  // first warps: the box scans and the climb below then run on full warps instead of on ~3
  // lanes of every warp.
  __shared__ uint16_t s_lead[HB];
  {
    const bool lead = i < n && s_bnd[tid];
    const uint32_t bal = __ballot_sync(~0u, lead);
    const int lane = tid & 31, w = tid >> 5;
    if (lane == 0) s_w[w] = __popc(bal);
    __syncthreads();
    int base = 0, total = 0;
    for (int k = 0; k < HB / 32; ++k) { const int c = s_w[k]; base += k < w ? c : 0; total += c; }
    if (lead) s_lead[base + __popc(bal & ((1u << lane) - 1u))] = (uint16_t)tid;
    __syncthreads();
    if (tid >= total) return;
  }
  const int i0 = c0 + s_lead[tid];
  int l = i0, r = i0;
  for (;; ++r) {                         // the range ends at the next boundary split
    const int t = r - c0 + 1;
    if (t <= HB ? s_bnd[t] != 0 : is_boundary(r)) break;
  }
  int32_t ref = ~l;
  float lo[D], hi[D];
#pragma unroll
  for (int a = 0; a < D; ++a) { lo[a] = INFINITY; hi[a] = -INFINITY; }
  for (int j = l; j <= r; ++j) {
    float bl[D], bh[D];
    if (STAGE_LEAF && j < c0 + HB) {
#pragma unroll
      for (int a = 0; a < D; ++a) { bl[a] = s_leaf[j - c0][a]; bh[a] = s_leaf[j - c0][D + a]; }
    } else {
      float v[W];
      const float* lf = leaves + (int64_t)j * LW;
#pragma unroll
      for (int e = 0; e < W; ++e) v[e] = lf[e];
      box_of<D, PK>(v, bl, bh);
    }
#pragma unroll
    for (int a = 0; a < D; ++a) { lo[a] = fminf(lo[a], bl[a]); hi[a] = fmaxf(hi[a], bh[a]); }
  }
  reinterpret_cast<uint32_t*>(leaves)[(int64_t)r * LW + W] |= LEAF_END;   // last record of the range
  for (;;) {
    if (l == 0 && r == n - 1) {   // root
      *root = ref;
      return;
    }
    // the parent splits either right after r (we are its left child) or right before l
    const bool inside = l >= c0 && r < c0 + HB;     // still chunk-local: levels come from shared memory
    const int lvl_l = inside ? s_lvl[l - c0] : split_level(codes, l - 1, n);
    const int lvl_r = inside ? s_lvl[r - c0 + 1] : split_level(codes, r, n);
    const bool left_child = lvl_r < lvl_l;
    const int p = left_child ? r : l - 1;
    const int t = p - c0 + 1;                        // index of split p in s_lvl
    const bool local = inside && t >= 1 && t <= HB - 1 &&
                       (left_child ? s_lvl[t] < s_suf[t + 1] : s_lvl[t] < s_pre[t - 1]);
    float* node = nodes + (int64_t)p * NW;
    const int slot = left_child ? 0 : 1;
    const int sib = 1 - slot;
    auto store_half = [&]() {   // this child's box and reference, for the traversal kernels
#pragma unroll
      for (int a = 0; a < D; ++a) {
        __stcg(node + slot * 2 * D + a, lo[a]);
        __stcg(node + slot * 2 * D + D + a, hi[a]);
      }
      __stcg(reinterpret_cast<int*>(node) + 4 * D + slot, ref);
    };
    if (!local) {
      // The parent reaches outside this chunk: park the subtree for hierarchy_top_kernel, so
      // that this block is not kept alive by a chain of global round trips.
      const int e = atomicAdd(open_count, 1);
      if (e < open_cap) {
        open_lrf[3 * e] = l; open_lrf[3 * e + 1] = r; open_lrf[3 * e + 2] = ref;
#pragma unroll
        for (int a = 0; a < D; ++a) { open_box[(int64_t)e * 2 * D + a] = lo[a]; open_box[(int64_t)e * 2 * D + D + a] = hi[a]; }
      } else {
        atomicOr(root + 1, BUILD_FAULT_OPEN_OVERFLOW);   // never silent: every query on this handle fails
      }
      return;
    }
    // the sibling reads our box from shared memory, so the global stores stay outside the
    // fence -> atomic window (a fence would otherwise wait for them)
    float* mine = s_box[slot][p - c0];
#pragma unroll
    for (int a = 0; a < D; ++a) { mine[a] = lo[a]; mine[D + a] = hi[a]; }
    __threadfence_block();
    const int other = atomicExch(&s_flag[p - c0], left_child ? l : r);
    store_half();
    if (other == -1) return;   // first to arrive: the sibling's thread carries on
    __threadfence_block();
    const volatile float* theirs = s_box[sib][p - c0];
#pragma unroll
    for (int a = 0; a < D; ++a) { lo[a] = fminf(lo[a], theirs[a]); hi[a] = fmaxf(hi[a], theirs[D + a]); }
    // second to arrive: `other` is the far end of the sibling's range
    if (left_child) r = other; else l = other;
    __stcg(reinterpret_cast<int*>(node) + 4 * D + 2, l);
    __stcg(reinterpret_cast<int*>(node) + 4 * D + 3, r);
    ref = p;   // leaf ranges are maximal, so every merge makes a real node
  }
}

// Top of the tree: one thread per parked subtree, every merge through global memory (node
// record + atomicExch flag + __threadfence), the classic bottom-up scheme.  Only O(log chunk)
// subtrees per chunk get here.
template <int D>
__global__ void __launch_bounds__(256)
hierarchy_top_kernel(const unsigned long long* __restrict__ codes, float* __restrict__ nodes,
                     int* __restrict__ flags, int n, int32_t* __restrict__ root,
                     const int* __restrict__ open_count, const int* __restrict__ open_lrf,
                     const float* __restrict__ open_box, int open_cap) {
  constexpr int NW = node_width(D);
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= min(*open_count, open_cap)) return;
  int l = open_lrf[3 * e], r = open_lrf[3 * e + 1];
  int32_t ref = open_lrf[3 * e + 2];
  float lo[D], hi[D];
#pragma unroll
  for (int a = 0; a < D; ++a) { lo[a] = open_box[(int64_t)e * 2 * D + a]; hi[a] = open_box[(int64_t)e * 2 * D + D + a]; }
  for (;;) {
    if (l == 0 && r == n - 1) { *root = ref; return; }
    const bool left_child = split_level(codes, r, n) < split_level(codes, l - 1, n);
    const int p = left_child ? r : l - 1;
    float* node = nodes + (int64_t)p * NW;
    const int slot = left_child ? 0 : 1, sib = 1 - slot;
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
#pragma unroll
    for (int a = 0; a < D; ++a) {
      lo[a] = fminf(lo[a], __ldcg(node + sib * 2 * D + a));
      hi[a] = fmaxf(hi[a], __ldcg(node + sib * 2 * D + D + a));
    }
    if (left_child) r = other; else l = other;
    __stcg(reinterpret_cast<int*>(node) + 4 * D + 2, l);
    __stcg(reinterpret_cast<int*>(node) + 4 * D + 3, r);
    ref = p;
  }
}

template <int D, int PK>
arbx_status build_typed(const float* prims, int64_t n, cudaStream_t s, Index* ix, int sms) {
  constexpr int LW = leaf_width(PK, D);
  constexpr int NW = node_width(D);
  Scratch<uint32_t> enc, perm, perm_alt;
  Scratch<unsigned long long> codes, codes_alt;
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

  // Tiny inputs: a tree costs ~25 dependent launches to build and saves nothing at query time
  int brute_max = g_cfg.brute_max.load(std::memory_order_relaxed);
  if (brute_max < 0) brute_max = 512;
  if (n <= brute_max) {
    ix->brute = true;
    ix->leaf_max = (int)std::max<int64_t>(n, 1);
    ARBX_TRY(scratch_alloc((void**)&ix->leaves, (size_t)n * LW * sizeof(float), s));
    ProfScope ps(K_LEAVES, s);
    brute_leaves_kernel<D, PK><<<(unsigned)((n + BT - 1) / BT), BT, 0, s>>>(prims, n, ix->leaves, ix->root);
    ARBX_LAUNCH_CHECK();
    return ARBX_OK;
  }

  // Code width (reading A15): b bits per axis, b <= floor(64/D).  The tree shape is not
  // observable in results and duplicate codes are split by sorted position (A16), so the codes
  // only need to resolve the primitives: b = ceil(log2(n)/D) + 4 bits per axis (16^D cells per
  // primitive on average), rounded up to fill whole 8-bit sort passes.
  constexpr int BMAX = code_bits_per_axis(D);
  int b = g_cfg.code_bits.load(std::memory_order_relaxed);
  if (b <= 0) {
    int lg = 0;
    while ((int64_t(1) << lg) < n) ++lg;
    b = std::min(BMAX, (lg + D - 1) / D + 4);
    b = std::max(b, 8 * ((D * b + 7) / 8) / D);
  }
  b = std::max(1, std::min(BMAX, b));
  ix->code_bits = b;
  ARBX_TRY(codes.alloc((size_t)n, s));
  ARBX_TRY(codes_alt.alloc((size_t)n, s));
  {
    ProfScope ps(K_CODES, s);
    codes_kernel<D, PK><<<sgrid, BT, 0, s>>>(prims, n, ix->bounds, codes.p, D * (BMAX - b));
    ARBX_LAUNCH_CHECK();
  }
  ARBX_TRY(perm.alloc((size_t)n, s));
  ARBX_TRY(perm_alt.alloc((size_t)n, s));
  unsigned long long* scodes = nullptr;   // sorted codes / permutation: whichever ping-pong buffer holds them
  uint32_t* sperm = nullptr;
  ARBX_TRY(radix_sort_u64(codes.p, codes_alt.p, perm.p, perm_alt.p, true, n, D * b, s, &scodes, &sperm));

  ARBX_TRY(scratch_alloc((void**)&ix->leaves, (size_t)n * LW * sizeof(float), s));
  const int fgrid = (int)((n + BT - 1) / BT);
  {
    ProfScope ps(K_LEAVES, s);
    leaves_kernel<D, PK><<<fgrid, BT, 0, s>>>(prims, sperm, n, ix->leaves);
    ARBX_LAUNCH_CHECK();
  }

  const size_t nn = n > 1 ? (size_t)(n - 1) : 1;
  ARBX_TRY(scratch_alloc((void**)&ix->nodes, nn * NW * sizeof(float), s));
  ARBX_TRY(flags.alloc(nn, s));
  ProfScope ps(K_HIERARCHY, s);
  constexpr int HB = HierCfg<D>::HB;
  const unsigned nchunks = (unsigned)((n + HB - 1) / HB);
  // A chunk parks at most one subtree per distinct prefix maximum and one per distinct suffix
  // maximum of its level bytes.  Levels take the values 1..31 (equal codes), 33..96 (distinct
  // codes) and 255 (array ends): at most 96 distinct values per side, 2*96 + 2 < 200.  An
  // overflow would still not be silent: it raises BUILD_FAULT_OPEN_OVERFLOW in root[1].
  static_assert(2 * (31 + 64 + 1) + 2 <= 200, "open_cap per chunk must cover every distinct level twice");
  const int64_t open_cap = std::min<int64_t>(n, (int64_t)nchunks * 200);
  Scratch<int> open_lrf, open_count;
  Scratch<float> open_box;
  ARBX_TRY(open_count.alloc(1, s));
  ARBX_TRY(open_lrf.alloc((size_t)open_cap * 3, s));
  ARBX_TRY(open_box.alloc((size_t)open_cap * 2 * D, s));
  ARBX_CUDA(cudaMemsetAsync(open_count.p, 0, sizeof(int), s));
  ARBX_CUDA(cudaMemsetAsync(flags.p, 0xff, nn * sizeof(int), s));
  hierarchy_kernel<D, PK><<<nchunks, HB, 0, s>>>(scodes, ix->leaves, ix->nodes, (int)n, ix->leaf_max, ix->root,
                                                 open_count.p, open_lrf.p, open_box.p, (int)open_cap);
  ARBX_LAUNCH_CHECK();
  hierarchy_top_kernel<D><<<(unsigned)((open_cap + 255) / 256), 256, 0, s>>>(scodes, ix->nodes, flags.p, (int)n, ix->root,
                                                                           open_count.p, open_lrf.p, open_box.p, (int)open_cap);
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
  ARBX_TRY(scratch_alloc((void**)&ix->root, 2 * sizeof(int32_t), s));
  ARBX_CUDA(cudaMemsetAsync(ix->root, 0, 2 * sizeof(int32_t), s));
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
