// sort.cu -- build step B3 / query step Q2: stable LSD radix sort of (code, index) pairs.
// PAPER.md:L307 (§3 "Sorting in both construction and search"), L309 (sort is "critical").
//
// Hand-written single-sweep radix sort (8-bit digits): ONE histogram kernel over all digits,
// then one kernel per digit that ranks a tile, publishes the tile's digit counts, resolves
// its global offsets by decoupled look-back over the predecessor tiles and scatters through
// shared memory so that global stores are coalesced runs.  No CUB/Thrust.
//
// Algorithmic HBM bytes per element: histogram K; per pass 2*(K+4)
// (K = key bytes; the first pass of an iota sort reads no values).
#include <algorithm>
#include <atomic>

#include "common.cuh"

namespace arbx {
namespace {

constexpr int SORT_THREADS = 512;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_IPT = 8;                          // items per thread
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;   // 4096 elements per tile
constexpr uint32_t FLAG_AGG = 1u << 30, FLAG_INCL = 2u << 30, VAL_MASK = (1u << 30) - 1;
constexpr int MAX_PASSES = 8;
constexpr int SORT_LB = 4;                           // predecessor tiles per look-back round trip
#ifndef SORT_BLOCKS_PER_SM
#define SORT_BLOCKS_PER_SM 3
#endif

__device__ __forceinline__ uint2 ld_volatile_u32x2(const uint2* p) {
  uint2 v;
  asm volatile("ld.volatile.global.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_volatile_u32x2(uint2* p, uint2 v) {
  asm volatile("st.volatile.global.v2.u32 [%0], {%1, %2};" ::"l"(p), "r"(v.x), "r"(v.y) : "memory");
}

// lanes of the warp holding the same digit: one ballot per digit bit (plain ALU/vote work; the
// match.any instruction measured 1.3x slower than this on sm_100)
template <int BITS>
__device__ __forceinline__ uint32_t match_digit(uint32_t d) {
  uint32_t peers = ~0u;
#pragma unroll
  for (int b = 0; b < BITS; ++b) {
    const bool bit = (d >> b) & 1u;
    const uint32_t bal = __ballot_sync(~0u, bit);
    peers &= bit ? bal : ~bal;
  }
  return peers;
}

// ---- histogram of every digit in one read of the keys ---------------------------------------
template <typename K, int BITS>
__global__ void __launch_bounds__(512) hist_kernel(const K* __restrict__ keys, uint32_t n, int npass,
                                                   uint32_t top_mask, uint32_t* __restrict__ ghist) {
  constexpr int RADIX = 1 << BITS;
  // top_mask: bits of the last digit that belong to the key (bits at or above key_bits are ignored)
  auto digit = [&](K k, int p) -> uint32_t { return (uint32_t)(k >> (BITS * p)) & (p == npass - 1 ? top_mask : (uint32_t)(RADIX - 1)); };
  __shared__ uint32_t sh[(BITS == 8 ? MAX_PASSES : 7) * RADIX];
  for (int i = threadIdx.x; i < npass * RADIX; i += blockDim.x) sh[i] = 0;
  __syncthreads();
  constexpr int VEC = 16 / sizeof(K);
  const uint32_t nvec = (reinterpret_cast<uintptr_t>(keys) & 15) == 0 ? n / VEC : 0u;
  const uint4* kv = reinterpret_cast<const uint4*>(keys);
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += gridDim.x * blockDim.x) {
    uint4 v = __ldg(kv + i);
    K k[VEC];
    if constexpr (sizeof(K) == 8) {
      k[0] = ((K)v.y << 32) | v.x;
      k[1] = ((K)v.w << 32) | v.z;
    } else {
      k[0] = v.x; k[1] = v.y; k[2] = v.z; k[3] = v.w;
    }
#pragma unroll
    for (int e = 0; e < VEC; ++e)
      for (int p = 0; p < npass; ++p) atomicAdd(&sh[p * RADIX + digit(k[e], p)], 1u);
  }
  if (blockIdx.x == 0) {
    for (uint32_t i = nvec * VEC + threadIdx.x; i < n; i += blockDim.x) {
      K k = keys[i];
      for (int p = 0; p < npass; ++p) atomicAdd(&sh[p * RADIX + digit(k, p)], 1u);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < npass * RADIX; i += blockDim.x)
    if (sh[i]) atomicAdd(&ghist[i], sh[i]);
}

// exclusive scan of each digit histogram, one block per pass
template <int BITS>
__global__ void __launch_bounds__(256) hist_scan_kernel(uint32_t* ghist) {
  constexpr int RADIX = 1 << BITS;
  constexpr int PER = RADIX / 256;
  __shared__ uint32_t wsum[8];
  uint32_t* h = ghist + blockIdx.x * RADIX;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t v[PER], tot = 0;
#pragma unroll
  for (int e = 0; e < PER; ++e) { v[e] = h[threadIdx.x * PER + e]; tot += v[e]; }
  uint32_t x = tot;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t y = __shfl_up_sync(~0u, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  uint32_t base = 0;
  for (int i = 0; i < w; ++i) base += wsum[i];
  uint32_t run = base + x - tot;
#pragma unroll
  for (int e = 0; e < PER; ++e) { h[threadIdx.x * PER + e] = run; run += v[e]; }
}

// ---- one digit pass ------------------------------------------------------------------------
// Per tile of 4096 pairs: rank every key among the keys of its warp with the same digit (ballot
// matching + one shared-memory atomic per digit group on PACKED 16-bit per-warp counters), scan
// the per-warp counts, publish the tile's digit counts, resolve the tile's global offsets by
// decoupled look-back (two digits per 64-bit status word pair, SORT_LB predecessors per round
// trip), scatter keys AND values through shared memory in one step, and store them as runs.
template <typename K, int BITS, bool IOTA, bool VALS>
__global__ void __launch_bounds__(SORT_THREADS, SORT_BLOCKS_PER_SM)
onesweep_pass(const K* __restrict__ kin, K* __restrict__ kout, const uint32_t* __restrict__ vin,
              uint32_t* __restrict__ vout, uint32_t n, int shift, uint32_t dmask,
              const uint32_t* __restrict__ digit_base, uint32_t* __restrict__ counter,
              uint32_t* __restrict__ status) {
  constexpr int RADIX = 1 << BITS;
  constexpr int HW = RADIX / 2;          // packed words per warp: digit d lives in half (d & 1) of word d >> 1
  extern __shared__ __align__(16) unsigned char sort_smem[];
  K* skeys = reinterpret_cast<K*>(sort_smem);
  uint32_t* svals = reinterpret_cast<uint32_t*>(sort_smem + sizeof(K) * SORT_TILE);
  uint32_t (*whist)[HW] = reinterpret_cast<uint32_t (*)[HW]>(sort_smem + (sizeof(K) + (VALS ? 4 : 0)) * SORT_TILE);
  __shared__ uint32_t s_toff[RADIX];    // first position of digit d inside the sorted tile
  __shared__ uint32_t s_goff[RADIX];    // global position of tile position p with digit d = s_goff[d] + p
  __shared__ uint32_t s_wsum[SORT_WARPS];
  __shared__ uint32_t s_tile;

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_tile = atomicAdd(counter, 1u);   // ticket: tile t starts only after tiles < t did
  for (int i = tid; i < SORT_WARPS * HW; i += SORT_THREADS) (&whist[0][0])[i] = 0;
  static_assert(sizeof(K) * SORT_TILE >= sizeof(uint32_t) * SORT_WARPS * RADIX, "the lane-mask tables borrow the tile");
  for (int i = tid; i < SORT_WARPS * RADIX; i += SORT_THREADS) reinterpret_cast<uint32_t*>(sort_smem)[i] = 0;
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t tile_base = tile * (uint32_t)SORT_TILE;
  const uint32_t nvalid = min((uint32_t)SORT_TILE, n - tile_base);

  // warp-striped load: warp w owns SORT_IPT*32 consecutive elements.  Padding keys of a partial
  // last tile carry the largest digit of this pass, so they sort behind every real key.  Only
  // the DIGITS stay in registers (one byte each): the keys and values are read again for the
  // scatter, from L2, which keeps the kernel at 40 registers and three resident blocks per SM.
  const uint32_t wbase = tile_base + w * (32 * SORT_IPT) + lane;
  const K pad_key = (K)dmask << shift;
  uint32_t dig[SORT_IPT];
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    const uint32_t idx = wbase + j * 32;
    const K k = idx < n ? kin[idx] : pad_key;
    dig[j] = (uint32_t)(k >> shift) & dmask;
  }

  // stable rank of every key among the keys of its warp with the same digit.  The match
  // instructions of a batch are independent (their latency overlaps); program order inside the
  // warp keeps item j ahead of item j+1.
  uint16_t rank[SORT_IPT];
  const uint32_t lt_mask = (1u << lane) - 1u;
  // Lanes with the same digit find each other through a per-warp table of lane masks in shared
  // memory (it borrows the tile's space, which is idle until the scatter): atomicOr of the own
  // lane bit, read back, the group's first lane clears the entry and bumps the packed counter.
  // Three shared-memory operations per key where eight ballots + sixteen logic operations were.
  uint32_t* const wmask = reinterpret_cast<uint32_t*>(sort_smem) + w * RADIX;
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    const uint32_t d = dig[j];
    atomicOr(&wmask[d], 1u << lane);
    __syncwarp();
    const uint32_t peers = wmask[d];
    __syncwarp();
    const int leader = __ffs(peers) - 1;
    const int sh16 = (d & 1u) * 16;
    uint32_t old = 0;
    if (lane == leader) {
      wmask[d] = 0;
      old = atomicAdd(&whist[w][d >> 1], (uint32_t)__popc(peers) << sh16);
    }
    old = (__shfl_sync(~0u, old, leader) >> sh16) & 0xffffu;
    rank[j] = (uint16_t)(old + __popc(peers & lt_mask));
  }
  __syncthreads();

  // thread t < HW owns digits 2t and 2t+1: exclusive scan over warps, tile counts, publish, look back
  uint32_t run0 = 0, run1 = 0, pub0 = 0, pub1 = 0, x = 0;
  uint2* status2 = reinterpret_cast<uint2*>(status);
  if (tid < HW) {
#pragma unroll
    for (int i = 0; i < SORT_WARPS; ++i) {
      const uint32_t t = whist[i][tid];
      whist[i][tid] = run0 | (run1 << 16);
      run0 += t & 0xffffu;
      run1 += t >> 16;
    }
    // padding keys of a partial last tile sit in digit dmask; nobody reads their count
    pub0 = run0; pub1 = run1;
    if ((uint32_t)(2 * tid) == dmask) pub0 -= (uint32_t)SORT_TILE - nvalid;
    if ((uint32_t)(2 * tid + 1) == dmask) pub1 -= (uint32_t)SORT_TILE - nvalid;
    const uint32_t fl = tile == 0 ? FLAG_INCL : FLAG_AGG;
    st_volatile_u32x2(&status2[(size_t)tile * HW + tid], make_uint2(fl | pub0, fl | pub1));
    x = run0 + run1;
  }
  // exclusive scan of the tile counts over digits (threads >= HW contribute nothing)
  {
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(~0u, incl, o);
      if (lane >= o) incl += y;
    }
    if (lane == 31) s_wsum[w] = incl;
    __syncthreads();
    uint32_t wb = 0;
#pragma unroll
    for (int i = 0; i < SORT_WARPS; ++i) wb += i < w ? s_wsum[i] : 0u;
    x = wb + incl - x;     // first tile position of digit 2*tid
  }
  const uint32_t toff0 = x, toff1 = x + run0;
  if (tid < HW) {
    s_toff[2 * tid] = toff0;
    s_toff[2 * tid + 1] = toff1;
  }
  __syncthreads();
  // The look-back (a few global round trips) is walked by the first HW threads only; the other
  // warps go straight on to the scatter, which needs s_toff but not the global offsets.
  if (tid < HW) {
    uint32_t ex0 = 0, ex1 = 0;
    if (tile > 0) {
      // decoupled look-back: SORT_LB predecessors per round trip (independent loads), both digits
      // of this thread ride on the same 8-byte loads; a predecessor is consumed once the digits
      // still walking have both been published by it, an inclusive prefix ends a digit's walk
      int t = (int)tile - 1;
      bool dn0 = false, dn1 = false;
      while (!(dn0 && dn1)) {
        uint2 v[SORT_LB];
#pragma unroll
        for (int i = 0; i < SORT_LB; ++i)
          v[i] = t - i >= 0 ? ld_volatile_u32x2(&status2[(size_t)(t - i) * HW + tid]) : make_uint2(FLAG_INCL, FLAG_INCL);
        int used = 0;
#pragma unroll
        for (int i = 0; i < SORT_LB; ++i) {
          if (used == i && !(dn0 && dn1)) {
            const uint32_t f0 = v[i].x >> 30, f1 = v[i].y >> 30;
            if ((dn0 || f0 != 0u) && (dn1 || f1 != 0u)) {
              if (!dn0) { ex0 += v[i].x & VAL_MASK; dn0 = f0 == 2u; }
              if (!dn1) { ex1 += v[i].y & VAL_MASK; dn1 = f1 == 2u; }
              used = i + 1;
            }
          }
        }
        t -= used;                    // resume at the first predecessor that was not ready
      }
      st_volatile_u32x2(&status2[(size_t)tile * HW + tid], make_uint2(FLAG_INCL | (ex0 + pub0), FLAG_INCL | (ex1 + pub1)));
    }
    s_goff[2 * tid] = digit_base[2 * tid] + ex0 - toff0;
    s_goff[2 * tid + 1] = digit_base[2 * tid + 1] + ex1 - toff1;
  }

  // scatter keys and values to their position inside the sorted tile, then store runs
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    const uint32_t idx = wbase + j * 32;
    const uint32_t d = dig[j];
    const uint32_t wpre = (whist[w][d >> 1] >> ((d & 1u) * 16)) & 0xffffu;
    const uint32_t pos = s_toff[d] + wpre + rank[j];
    skeys[pos] = idx < n ? __ldcg(kin + idx) : pad_key;
    if constexpr (VALS) svals[pos] = IOTA ? idx : (idx < n ? __ldcg(vin + idx) : 0u);
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    const uint32_t p = j * SORT_THREADS + tid;
    const K k = skeys[p];
    const uint32_t d = (uint32_t)(k >> shift) & dmask;
    const uint32_t g = s_goff[d] + p;
    if (p < nvalid) {
      kout[g] = k;
      if constexpr (VALS) vout[g] = svals[p];
    }
  }
}

template <typename K, int BITS>
arbx_status radix_sort_bits(K* keys, K* kalt, uint32_t* vals, uint32_t* valt, bool iota, int64_t n, int key_bits,
                            cudaStream_t s, K** keys_out, uint32_t** vals_out) {
  constexpr int RADIX = 1 << BITS;
  const bool has_vals = vals != nullptr;
  const int npass = (key_bits + BITS - 1) / BITS;
  const uint32_t top_mask = key_bits % BITS ? (1u << (key_bits % BITS)) - 1u : (uint32_t)(RADIX - 1);
  const uint32_t ntiles = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);

  Scratch<uint32_t> meta;
  // meta: [npass*RADIX] digit histograms | [MAX_PASSES] tile counters | [npass*ntiles*RADIX] look-back status
  const size_t meta_words = (size_t)npass * RADIX + MAX_PASSES + (size_t)npass * ntiles * RADIX;
  ARBX_TRY(meta.alloc(meta_words, s));
  ARBX_CUDA(cudaMemsetAsync(meta.p, 0, meta_words * sizeof(uint32_t), s));
  uint32_t* ghist = meta.p;
  uint32_t* counters = meta.p + (size_t)npass * RADIX;
  uint32_t* status = counters + MAX_PASSES;

  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  constexpr int kHistId = sizeof(K) == 8 ? K_SORT_HIST : K_QSORT_HIST;
  constexpr int kPassId = sizeof(K) == 8 ? K_SORT_PASS : K_QSORT_PASS;
  {
    ProfScope ps(kHistId, s);
    int64_t want = (n / (16 / (int)sizeof(K)) + 511) / 512;
    int grid = (int)std::min<int64_t>(std::max<int64_t>(want, 1), (int64_t)sms * 4);
    hist_kernel<K, BITS><<<grid, 512, 0, s>>>(keys, (uint32_t)n, npass, top_mask, ghist);
    ARBX_LAUNCH_CHECK();
    hist_scan_kernel<BITS><<<npass, 256, 0, s>>>(ghist);
    ARBX_LAUNCH_CHECK();
  }
  const size_t smem_k = sizeof(K) * SORT_TILE + sizeof(uint32_t) * SORT_WARPS * (RADIX / 2);
  const size_t smem_kv = smem_k + sizeof(uint32_t) * SORT_TILE;
  static std::atomic<bool> attr_set{false};   // one instance per (K, BITS)
  if (!attr_set.load(std::memory_order_acquire)) {
    ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, BITS, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_k));
    ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, BITS, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_kv));
    ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, BITS, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_kv));
    attr_set.store(true, std::memory_order_release);
  }
  K* kin = keys; K* kout = kalt;
  uint32_t* vin = vals; uint32_t* vout = valt;
  for (int p = 0; p < npass; ++p) {
    const uint32_t* base = ghist + (size_t)p * RADIX;
    uint32_t* st = status + (size_t)p * ntiles * RADIX;
    const uint32_t dmask = p == npass - 1 ? top_mask : (uint32_t)(RADIX - 1);
    ProfScope ps(kPassId, s);
    if (!has_vals)
      onesweep_pass<K, BITS, false, false><<<ntiles, SORT_THREADS, smem_k, s>>>(kin, kout, nullptr, nullptr, (uint32_t)n, BITS * p, dmask, base, counters + p, st);
    else if (p == 0 && iota)
      onesweep_pass<K, BITS, true, true><<<ntiles, SORT_THREADS, smem_kv, s>>>(kin, kout, nullptr, vout, (uint32_t)n, BITS * p, dmask, base, counters + p, st);
    else
      onesweep_pass<K, BITS, false, true><<<ntiles, SORT_THREADS, smem_kv, s>>>(kin, kout, vin, vout, (uint32_t)n, BITS * p, dmask, base, counters + p, st);
    ARBX_LAUNCH_CHECK();
    std::swap(kin, kout);
    std::swap(vin, vout);
  }
  *keys_out = kin;
  *vals_out = vin;
  return ARBX_OK;
}

template <typename K>
arbx_status radix_sort_impl(K* keys, K* kalt, uint32_t* vals, uint32_t* valt, bool iota, int64_t n, int key_bits,
                            cudaStream_t s, K** keys_out, uint32_t** vals_out) {
  *keys_out = keys;
  *vals_out = vals;
  if (n <= 0) return ARBX_OK;
  if (n > (int64_t(1) << 30)) { set_error("radix sort: n > 2^30"); return ARBX_ERR_UNSUPPORTED; }
  if (n == 1) {
    if (vals && iota) { ARBX_CUDA(cudaMemsetAsync(vals, 0, sizeof(uint32_t), s)); }
    return ARBX_OK;
  }
  if (key_bits < 1) key_bits = 1;
  if (key_bits > 8 * (int)sizeof(K)) key_bits = 8 * (int)sizeof(K);
  // 8-bit digits.  Measured on B200 (10^7 pairs): 10-bit digits save one pass at 30- and 39-bit
  // keys but cost 0.167 instead of 0.136 ms per pass (1024-entry look-back rows, ten ballots per
  // key, 32 KB of packed counters per block): 0.545 vs 0.469 ms at 30 bits, 0.667 vs 0.681 ms at
  // 39 bits -- no gain, so only the 8-bit kernels are instantiated.
  return radix_sort_bits<K, 8>(keys, kalt, vals, valt, iota, n, key_bits, s, keys_out, vals_out);
}

}  // namespace

// The query sort (32-bit keys, values = positions) with every buffer provided by the caller,
// including the sort's own `meta` words (digit histograms, tile tickets, look-back status:
// sort_meta_words(n, key_bits) of them, cleared here on the stream).  Calls no allocator: this
// is the sort of arbx_query_count_noalloc.  Same kernels as radix_sort_u32.
size_t sort_meta_words(int64_t n, int key_bits) {
  const int npass = (std::max(key_bits, 1) + 7) / 8;
  const size_t ntiles = (size_t)((n + SORT_TILE - 1) / SORT_TILE);
  return (size_t)npass * 256 + MAX_PASSES + (size_t)npass * ntiles * 256;
}
arbx_status radix_sort_u32_noalloc(uint32_t* keys, uint32_t* kalt, uint32_t* vals, uint32_t* valt, int64_t n,
                                   int key_bits, uint32_t* meta, size_t meta_capacity_words, cudaStream_t s,
                                   uint32_t** keys_out, uint32_t** vals_out) {
  using K = uint32_t;
  constexpr int BITS = 8, RADIX = 256;
  *keys_out = keys;
  *vals_out = vals;
  if (n <= 0) return ARBX_OK;
  if (n == 1) { ARBX_CUDA(cudaMemsetAsync(vals, 0, sizeof(uint32_t), s)); return ARBX_OK; }
  key_bits = std::max(1, std::min(32, key_bits));
  const int npass = (key_bits + BITS - 1) / BITS;
  const uint32_t top_mask = key_bits % BITS ? (1u << (key_bits % BITS)) - 1u : (uint32_t)(RADIX - 1);
  const uint32_t ntiles = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);
  const size_t meta_words = sort_meta_words(n, key_bits);
  if (meta_words > meta_capacity_words) { set_error("radix sort (no-alloc): meta buffer too small"); return ARBX_ERR_UNSUPPORTED; }
  ARBX_CUDA(cudaMemsetAsync(meta, 0, meta_words * sizeof(uint32_t), s));   // the buffer keeps the last call's contents
  uint32_t* ghist = meta;
  uint32_t* counters = meta + (size_t)npass * RADIX;
  uint32_t* status = counters + MAX_PASSES;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  {
    ProfScope ps(K_QSORT_HIST, s);
    const int64_t want = (n / 4 + 511) / 512;
    const int grid = (int)std::min<int64_t>(std::max<int64_t>(want, 1), (int64_t)sms * 4);
    hist_kernel<K, BITS><<<grid, 512, 0, s>>>(keys, (uint32_t)n, npass, top_mask, ghist);
    ARBX_LAUNCH_CHECK();
    hist_scan_kernel<BITS><<<npass, 256, 0, s>>>(ghist);
    ARBX_LAUNCH_CHECK();
  }
  const size_t smem_kv = sizeof(K) * SORT_TILE + sizeof(uint32_t) * SORT_WARPS * (RADIX / 2) + sizeof(uint32_t) * SORT_TILE;
  ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, BITS, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_kv));
  ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, BITS, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_kv));
  K* kin = keys; K* kout = kalt;
  uint32_t* vin = vals; uint32_t* vout = valt;
  for (int p = 0; p < npass; ++p) {
    const uint32_t* base = ghist + (size_t)p * RADIX;
    uint32_t* st = status + (size_t)p * ntiles * RADIX;
    const uint32_t dmask = p == npass - 1 ? top_mask : (uint32_t)(RADIX - 1);
    ProfScope ps(K_QSORT_PASS, s);
    if (p == 0)
      onesweep_pass<K, BITS, true, true><<<ntiles, SORT_THREADS, smem_kv, s>>>(kin, kout, nullptr, vout, (uint32_t)n, BITS * p, dmask, base, counters + p, st);
    else
      onesweep_pass<K, BITS, false, true><<<ntiles, SORT_THREADS, smem_kv, s>>>(kin, kout, vin, vout, (uint32_t)n, BITS * p, dmask, base, counters + p, st);
    ARBX_LAUNCH_CHECK();
    std::swap(kin, kout);
    std::swap(vin, vout);
  }
  *keys_out = kin;
  *vals_out = vin;
  return ARBX_OK;
}

arbx_status radix_sort_u64(unsigned long long* keys, unsigned long long* keys_alt, uint32_t* vals,
                           uint32_t* vals_alt, bool iota_vals, int64_t n, int key_bits,
                           cudaStream_t s, unsigned long long** keys_out, uint32_t** vals_out) {
  return radix_sort_impl<unsigned long long>(keys, keys_alt, vals, vals_alt, iota_vals, n, key_bits, s, keys_out, vals_out);
}
arbx_status radix_sort_u32(uint32_t* keys, uint32_t* keys_alt, uint32_t* vals, uint32_t* vals_alt,
                           bool iota_vals, int64_t n, int key_bits, cudaStream_t s,
                           uint32_t** keys_out, uint32_t** vals_out) {
  return radix_sort_impl<uint32_t>(keys, keys_alt, vals, vals_alt, iota_vals, n, key_bits, s, keys_out, vals_out);
}

}  // namespace arbx
