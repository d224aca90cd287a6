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
#include <atomic>

#include "common.cuh"

namespace arbx {
namespace {

constexpr int RADIX = 256;
constexpr int SORT_THREADS = 512;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_IPT = 8;                          // items per thread
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;   // 4096 elements per tile
constexpr uint32_t FLAG_AGG = 1u << 30, FLAG_INCL = 2u << 30, VAL_MASK = (1u << 30) - 1;
constexpr int MAX_PASSES = 8;
#ifndef SORT_LB
#define SORT_LB 8
#endif

__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v) {
  asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// lanes of the warp holding the same 8-bit digit: eight ballots, one per bit (plain ALU/vote
// work; the match.any instruction is far slower than this on sm_100)
__device__ __forceinline__ uint32_t match_digit(uint32_t d) {
  uint32_t peers = ~0u;
#pragma unroll
  for (int b = 0; b < 8; ++b) {
    const bool bit = (d >> b) & 1u;
    const uint32_t bal = __ballot_sync(~0u, bit);
    peers &= bit ? bal : ~bal;
  }
  return peers;
}

// ---- histogram of every digit in one read of the keys ---------------------------------------
template <typename K>
__global__ void __launch_bounds__(512) hist_kernel(const K* __restrict__ keys, uint32_t n, int npass,
                                                   uint32_t top_mask, uint32_t* __restrict__ ghist) {
  // top_mask: bits of the last digit that belong to the key (bits at or above key_bits are ignored)
  auto digit = [&](K k, int p) -> uint32_t { return (uint32_t)(k >> (8 * p)) & (p == npass - 1 ? top_mask : 255u); };
  __shared__ uint32_t sh[MAX_PASSES * RADIX];
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

// exclusive scan of each digit histogram, one block (256 threads) per pass
__global__ void __launch_bounds__(RADIX) hist_scan_kernel(uint32_t* ghist) {
  __shared__ uint32_t wsum[RADIX / 32];
  uint32_t* h = ghist + blockIdx.x * RADIX;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t v = h[threadIdx.x], x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t y = __shfl_up_sync(~0u, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  uint32_t base = 0;
  for (int i = 0; i < w; ++i) base += wsum[i];
  h[threadIdx.x] = base + x - v;
}

// ---- one digit pass ------------------------------------------------------------------------
template <typename K, bool IOTA, bool VALS>
__global__ void __launch_bounds__(SORT_THREADS, 2)
onesweep_pass(const K* __restrict__ kin, K* __restrict__ kout, const uint32_t* __restrict__ vin,
              uint32_t* __restrict__ vout, uint32_t n, int shift, uint32_t dmask,
              const uint32_t* __restrict__ digit_base, uint32_t* __restrict__ counter,
              uint32_t* __restrict__ status) {
  // dynamic shared memory: the tile (keys, later reused for values) then the per-warp digit counters
  extern __shared__ __align__(16) unsigned char sort_smem[];
  union Tile { K keys[SORT_TILE]; uint32_t vals[SORT_TILE]; };
  Tile& sm = *reinterpret_cast<Tile*>(sort_smem);
  uint32_t (*whist)[RADIX] = reinterpret_cast<uint32_t (*)[RADIX]>(sort_smem + sizeof(Tile));
  __shared__ uint32_t s_toff[RADIX];    // first position of digit d inside the sorted tile
  __shared__ uint32_t s_goff[RADIX];    // global position of tile position p with digit d = s_goff[d] + p
  __shared__ uint32_t s_wsum[RADIX / 32];
  __shared__ uint32_t s_tile;

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_tile = atomicAdd(counter, 1u);   // ticket: tile t starts only after tiles < t did
  for (int i = tid; i < SORT_WARPS * RADIX; i += SORT_THREADS) (&whist[0][0])[i] = 0;
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t tile_base = tile * (uint32_t)SORT_TILE;
  const uint32_t nvalid = min((uint32_t)SORT_TILE, n - tile_base);

  // warp-striped load: warp w owns SORT_IPT*32 consecutive elements.  Padding keys of a partial
  // last tile carry the largest digit of this pass, so they sort behind every real key.
  K key[SORT_IPT];
  uint32_t val[SORT_IPT];
  const uint32_t wbase = tile_base + w * (32 * SORT_IPT) + lane;
  const K pad_key = (K)dmask << shift;
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    uint32_t idx = wbase + j * 32;
    key[j] = idx < n ? kin[idx] : pad_key;
    if constexpr (VALS) val[j] = IOTA ? idx : (idx < n ? vin[idx] : 0u);
  }

  // stable rank of every key among the keys of its warp with the same digit.  The match
  // instructions of a batch are independent (their latency overlaps); the per-digit counters
  // are bumped by one leader lane per digit group with a shared-memory atomic, and program
  // order inside the warp keeps item j ahead of item j+1.
  uint16_t rank[SORT_IPT];
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr int MB = 8;
#pragma unroll
  for (int j0 = 0; j0 < SORT_IPT; j0 += MB) {
    uint32_t peers[MB];
#pragma unroll
    for (int j = 0; j < MB; ++j)
      peers[j] = match_digit((uint32_t)(key[j0 + j] >> shift) & dmask);
#pragma unroll
    for (int j = 0; j < MB; ++j) {
      const uint32_t d = (uint32_t)(key[j0 + j] >> shift) & dmask;
      const int leader = __ffs(peers[j]) - 1;
      uint32_t old = 0;
      if (lane == leader) old = atomicAdd(&whist[w][d], (uint32_t)__popc(peers[j]));
      old = __shfl_sync(~0u, old, leader);
      rank[j0 + j] = (uint16_t)(old + __popc(peers[j] & lt_mask));
    }
  }
  __syncthreads();

  // thread d < 256 owns digit d: exclusive scan over warps, tile count, publish, look back
  const int d = tid;
  uint32_t run = 0, pub = 0, x = 0;
  if (tid < RADIX) {
#pragma unroll
    for (int i = 0; i < SORT_WARPS; ++i) {
      uint32_t t = whist[i][d];
      whist[i][d] = run;
      run += t;
    }
    // padding keys of a partial last tile sit in digit dmask; nobody reads their count
    pub = run;
    if (d == (int)dmask) pub -= (uint32_t)SORT_TILE - nvalid;
    st_volatile_u32(&status[(size_t)tile * RADIX + d], (tile == 0 ? FLAG_INCL : FLAG_AGG) | pub);

    // exclusive scan of the tile counts over digits
    x = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(~0u, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) s_wsum[w] = x;
  }
  __syncthreads();
  if (tid < RADIX) {
    uint32_t wb = 0;
#pragma unroll
    for (int i = 0; i < RADIX / 32; ++i) wb += i < w ? s_wsum[i] : 0u;
    const uint32_t toff = wb + x - run;
    s_toff[d] = toff;

    uint32_t excl = 0;
    if (tile > 0) {
      // decoupled look-back, LB predecessors per round trip: the loads of a batch are
      // independent, so a walk over many aggregate-only tiles costs one latency per batch
      constexpr int LB = SORT_LB;
      int t = (int)tile - 1;
      bool done = false;
      while (!done) {
        uint32_t v[LB];
#pragma unroll
        for (int i = 0; i < LB; ++i)
          v[i] = t - i >= 0 ? ld_volatile_u32(&status[(size_t)(t - i) * RADIX + d]) : FLAG_INCL;
        int used = 0;
#pragma unroll
        for (int i = 0; i < LB; ++i) {
          if (!done && used == i) {
            const uint32_t f = v[i] >> 30;
            if (f != 0u) {            // published: take it; an inclusive prefix ends the walk
              excl += v[i] & VAL_MASK;
              used = i + 1;
              done = f == 2u;
            }
          }
        }
        t -= used;                    // resume at the first predecessor that was not ready
      }
      st_volatile_u32(&status[(size_t)tile * RADIX + d], FLAG_INCL | (excl + pub));
    }
    s_goff[d] = digit_base[d] + excl - toff;
  }
  __syncthreads();

  // scatter keys to their position inside the sorted tile
  uint16_t pos[SORT_IPT];
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    const uint32_t d = (uint32_t)(key[j] >> shift) & dmask;
    pos[j] = (uint16_t)(s_toff[d] + whist[w][d] + rank[j]);
    sm.keys[pos[j]] = key[j];
  }
  __syncthreads();
  uint32_t gpos[SORT_IPT];
#pragma unroll
  for (int j = 0; j < SORT_IPT; ++j) {
    const uint32_t p = j * SORT_THREADS + tid;
    const K k = sm.keys[p];
    const uint32_t d = (uint32_t)(k >> shift) & dmask;
    gpos[j] = s_goff[d] + p;
    if (p < nvalid) kout[gpos[j]] = k;
  }
  if constexpr (VALS) {
    __syncthreads();
#pragma unroll
    for (int j = 0; j < SORT_IPT; ++j) sm.vals[pos[j]] = val[j];
    __syncthreads();
#pragma unroll
    for (int j = 0; j < SORT_IPT; ++j) {
      const uint32_t p = j * SORT_THREADS + tid;
      if (p < nvalid) vout[gpos[j]] = sm.vals[p];
    }
  }
}

template <typename K>
arbx_status radix_sort_impl(K* keys, K* kalt, uint32_t* vals, uint32_t* valt, bool iota, int64_t n, int key_bits,
                            cudaStream_t s, K** keys_out, uint32_t** vals_out) {
  *keys_out = keys;
  *vals_out = vals;
  if (n <= 0) return ARBX_OK;
  if (n > (int64_t(1) << 30)) { set_error("radix sort: n > 2^30"); return ARBX_ERR_UNSUPPORTED; }
  const bool has_vals = vals != nullptr;
  if (n == 1) {
    if (has_vals && iota) { ARBX_CUDA(cudaMemsetAsync(vals, 0, sizeof(uint32_t), s)); }
    return ARBX_OK;
  }
  if (key_bits < 1) key_bits = 1;
  if (key_bits > 8 * (int)sizeof(K)) key_bits = 8 * (int)sizeof(K);
  const int npass = (key_bits + 7) / 8;
  const uint32_t top_mask = key_bits % 8 ? (1u << (key_bits % 8)) - 1u : 255u;
  const uint32_t ntiles = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);

  Scratch<uint32_t> meta;
  // meta: [npass*256] digit histograms | [npass] tile counters | [npass*ntiles*256] look-back status
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
    hist_kernel<K><<<grid, 512, 0, s>>>(keys, (uint32_t)n, npass, top_mask, ghist);
    ARBX_LAUNCH_CHECK();
    hist_scan_kernel<<<npass, RADIX, 0, s>>>(ghist);
    ARBX_LAUNCH_CHECK();
  }
  const size_t smem = (sizeof(K) > 4 ? sizeof(K) : 4) * SORT_TILE + sizeof(uint32_t) * SORT_WARPS * RADIX;
  static std::atomic<bool> attr_set{false};   // one instance per key type K
  if (!attr_set.load(std::memory_order_acquire)) {
    ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ARBX_CUDA(cudaFuncSetAttribute(onesweep_pass<K, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_set.store(true, std::memory_order_release);
  }
  K* kin = keys; K* kout = kalt;
  uint32_t* vin = vals; uint32_t* vout = valt;
  for (int p = 0; p < npass; ++p) {
    const uint32_t* base = ghist + (size_t)p * RADIX;
    uint32_t* st = status + (size_t)p * ntiles * RADIX;
    const uint32_t dmask = p == npass - 1 ? top_mask : 255u;
    ProfScope ps(kPassId, s);
    if (!has_vals)
      onesweep_pass<K, false, false><<<ntiles, SORT_THREADS, smem, s>>>(kin, kout, nullptr, nullptr, (uint32_t)n, 8 * p, dmask, base, counters + p, st);
    else if (p == 0 && iota)
      onesweep_pass<K, true, true><<<ntiles, SORT_THREADS, smem, s>>>(kin, kout, nullptr, vout, (uint32_t)n, 8 * p, dmask, base, counters + p, st);
    else
      onesweep_pass<K, false, true><<<ntiles, SORT_THREADS, smem, s>>>(kin, kout, vin, vout, (uint32_t)n, 8 * p, dmask, base, counters + p, st);
    ARBX_LAUNCH_CHECK();
    std::swap(kin, kout);
    std::swap(vin, vout);
  }
  *keys_out = kin;
  *vals_out = vin;
  return ARBX_OK;
}

}  // namespace

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
