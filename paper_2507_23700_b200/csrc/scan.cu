// scan.cu -- query step T2: offsets = exclusive prefix sum of per-query counts (CSR offsets,
// PAPER.md:L69 "offsets").  Totals are carried in 64 bits so that a result
// larger than INT32_MAX is detected instead of wrapping (reading A11).
#include <algorithm>

#include "common.cuh"

namespace arbx {
namespace {

constexpr int ST = 256, SI = 8, SB = ST * SI;   // 2048 counts per block

__device__ __forceinline__ long long block_exclusive_scan(long long v, long long* total) {
  __shared__ long long wsum[ST / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  long long x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    long long y = __shfl_up_sync(~0u, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  long long base = 0, tot = 0;
#pragma unroll
  for (int i = 0; i < ST / 32; ++i) { if (i < w) base += wsum[i]; tot += wsum[i]; }
  *total = tot;
  __syncthreads();
  return base + x - v;
}

__global__ void __launch_bounds__(ST) block_sums_kernel(const int32_t* __restrict__ counts, int64_t nq,
                                                        long long* __restrict__ sums) {
  const int64_t base = (int64_t)blockIdx.x * SB + (int64_t)threadIdx.x * SI;
  long long v = 0;
#pragma unroll
  for (int e = 0; e < SI; ++e) if (base + e < nq) v += counts[base + e];
  long long tot;
  block_exclusive_scan(v, &tot);
  if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

// single block: exclusive scan of the block sums in place, grand total to *total
__global__ void __launch_bounds__(ST) scan_sums_kernel(long long* sums, int nb, long long* total) {
  long long carry = 0;
  for (int b0 = 0; b0 < nb; b0 += ST) {
    const int i = b0 + threadIdx.x;
    long long v = i < nb ? sums[i] : 0, tot;
    long long ex = block_exclusive_scan(v, &tot);
    if (i < nb) sums[i] = carry + ex;
    carry += tot;
  }
  if (threadIdx.x == 0) *total = carry;
}

__global__ void __launch_bounds__(ST) apply_kernel(const int32_t* __restrict__ counts, int64_t nq,
                                                   const long long* __restrict__ sums,
                                                   const long long* __restrict__ total,
                                                   int32_t* __restrict__ offsets) {
  const int64_t base = (int64_t)blockIdx.x * SB + (int64_t)threadIdx.x * SI;
  int32_t c[SI];
  long long v = 0;
#pragma unroll
  for (int e = 0; e < SI; ++e) { c[e] = base + e < nq ? counts[base + e] : 0; v += c[e]; }
  long long tot;
  long long run = sums[blockIdx.x] + block_exclusive_scan(v, &tot);
#pragma unroll
  for (int e = 0; e < SI; ++e) {
    if (base + e < nq) offsets[base + e] = (int32_t)run;
    run += c[e];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
    const long long t = *total;
    offsets[nq] = t > 0x7fffffffLL ? 0x7fffffff : (int32_t)t;
  }
}

__global__ void zero_total_kernel(int32_t* offsets, long long* total) { offsets[0] = 0; *total = 0; }

// A warp copies the stored rows of 32 consecutive queries into their CSR slices, which are
// adjacent: lane-strided over the ELEMENTS of the 32 slices (coalesced stores, independent
// loads); the row of an element is found by a 5-step search over the warp's 32 offsets.
__global__ void __launch_bounds__(ST) compact_rows_kernel(const int32_t* __restrict__ rows, int cap,
                                                          const int32_t* __restrict__ counts,
                                                          const int32_t* __restrict__ offsets,
                                                          int32_t* __restrict__ indices, int64_t nq) {
  const int lane = threadIdx.x & 31;
  const int64_t q0 = ((int64_t)blockIdx.x * ST + threadIdx.x) - lane;   // first query of this warp
  if (q0 >= nq) return;
  const int64_t q = q0 + lane;
  const int64_t qend = q0 + 32 < nq ? q0 + 32 : nq;
  const int o0 = offsets[q0];
  const int T = offsets[qend] - o0;                 // elements in this warp's 32 slices
  const int c = q < nq ? counts[q] : 0;
  const int rel = q < nq ? offsets[q] - o0 : T;     // start of lane's slice relative to the warp's
#pragma unroll 4   // loads of four steps in flight: the copy waits on memory (long scoreboard), 0.47 -> 0.36 ms at C3
  for (int e0 = 0; e0 < T; e0 += 32) {
    const int e = e0 + lane;
    int row = 0;
#pragma unroll
    for (int step = 16; step > 0; step >>= 1) {
      const int cand = row + step;                  // <= 31
      if (__shfl_sync(~0u, rel, cand) <= e) row = cand;
    }
    const int cr = __shfl_sync(~0u, c, row);
    const int rr = __shfl_sync(~0u, rel, row);
    if (e < T && cr <= cap) indices[o0 + e] = rows[(q0 + row) * cap + (e - rr)];   // cr > cap: traversal pass
  }
}

}  // namespace

arbx_status compact_rows(const int32_t* rows, int cap, const int32_t* counts, const int32_t* offsets,
                         int32_t* indices, int64_t nq, cudaStream_t s) {
  if (nq == 0) return ARBX_OK;
  ProfScope ps(K_SPATIAL_FILL, s);
  compact_rows_kernel<<<(unsigned)((nq + ST - 1) / ST), ST, 0, s>>>(rows, cap, counts, offsets, indices, nq);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

arbx_status exclusive_scan_i32(const int32_t* counts, int32_t* offsets, int64_t nq, long long* total_dev,
                               cudaStream_t s) {
  if (nq == 0) {
    zero_total_kernel<<<1, 1, 0, s>>>(offsets, total_dev);
    ARBX_LAUNCH_CHECK();
    return ARBX_OK;
  }
  const int nb = (int)((nq + SB - 1) / SB);
  ProfScope ps(K_SCAN, s);
  Scratch<long long> sums;
  ARBX_TRY(sums.alloc(nb, s));
  block_sums_kernel<<<nb, ST, 0, s>>>(counts, nq, sums.p);
  ARBX_LAUNCH_CHECK();
  scan_sums_kernel<<<1, ST, 0, s>>>(sums.p, nb, total_dev);
  ARBX_LAUNCH_CHECK();
  apply_kernel<<<nb, ST, 0, s>>>(counts, nq, sums.p, total_dev, offsets);
  ARBX_LAUNCH_CHECK();
  return ARBX_OK;
}

}  // namespace arbx
