// eviction_order.cuh -- NEXT-3: typed eviction order of the engine's KV pages.
// Declared in include/mori.h (mori_eviction_order).
//
//   GPU HBM : evict inactive first, then idle, then busy.   CPU DRAM: inactive, busy, idle.
//   Inside a type LRU; equal last-access times -> lower page id first (E1).
//   A page's type is its owner's placement: GPU queue busy, CPU queue idle, Waiting inactive.
//
// A stable least-significant-digit radix sort of the page ids over the 34-bit key
// (type rank : 2 | last access : 32), 8 bits per pass, five passes; stability gives the page-id
// tie-break for free because the first pass reads the pages in id order.  Free pages carry the
// all-ones key and end up behind every resident page.  Per pass, three small kernels:
//   evict_hist     per 1024-page tile, a shared-memory histogram of the pass's digit
//   evict_scan     exclusive scan of the [256][tiles] table in digit-major order (one CTA)
//   evict_scatter  per tile: rank of every page among the equal digits of its tile
//                  (__match_any_sync inside a warp, a [32][256] table across warps), then
//                  perm_out[table[digit][tile] + rank] = page
// Keys are never materialised: every pass recomputes them from owner / tier / last_access.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "rank_partition.cuh"

namespace mori {

constexpr int kEvictTile = 1024;
constexpr int kEvictPasses = 5;

struct EvictArgs {
  long long n_pages;
  int n_programs, which_tier, tiles;
  const int32_t* page_owner;
  const uint8_t* program_tier;
  const uint32_t* last_access;
};

// digit of `page` in pass 0..3 (last_access, low byte first) or 4 (type rank); free page: 0xFF / 3
__device__ __forceinline__ int evict_digit(const EvictArgs& a, int page, int pass) {
  const int o = a.page_owner[page];
  if (o < 0 || o >= a.n_programs) return pass == 4 ? 3 : 0xFF;
  if (pass < 4) return (int)((a.last_access[page] >> (8 * pass)) & 0xFF);
  const int t = a.program_tier[o];
  if (t > 1) return 0;                                               // inactive first in both tiers
  return a.which_tier == 0 ? (t == 1 ? 1 : 2) : (t == 0 ? 1 : 2);    // GPU: idle, busy / CPU: busy, idle
}

// Passes 1..3 sort on a byte of last_access that is zero for every resident page when the
// counters are small (ticks): such a pass cannot change the order of the resident pages -- it would
// only move free pages behind them, which the final type-rank pass does anyway -- so its three
// kernels return at once.  max_last is the largest resident last_access, found by pass 0.
__device__ __forceinline__ bool evict_pass_is_noop(int pass, const unsigned int* max_last) {
  return pass >= 1 && pass <= 3 && (*max_last >> (8 * pass)) == 0;
}

__global__ void __launch_bounds__(kEvictTile)
evict_hist_kernel(EvictArgs a, int pass, const int32_t* __restrict__ perm_in, int32_t* __restrict__ table,
                  int32_t* __restrict__ n_resident, unsigned int* __restrict__ max_last) {
  if (evict_pass_is_noop(pass, max_last)) return;
  __shared__ int hist[256];
  __shared__ int resident;
  __shared__ unsigned int tile_max;
  if (threadIdx.x == 0) tile_max = 0;
  if (threadIdx.x < 256) hist[threadIdx.x] = 0;
  if (threadIdx.x == 0) resident = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * kEvictTile + threadIdx.x;
  if (i < a.n_pages) {
    const int page = perm_in ? perm_in[i] : (int)i;
    atomicAdd(&hist[evict_digit(a, page, pass)], 1);
    if (pass == 0) {
      const int o = a.page_owner[page];
      if (o >= 0 && o < a.n_programs) { atomicAdd(&resident, 1); atomicMax(&tile_max, a.last_access[page]); }
    }
  }
  __syncthreads();
  if (threadIdx.x < 256) table[threadIdx.x * a.tiles + blockIdx.x] = hist[threadIdx.x];
  if (pass == 0 && threadIdx.x == 0 && resident) { atomicAdd(n_resident, resident); atomicMax(max_last, tile_max); }
}

// exclusive scan of table[256 * tiles] in place (digit-major), one CTA of 1024 threads
__global__ void __launch_bounds__(kRankMaxThreads)
evict_scan_kernel(int32_t* __restrict__ table, int entries, int pass, const unsigned int* __restrict__ max_last) {
  if (evict_pass_is_noop(pass, max_last)) return;
  __shared__ uint64_t warp_tot[33];
  const int per = (entries + blockDim.x - 1) / blockDim.x;
  const int lo = threadIdx.x * per, hi = min(entries, lo + per);
  long long s = 0;
  for (int e = lo; e < hi; ++e) s += table[e];
  uint64_t total;
  long long run = (long long)block_excl_scan((uint64_t)s, warp_tot, &total);
  for (int e = lo; e < hi; ++e) { const int v = table[e]; table[e] = (int)run; run += v; }
}

__global__ void __launch_bounds__(kEvictTile)
evict_scatter_kernel(EvictArgs a, int pass, const int32_t* __restrict__ perm_in,
                     const int32_t* __restrict__ table, int32_t* __restrict__ perm_out,
                     const unsigned int* __restrict__ max_last) {
  if (evict_pass_is_noop(pass, max_last)) {                          // identity pass: just hand the order on
    const long long j = (long long)blockIdx.x * kEvictTile + threadIdx.x;
    if (j < a.n_pages) perm_out[j] = perm_in[j];
    return;
  }
  __shared__ int wcnt[32][257];                                      // [warp][digit]; 257: no bank clash
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int e = threadIdx.x; e < 32 * 257; e += kEvictTile) (&wcnt[0][0])[e] = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * kEvictTile + threadIdx.x;
  const bool live = i < a.n_pages;
  const int page = live ? (perm_in ? perm_in[i] : (int)i) : -1;
  const int digit = live ? evict_digit(a, page, pass) : 256;         // padding matches only padding
  const unsigned peers = __match_any_sync(0xFFFFFFFFu, digit);
  const int rank_in_warp = __popc(peers & ((1u << lane) - 1u));
  if (live && rank_in_warp == 0) wcnt[warp][digit] = __popc(peers);
  __syncthreads();
  if (threadIdx.x < 256) {                                           // exclusive prefix over the 32 warps
    int base = 0;
    for (int w = 0; w < 32; ++w) { const int t = wcnt[w][threadIdx.x]; wcnt[w][threadIdx.x] = base; base += t; }
  }
  __syncthreads();
  if (live) perm_out[table[digit * a.tiles + blockIdx.x] + wcnt[warp][digit] + rank_in_warp] = page;
}

}  // namespace mori
