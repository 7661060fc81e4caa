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
//
// Pools of up to 131 072 pages (every BASELINE.json config: 10 240 ... 65 536) take ONE launch
// instead: evict_order_cluster_kernel, a thread-block CLUSTER of 8 CTAs that keeps the whole sort
// on chip -- items ride in registers, per-warp digit counters in shared memory, the per-CTA digit
// totals are exchanged through distributed shared memory, and the only global traffic is one
// coalesced 8-byte scatter and reload per pass.  Passes separated by cluster barriers, not launches.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include <cooperative_groups.h>

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

// ---------------------------------------------------------------------------------------------
// One launch, one cluster of 8 CTAs x 1024 threads.
//
// An item is (key : 34 | page : 30) in one 64-bit word, key = type rank : 2 | last access : 32
// (free pages: all ones, they end up behind every resident page).  CTA c owns the contiguous
// segment [c*seg, (c+1)*seg) of the current order, warp w of it a contiguous sub-segment, walked
// in rounds of 32 consecutive items -- so "CTA, warp, round, lane" IS the current order and a
// counting pass that respects it is stable.  Per 8-bit pass:
//   sweep A   every warp counts its items per digit in its OWN row of wc[32][256]
//             (__match_any_sync groups equal digits, the group's first lane adds the group size)
//   prefix    thread d turns column d into exclusive offsets over the warps; tot[d] = column sum
//   exchange  cluster barrier; thread d reads tot[d] of all 8 CTAs through distributed shared
//             memory: digits below d anywhere + digit d in lower CTAs = where this CTA's digit-d
//             items start (one block scan over the 256 digits)
//   sweep B   the same walk again, now handing out positions; the item goes to out[position]
//   reload    cluster barrier; every thread reloads its (coalesced) share of the new order
// Pass 0 also counts the resident pages and finds the largest last-access value; passes whose
// byte of it is zero for every resident page are skipped outright (tick-sized counters: 2 passes
// instead of 5).
constexpr int kEvictCluster = 8;                                    // portable cluster size
constexpr int kEvictClusterMaxPages = kEvictCluster * 1024 * 16;

__device__ __forceinline__ uint64_t evict_item(const EvictArgs& a, int page, bool& resident, unsigned& last) {
  const int o = a.page_owner[page];
  resident = o >= 0 && o < a.n_programs;
  if (!resident) { last = 0; return (~0ull << 30) | (uint32_t)page; }
  last = a.last_access[page];
  const int t = a.program_tier[o];
  const int rank = t > 1 ? 0 : (a.which_tier == 0 ? (t == 1 ? 1 : 2) : (t == 0 ? 1 : 2));
  return ((uint64_t)rank << 62) | ((uint64_t)last << 30) | (uint32_t)page;
}
__device__ __forceinline__ int evict_item_digit(uint64_t item, int pass) {
  return pass == 4 ? (int)(item >> 62) : (int)((item >> (30 + 8 * pass)) & 0xFF);
}

// The cluster size is a launch attribute (8, or 16 where the device allows the non-portable size).
template <int R>
__global__ void __launch_bounds__(1024, 1)
evict_order_cluster_kernel(EvictArgs a, uint64_t* __restrict__ buf0, uint64_t* __restrict__ buf1,
                           int32_t* __restrict__ victims, int32_t* __restrict__ n_resident) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = (int)cluster.block_rank();
  const int csize = (int)cluster.num_blocks();
  __shared__ int wc[32][257];
  __shared__ int tot[256];
  __shared__ int s_stat[2];                                          // resident pages, max last access (this CTA)
  __shared__ unsigned s_gmax;
  __shared__ uint64_t warp_tot[33];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long N = a.n_pages;
  const int seg = (int)(((N + csize - 1) / csize + 1023) / 1024 * 1024);
  const int per_warp = seg / 32, rounds = per_warp / 32;             // rounds <= R (host checks)
  const long long first = (long long)crank * seg + (long long)warp * per_warp + lane;

  if (tid < 2) s_stat[tid] = 0;
  __syncthreads();
  uint64_t item[R];
  {
    int res = 0; unsigned mx = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const long long i = first + r * 32;
      item[r] = ~0ull;                                               // "no item": skipped everywhere
      if (r < rounds && i < N) {
        bool rs; unsigned la;
        item[r] = evict_item(a, (int)i, rs, la);
        res += rs; mx = max(mx, la);
      }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { res += __shfl_xor_sync(0xFFFFFFFFu, res, d); mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, d)); }
    if (lane == 0) { atomicAdd(&s_stat[0], res); atomicMax(reinterpret_cast<unsigned*>(&s_stat[1]), mx); }
  }
  unsigned gmax = 0xFFFFFFFFu;                                       // unknown until pass 0 has exchanged it
  uint64_t* out = buf0;
  for (int pass = 0; pass < 5; ++pass) {
    if (pass >= 1 && pass <= 3 && (gmax >> (8 * pass)) == 0) continue;   // cannot reorder resident pages
    const bool last_pass = pass == 4;
    for (int e = tid; e < 32 * 257; e += 1024) (&wc[0][0])[e] = 0;
    __syncthreads();
    // ---- sweep A: per-warp digit counts (the lanes with the same digit are remembered for sweep B) --
    unsigned peers_of[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      peers_of[r] = 0;
      if (r < rounds) {
        const int d = item[r] == ~0ull ? 256 : evict_item_digit(item[r], pass);
        const unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
        peers_of[r] = peers;
        if (d < 256 && lane == __ffs(peers) - 1) wc[warp][d] += __popc(peers);
        __syncwarp();
      }
    }
    __syncthreads();
    if (tid < 256) {
      int run = 0;
      for (int w = 0; w < 32; ++w) { const int t = wc[w][tid]; wc[w][tid] = run; run += t; }
      tot[tid] = run;
    }
    cluster.sync();
    // ---- exchange: where this CTA's items of every digit start -----------------------------------
    int all = 0, below = 0;
    if (tid < 256) {
      for (int c = 0; c < csize; ++c) {
        const int v = *cluster.map_shared_rank(&tot[tid], c);
        all += v; below += c < crank ? v : 0;
      }
    }
    if (pass == 0 && tid == 0) {
      int res = 0; unsigned mx = 0;
      for (int c = 0; c < csize; ++c) {
        const int* st = cluster.map_shared_rank(&s_stat[0], c);
        res += st[0]; mx = max(mx, (unsigned)st[1]);
      }
      s_gmax = mx;
      if (crank == 0) *n_resident = res;
    }
    uint64_t total;
    const int gbase = (int)block_excl_scan((uint64_t)all, warp_tot, &total) + below;   // (syncs the block)
    if (pass == 0) gmax = s_gmax;
    if (tid < 256)
      for (int w = 0; w < 32; ++w) wc[w][tid] += gbase;
    __syncthreads();
    // ---- sweep B: positions, scatter --------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (r < rounds) {
        const int d = item[r] == ~0ull ? 256 : evict_item_digit(item[r], pass);
        const unsigned peers = peers_of[r];
        const int leader = __ffs(peers) - 1;
        int start = 0;
        if (d < 256 && lane == leader) { start = wc[warp][d]; wc[warp][d] = start + __popc(peers); }
        start = __shfl_sync(0xFFFFFFFFu, start, leader);
        if (d < 256) {
          const int pos = start + __popc(peers & ((1u << lane) - 1u));
          if (last_pass) victims[pos] = (int)(item[r] & 0x3FFFFFFFu);
          else out[pos] = item[r];
        }
        __syncwarp();
      }
    }
    cluster.sync();                                                  // the new order is complete and visible
    if (!last_pass) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const long long i = first + r * 32;
        if (r < rounds && i < N) item[r] = __ldcg(out + i);
      }
      out = out == buf0 ? buf1 : buf0;
    }
  }
}

}  // namespace mori
