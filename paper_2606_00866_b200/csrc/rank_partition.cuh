// rank_partition.cuh -- steps a1-a4 of the MORI hot path in ONE launch of ONE CTA (sm_100a).
//
// What it computes is declared in include/mori.h (mori_rank_partition): rank by idleness
// (P:L11, L151-152), prefix-sum the KV footprints, cut at both capacities,
// label the overflow WAITING and compact the five transition lists.
//
// n <= 8192 programs fit one CTA's shared memory as 64-bit (key, index) pairs, so the whole
// path is latency-bound: one launch, no global atomics, no host round trip.  The sort is a
// bitonic network in shared memory over keys padded to a power of two; strides <= 32 are
// warp-local (__syncwarp), only strides >= 64 cost a block barrier.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mori {

constexpr int kRankMaxN = 8192;
constexpr int kRankMaxThreads = 1024;

// Order-preserving 32-bit key of a float: canonical NaN last, -0 folded onto +0.
__device__ __forceinline__ uint32_t idleness_key(float x) {
  uint32_t b = __float_as_uint(x);
  if ((b & 0x7FFFFFFFu) > 0x7F800000u) return 0xFFFFFFFFu;  // any NaN
  if (b == 0x80000000u) b = 0u;                              // -0 == +0
  return b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u);
}

// Exclusive scan of one 64-bit value per thread across the CTA (blockDim.x multiple of 32).
// `warp_tot` is 33 words of shared memory; returns the exclusive prefix, *total gets the sum.
__device__ __forceinline__ uint64_t block_excl_scan(uint64_t v, uint64_t* warp_tot, uint64_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  uint64_t incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint64_t o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= d) incl += o;
  }
  __syncthreads();  // warp_tot may still be read from a previous scan
  if (lane == 31) warp_tot[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    uint64_t w = lane < n_warps ? warp_tot[lane] : 0;
    uint64_t wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint64_t o = __shfl_up_sync(0xFFFFFFFFu, wi, d);
      if (lane >= d) wi += o;
    }
    if (lane < n_warps) warp_tot[lane] = wi - w;  // exclusive warp offsets
    if (lane == 31) warp_tot[32] = wi;            // grand total
  }
  __syncthreads();
  *total = warp_tot[32];
  return warp_tot[warp] + incl - v;
}

// The same for N values per thread at once (one set of barriers for all of them): v[] come in as
// the thread's values and go out as their exclusive prefixes, total[] gets the sums.  warp_tot is
// 33 * N words of shared memory.
template <int N>
__device__ __forceinline__ void block_excl_scan_n(uint64_t (&v)[N], uint64_t* warp_tot, uint64_t (&total)[N]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  uint64_t incl[N];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    incl[k] = v[k];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint64_t o = __shfl_up_sync(0xFFFFFFFFu, incl[k], d);
      if (lane >= d) incl[k] += o;
    }
  }
  __syncthreads();  // warp_tot may still be read from a previous scan
  if (lane == 31) {
#pragma unroll
    for (int k = 0; k < N; ++k) warp_tot[33 * k + warp] = incl[k];
  }
  __syncthreads();
  if (warp < N) {                                    // warp k scans the warp totals of value k
    uint64_t* wt = warp_tot + 33 * warp;
    uint64_t w = lane < n_warps ? wt[lane] : 0;
    uint64_t wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint64_t o = __shfl_up_sync(0xFFFFFFFFu, wi, d);
      if (lane >= d) wi += o;
    }
    if (lane < n_warps) wt[lane] = wi - w;
    if (lane == 31) wt[32] = wi;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < N; ++k) {
    total[k] = warp_tot[33 * k + 32];
    v[k] = warp_tot[33 * k + warp] + incl[k] - v[k];
  }
}

// Per-program byte outputs (tier, lazy) are produced in RANK order but indexed by PROGRAM: as
// scattered one-byte global stores they cost a memory transaction each (n = 4096: ~2 us from the one
// SM that runs the tail).  They are staged in shared memory instead and written out coalesced.
__device__ __forceinline__ void flush_bytes(const uint8_t* s, uint8_t* __restrict__ g, int n) {
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += blockDim.x) g[i] = s[i];
}

// Ranking by counting, shared by every kernel that orders more keys than one CTA sorts well
// (rank_partition_multi, rank_tiers, sticky_rebalance, bfd_assign).  Keys are unique, so
// position(i) = #{j : key_j < key_i}.  Every CTA holds all n keys in its shared memory (built by
// the caller, __syncthreads() done); this CTA ranks the items of its slice -- one warp per K items,
// lanes striding j, shuffle reduction -- and writes order[position] = item (rank_by_counting64 /
// rank_by_counting128 below).  They return true in exactly one CTA, the LAST to finish (atomic
// ticket, reset for the next launch), after every CTA's order[] writes are visible to it (read them
// with __ldcg): that CTA carries on with the part of the algorithm that needs the whole order.
// The tail of every rank-by-counting kernel: true in exactly one CTA, the LAST to finish.
__device__ __forceinline__ bool last_cta_ticket(unsigned int* __restrict__ ticket) {
  __shared__ unsigned int s_ticket;
  __syncthreads();                                   // the CTA's order[] writes are ordered before thread 0 ...
  if (threadIdx.x == 0) {
    __threadfence();                                 // ... whose ONE fence (fences are cumulative) makes them
    s_ticket = atomicAdd(ticket, 1u);                // visible device-wide before the ticket is taken
    if (s_ticket == gridDim.x - 1) {
      *ticket = 0;                                   // ready for the next launch that uses this counter
      __threadfence();                               // every other CTA's writes are visible to this one now
    }
  }
  __syncthreads();
  return s_ticket == gridDim.x - 1;
}

// Unique 128-bit keys (sticky_rebalance, bfd_assign) sit in shared memory as one 16-byte word each
// (x = low half, y = high half) -- one LDS.128 per key read -- and the compare is the borrow of a
// 128-bit subtraction (four carry-chained ISETPs), branch-free.
// acc -= (a < b): a < b <=> a - b borrows, so one carry chain over the 32-bit words and a final
// subtract-with-borrow INTO the accumulator: five instructions per 128-bit compare-and-count (the
// compiler's own 128-bit compare takes ten, and the counting loop is bound by instruction issue),
// three per 64-bit one.  The count is -acc.
__device__ __forceinline__ void count_lt128(int& acc, const ulonglong2& a, const ulonglong2& b) {
  asm("{\n\t.reg .u32 t;\n\t"
      "sub.cc.u32 t, %1, %5;\n\t"
      "subc.cc.u32 t, %2, %6;\n\t"
      "subc.cc.u32 t, %3, %7;\n\t"
      "subc.cc.u32 t, %4, %8;\n\t"
      "subc.u32 %0, %0, 0;\n\t}"
      : "+r"(acc)
      : "r"((unsigned int)a.x), "r"((unsigned int)(a.x >> 32)), "r"((unsigned int)a.y), "r"((unsigned int)(a.y >> 32)),
        "r"((unsigned int)b.x), "r"((unsigned int)(b.x >> 32)), "r"((unsigned int)b.y), "r"((unsigned int)(b.y >> 32)));
}
__device__ __forceinline__ void count_lt64(int& acc, uint64_t a, uint64_t b) {
  asm("{\n\t.reg .u32 t;\n\t"
      "sub.cc.u32 t, %1, %3;\n\t"
      "subc.cc.u32 t, %2, %4;\n\t"
      "subc.u32 %0, %0, 0;\n\t}"
      : "+r"(acc)
      : "r"((unsigned int)a), "r"((unsigned int)(a >> 32)), "r"((unsigned int)b), "r"((unsigned int)(b >> 32)));
}

// K programs per warp pass: every key read from shared memory is compared against K keys held in
// registers, so the loop's shared-memory traffic -- what bounds it: n^2 reads of 16 bytes per launch,
// 268 MB at n = 4096 against ~36 TB/s over 148 SMs -- drops K-fold.
template <int K>
__device__ __forceinline__ void count_positions128(int n, const ulonglong2* __restrict__ keys,
                                                   int32_t* __restrict__ order, int lo, int hi) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  for (int i0 = lo + warp * K; i0 < hi; i0 += n_warps * K) {
    ulonglong2 ki[K];
    int c[K];
#pragma unroll
    for (int k = 0; k < K; ++k) { ki[k] = keys[min(i0 + k, n - 1)]; c[k] = 0; }
    int j = lane;
    for (; j + 32 < n; j += 64) {
      const ulonglong2 k0 = keys[j], k1 = keys[j + 32];
#pragma unroll
      for (int k = 0; k < K; ++k) { count_lt128(c[k], k0, ki[k]); count_lt128(c[k], k1, ki[k]); }
    }
    for (; j < n; j += 32) {
      const ulonglong2 k0 = keys[j];
#pragma unroll
      for (int k = 0; k < K; ++k) count_lt128(c[k], k0, ki[k]);
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
      int v = -c[k];
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
      if (lane == 0 && i0 + k < hi) order[v] = i0 + k;
    }
  }
}
__device__ __forceinline__ bool rank_by_counting128(int n, const ulonglong2* __restrict__ keys,
                                                    int32_t* __restrict__ order, unsigned int* __restrict__ ticket) {
  const int per = (n + gridDim.x - 1) / gridDim.x;
  const int lo = blockIdx.x * per, hi = min(n, lo + per);
  if (per >= 48) count_positions128<4>(n, keys, order, lo, hi);
  else if (per >= 16) count_positions128<2>(n, keys, order, lo, hi);
  else count_positions128<1>(n, keys, order, lo, hi);
  return last_cta_ticket(ticket);
}

// The same for unique 64-bit keys (rank_partition_multi, rank_tiers).
template <int K>
__device__ __forceinline__ void count_positions64(int n, const uint64_t* __restrict__ keys,
                                                  int32_t* __restrict__ order, int lo, int hi) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  for (int i0 = lo + warp * K; i0 < hi; i0 += n_warps * K) {
    uint64_t ki[K];
    int c[K];
#pragma unroll
    for (int k = 0; k < K; ++k) { ki[k] = keys[min(i0 + k, n - 1)]; c[k] = 0; }
    int j = lane;
    for (; j + 96 < n; j += 128) {
      const uint64_t k0 = keys[j], k1 = keys[j + 32], k2 = keys[j + 64], k3 = keys[j + 96];
#pragma unroll
      for (int k = 0; k < K; ++k) {
        count_lt64(c[k], k0, ki[k]); count_lt64(c[k], k1, ki[k]); count_lt64(c[k], k2, ki[k]); count_lt64(c[k], k3, ki[k]);
      }
    }
    for (; j < n; j += 32) {
      const uint64_t k0 = keys[j];
#pragma unroll
      for (int k = 0; k < K; ++k) count_lt64(c[k], k0, ki[k]);
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
      int v = -c[k];
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
      if (lane == 0 && i0 + k < hi) order[v] = i0 + k;
    }
  }
}
__device__ __forceinline__ bool rank_by_counting64(int n, const uint64_t* __restrict__ keys,
                                                   int32_t* __restrict__ order, unsigned int* __restrict__ ticket) {
  const int per = (n + gridDim.x - 1) / gridDim.x;
  const int lo = blockIdx.x * per, hi = min(n, lo + per);
  if (per >= 48) count_positions64<4>(n, keys, order, lo, hi);
  else if (per >= 16) count_positions64<2>(n, keys, order, lo, hi);
  else count_positions64<1>(n, keys, order, lo, hi);
  return last_cta_ticket(ticket);
}

// Steps a2-a4 for one CTA whose thread t owns ranks [t*IPT, (t+1)*IPT): prog[i] is the program at
// rank t*IPT + i (or -1 past n).  warp_tot = 66 words, bcast = 2 words of shared memory.
template <int IPT>
__device__ __forceinline__ void partition_tail(
    int n, const int (&prog)[IPT], const int32_t* __restrict__ kv_pages,
    const uint8_t* __restrict__ prev_tier, long long cap_gpu, long long cap_cpu,
    int32_t* __restrict__ order, uint8_t* __restrict__ tier, int32_t* __restrict__ bounds,
    long long* __restrict__ used, int32_t* __restrict__ lists, int32_t* __restrict__ list_counts,
    uint64_t* warp_tot, long long* bcast, uint8_t* s_tier /* n bytes of (dead) shared memory */) {
  const int tid = threadIdx.x;
  // ---- a2: footprints in rank order + exclusive prefix sum (int64) ----------------------------
  long long sz[IPT];
  long long tsum = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    int s = r < n ? kv_pages[prog[i]] : 0;
    sz[i] = s > 0 ? s : 0;
    tsum += sz[i];
  }
  uint64_t total_pages;
  long long run = (long long)block_excl_scan((uint64_t)tsum, warp_tot, &total_pages);
  long long incl[IPT];
#pragma unroll
  for (int i = 0; i < IPT; ++i) { run += sz[i]; incl[i] = run; }

  // ---- a3: GPU boundary: inclusive sums are non-decreasing, so the longest prefix that fits is
  //          the COUNT of ranks whose inclusive sum is <= capacity ------------------------------
  int c = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) c += (tid * IPT + i < n) && (incl[i] <= cap_gpu);
  uint64_t tot;
  block_excl_scan((uint64_t)c, warp_tot, &tot);
  const int b_gpu = (int)tot;
  if (tid == 0) bcast[0] = 0;
  __syncthreads();
#pragma unroll
  for (int i = 0; i < IPT; ++i)
    if (tid * IPT + i == b_gpu - 1) bcast[0] = incl[i];              // pages held by the GPU tier
  __syncthreads();
  const long long base = bcast[0];

  // ---- a3: CPU boundary, same argument on the sums past the GPU tier --------------------------
  c = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    c += (r < n) && (r >= b_gpu) && (incl[i] - base <= cap_cpu);
  }
  block_excl_scan((uint64_t)c, warp_tot, &tot);
  const int b_cpu = b_gpu + (int)tot;
  if (tid == 0) bcast[1] = base;
  __syncthreads();
#pragma unroll
  for (int i = 0; i < IPT; ++i)
    if (tid * IPT + i == b_cpu - 1) bcast[1] = incl[i];
  __syncthreads();
  if (tid == 0) {
    bounds[0] = b_gpu;
    bounds[1] = b_cpu;
    used[0] = base;
    used[1] = bcast[1] - base;
  }

  // ---- a3/a4: tiers, and the transition class of every rank ------------------------------------
  // counters packed 16 bits each (n <= 8192 < 65536): demote | promote | drop | admit ; reserve
  int cls[IPT];
  uint64_t packed = 0, rsv = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    cls[i] = -1;
    if (r < n) {
      const int now = r < b_gpu ? 0 : (r < b_cpu ? 1 : 2);
      s_tier[prog[i]] = (uint8_t)now;
      order[r] = prog[i];
      if (prev_tier != nullptr) {
        const int pv = prev_tier[prog[i]];
        const int was = pv == 0 ? 0 : (pv == 1 ? 1 : 2);
        if (was == 0 && now == 1) cls[i] = 0;
        else if (was == 1 && now == 0) cls[i] = 1;
        else if (was != 2 && now == 2) cls[i] = 2;
        else if (was == 2 && now == 0) cls[i] = 3;
        else if (was == 2 && now == 1) cls[i] = 4;
        if (cls[i] >= 0 && cls[i] < 4) packed += 1ull << (16 * cls[i]);
        if (cls[i] == 4) rsv += 1;
      }
    }
  }
  flush_bytes(s_tier, tier, n);
  if (prev_tier == nullptr) return;

  // ---- a4: compaction by rank.  Ascending lists take the exclusive count below; descending
  //          lists (demote, drop: most idle first) take total - inclusive count ------------------
  uint64_t pr[2] = {packed, rsv}, prt[2];
  block_excl_scan_n<2>(pr, warp_tot, prt);                           // warp_tot: 66 words
  uint64_t pex = pr[0], rex = pr[1];
  const uint64_t ptot = prt[0], rtot = prt[1];
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int k = cls[i];
    if (k < 0) continue;
    int pos;
    if (k == 4) {
      pos = (int)rex++;
    } else {
      const int below = (int)((pex >> (16 * k)) & 0xFFFF);
      pex += 1ull << (16 * k);
      const int all = (int)((ptot >> (16 * k)) & 0xFFFF);
      pos = (k == 0 || k == 2) ? all - 1 - below : below;
    }
    lists[(size_t)k * n + pos] = prog[i];
  }
  if (tid < 4) list_counts[tid] = (int)((ptot >> (16 * tid)) & 0xFFFF);
  if (tid == 4) list_counts[4] = (int)rtot;
}

// IPT = ranks per thread (n_pad / blockDim.x), blocked: thread t owns ranks [t*IPT, (t+1)*IPT).
template <int IPT>
__global__ void __launch_bounds__(kRankMaxThreads, 1)
rank_partition_kernel(int n, int n_pad, const float* __restrict__ idleness,
                      const int32_t* __restrict__ kv_pages, const uint8_t* __restrict__ prev_tier,
                      long long cap_gpu, long long cap_cpu, int32_t* __restrict__ order,
                      uint8_t* __restrict__ tier, int32_t* __restrict__ bounds,
                      long long* __restrict__ used, int32_t* __restrict__ lists,
                      int32_t* __restrict__ list_counts) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint64_t* keys = reinterpret_cast<uint64_t*>(smem_raw);            // [n_pad]
  uint64_t* warp_tot = keys + n_pad;                                 // [2][33]
  long long* bcast = reinterpret_cast<long long*>(warp_tot + 66);    // [2]
  const int tid = threadIdx.x, nt = blockDim.x;

  // ---- a1: keys ------------------------------------------------------------------------------
  for (int i = tid; i < n_pad; i += nt)
    keys[i] = i < n ? ((uint64_t)idleness_key(idleness[i]) << 32) | (uint32_t)i
                    : 0xFFFFFFFFFFFFFFFFull;                         // padding sorts last
  __syncthreads();

  // ---- a1: bitonic sort, ascending ------------------------------------------------------------
  // Pair q of a stage with stride j touches elements i = ((q & ~(j-1)) << 1) | (q & (j-1)) and
  // i | j.  For j <= 32 the 32 pairs [32w, 32w+32) of one warp touch exactly the 64 elements
  // [64w, 64w+64) whatever j is, so the stages j = 32 ... 1 of every merge run back to back
  // inside a warp with __syncwarp only; a block barrier is needed only around strides >= 64.
  // (n_pad = 4096: 21 block barriers instead of 78; n_pad <= 64: none.)
  const int n_pairs = n_pad >> 1;                    // n_pad >= 64: a multiple of 32, whole warps
  for (int k = 2; k <= n_pad; k <<= 1) {
    int j = k >> 1;
    for (; j >= 64; j >>= 1) {
      for (int q = tid; q < n_pairs; q += nt) {
        const int i = ((q & ~(j - 1)) << 1) | (q & (j - 1));
        const int p = i | j;
        const uint64_t a = keys[i], b = keys[p];
        if ((a > b) == ((i & k) == 0)) { keys[i] = b; keys[p] = a; }
      }
      __syncthreads();
    }
    for (int q = tid; q < n_pairs; q += nt) {        // nt is a multiple of 32: whole warps iterate together
      for (int jj = j; jj > 0; jj >>= 1) {
        const int i = ((q & ~(jj - 1)) << 1) | (q & (jj - 1));
        const int p = i | jj;
        const uint64_t a = keys[i], b = keys[p];
        if ((a > b) == ((i & k) == 0)) { keys[i] = b; keys[p] = a; }
        __syncwarp();
      }
    }
    if (k >= 64 || k == n_pad) __syncthreads();      // next merge (or the scan) crosses warps
  }

  int prog[IPT];
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    prog[i] = r < n ? (int)(uint32_t)keys[r] : -1;
  }
  partition_tail<IPT>(n, prog, kv_pages, prev_tier, cap_gpu, cap_cpu, order, tier, bounds, used, lists,
                      list_counts, warp_tot, bcast, reinterpret_cast<uint8_t*>(keys));   // the keys are dead
}

// ---------------------------------------------------------------------------------------------
// n > 1024: the sort of one CTA is bound by ONE SM's shared-memory bandwidth (78 passes over
// 32-64 KiB).  Ranking by counting spreads a1 over the whole chip instead: the keys are unique
// (the index is their low half), so rank(i) = #{j : key_j < key_i} is the sorted position, and
// n^2 <= 6.7e7 compares over 148 SMs are ~1 us.  Every CTA builds all n keys in its shared
// memory, ranks its slice of programs (one warp per program, lanes striding j) and writes
// order[rank] = program.  The LAST CTA to finish (atomic ticket) runs a2-a4 on the completed
// order: one launch, no grid barrier, no co-residency requirement.
template <int IPT>
__global__ void __launch_bounds__(kRankMaxThreads, 1)
rank_partition_multi_kernel(int n, const float* __restrict__ idleness,
                            const int32_t* __restrict__ kv_pages, const uint8_t* __restrict__ prev_tier,
                            long long cap_gpu, long long cap_cpu, int32_t* __restrict__ order,
                            uint8_t* __restrict__ tier, int32_t* __restrict__ bounds,
                            long long* __restrict__ used, int32_t* __restrict__ lists,
                            int32_t* __restrict__ list_counts, int32_t* __restrict__ scratch_order,
                            unsigned int* __restrict__ ticket) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint64_t* keys = reinterpret_cast<uint64_t*>(smem_raw);            // [n]
  uint64_t* warp_tot = keys + n;                                     // [2][33]
  long long* bcast = reinterpret_cast<long long*>(warp_tot + 66);    // [2]
  // sizes and previous tiers, kept for the last CTA's tail: there they are read in RANK order, which
  // from global memory is a scattered gather (one transaction per program) and from here is free
  int32_t* s_kv = reinterpret_cast<int32_t*>(bcast + 2);             // [n]
  uint8_t* s_prev = reinterpret_cast<uint8_t*>(s_kv + n);            // [n]
  const int tid = threadIdx.x;
  for (int i = tid; i < n; i += blockDim.x) {
    keys[i] = ((uint64_t)idleness_key(idleness[i]) << 32) | (uint32_t)i;
    s_kv[i] = kv_pages[i];
    if (prev_tier != nullptr) s_prev[i] = prev_tier[i];
  }
  __syncthreads();
  // the CTAs exchange the order through library-owned DEVICE scratch; the caller's arrays are
  // written once, by the last CTA -- so they may be mapped host memory
  if (!rank_by_counting64(n, keys, scratch_order, ticket)) return;

  int prog[IPT];
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    prog[i] = r < n ? __ldcg(scratch_order + r) : -1;   // written by other CTAs: read through L2
  }
  partition_tail<IPT>(n, prog, s_kv, prev_tier != nullptr ? s_prev : nullptr, cap_gpu, cap_cpu, order, tier, bounds,
                      used, lists, list_counts, warp_tot, bcast, reinterpret_cast<uint8_t*>(keys));   // the keys are dead
}

// ---------------------------------------------------------------------------------------------
// NEXT-4(ii): the same ranking cut by T capacities instead of two ("a second idleness
// threshold", "an intermediate tier"): tier t = the longest run of the ranking right after tier
// t-1 whose pages fit cap[t]; the rest is Waiting (tier value T).  Declared in include/mori.h
// (mori_rank_partition_tiers).  Ranking by counting on every SM for every n, last CTA cuts.
constexpr int kMaxTiers = 8;
struct TierCaps { long long cap[kMaxTiers]; int n_tiers; };

template <int IPT>
__global__ void __launch_bounds__(kRankMaxThreads, 1)
rank_tiers_kernel(int n, const float* __restrict__ idleness, const int32_t* __restrict__ kv_pages,
                  const TierCaps caps, const uint8_t* __restrict__ prev_tier, int32_t* __restrict__ order,
                  uint8_t* __restrict__ tier, int32_t* __restrict__ bounds, long long* __restrict__ used,
                  int32_t* __restrict__ moves, int32_t* __restrict__ move_counts,
                  int32_t* __restrict__ scratch_order, unsigned int* __restrict__ ticket) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint64_t* keys = reinterpret_cast<uint64_t*>(smem_raw);            // [n]
  uint64_t* warp_tot = keys + n;                                     // [33]
  long long* bcast = reinterpret_cast<long long*>(warp_tot + 33);    // [2]
  const int tid = threadIdx.x;
  for (int i = tid; i < n; i += blockDim.x)
    keys[i] = ((uint64_t)idleness_key(idleness[i]) << 32) | (uint32_t)i;
  __syncthreads();
  if (!rank_by_counting64(n, keys, scratch_order, ticket)) return;

  int prog[IPT];
  long long incl[IPT];
  long long tsum = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    prog[i] = r < n ? __ldcg(scratch_order + r) : -1;
    if (r < n) order[r] = prog[i];                                   // the caller's array: written once, here
    const int s = r < n ? kv_pages[prog[i]] : 0;
    incl[i] = s > 0 ? s : 0;
    tsum += incl[i];
  }
  uint64_t tot;
  long long run = (long long)block_excl_scan((uint64_t)tsum, warp_tot, &tot);
#pragma unroll
  for (int i = 0; i < IPT; ++i) { run += incl[i]; incl[i] = run; }   // inclusive sums in rank order

  int my_tier[IPT];
#pragma unroll
  for (int i = 0; i < IPT; ++i) my_tier[i] = caps.n_tiers;           // Waiting unless a tier takes it
  int b_prev = 0;
  long long base = 0;
  for (int t = 0; t < caps.n_tiers; ++t) {
    int c = 0;
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
      const int r = tid * IPT + i;
      c += (r < n) && (r >= b_prev) && (incl[i] - base <= caps.cap[t]);
    }
    block_excl_scan((uint64_t)c, warp_tot, &tot);
    const int b = b_prev + (int)tot;
    if (tid == 0) bcast[0] = base;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
      const int r = tid * IPT + i;
      if (r >= b_prev && r < b) my_tier[i] = t;
      if (r == b - 1 && b > b_prev) bcast[0] = incl[i];
    }
    __syncthreads();
    const long long top = bcast[0];
    if (tid == 0) { bounds[t] = b; used[t] = top - base; }
    base = top;
    b_prev = b;
    __syncthreads();                                                 // bcast is rewritten next round
  }
  uint8_t* s_tier = reinterpret_cast<uint8_t*>(keys);                // the keys are dead (barriers above)
#pragma unroll
  for (int i = 0; i < IPT; ++i) if (prog[i] >= 0) s_tier[prog[i]] = (uint8_t)my_tier[i];
  flush_bytes(s_tier, tier, n);
  if (prev_tier == nullptr) return;

  // move lists (the two-tier rule of P:L206 / L208 carried over): DOWN the hierarchy most idle
  // first, UP least idle first; one scan of two 32-bit counters packed in a 64-bit word
  int dir[IPT];
  uint64_t packed = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    dir[i] = -1;
    if (prog[i] >= 0) {
      const int pv = prev_tier[prog[i]];
      const int was = pv < caps.n_tiers ? pv : caps.n_tiers;
      if (my_tier[i] > was) { dir[i] = 0; packed += 1ull; }
      else if (my_tier[i] < was) { dir[i] = 1; packed += 1ull << 32; }
    }
  }
  uint64_t ptot;
  uint64_t pex = block_excl_scan(packed, warp_tot, &ptot);
  const int n_down = (int)(ptot & 0xFFFFFFFFu);
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    if (dir[i] == 0) { moves[n_down - 1 - (int)(pex & 0xFFFFFFFFu)] = prog[i]; pex += 1ull; }
    else if (dir[i] == 1) { moves[(size_t)n + (int)(pex >> 32)] = prog[i]; pex += 1ull << 32; }
  }
  if (threadIdx.x == 0) { move_counts[0] = n_down; move_counts[1] = (int)(ptot >> 32); }
}

}  // namespace mori
