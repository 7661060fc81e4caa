// bfd_assign.cuh -- NEXT-4(i): Waiting-queue promotions packed across replicas:
// "Best-Fit-Decreasing bin packing across replicas, selecting the replica with the most available
// capacity first".  Declared in include/mori.h (mori_bfd_assign).
//
// Order: largest candidate first; equal sizes keep the promotion priority (returning before new,
// least idle, index).  The order comes from ranking unique 128-bit keys by counting on every SM
// (as in sticky_rebalance.cuh); the last CTA then walks the candidates in that order.  The walk is
// the one inherently sequential step of the rule (every admission changes the next arg-max), so
// what matters is the latency of one arg-max: with 32-bit capacities (the usual case) lane r of
// one warp holds replica r, the maximum is one redux.sync and the winner the lowest set bit of a
// ballot of "equals the maximum" (~100 cycles per admitted candidate); capacities beyond 2^31
// take a single-thread walk with the replicas in registers.  A shuffle-butterfly arg-max on
// 64-bit values measured 3x slower than either.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "rank_partition.cuh"

namespace mori {

constexpr int kBfdMaxReplicas = 32;


// The walk, by ONE thread with every replica's free pages in registers (RP = 8, 16 or 32 slots,
// unused ones hold -1 and never win): arg-max by an unrolled scan (first maximum = lowest index),
// recomputed only after an admission -- a candidate that does not fit leaves it unchanged.
template <int RP>
__device__ __forceinline__ void bfd_walk(int m, const int32_t* ssize, int32_t* sdest, int n_replicas,
                                         const long long* __restrict__ free_pages, long long* __restrict__ free_out) {
  long long fr[RP];
#pragma unroll
  for (int r = 0; r < RP; ++r) fr[r] = r < n_replicas ? free_pages[r] : -1;
  long long best = fr[0]; int who = 0;
#pragma unroll
  for (int r = 1; r < RP; ++r) if (fr[r] > best) { best = fr[r]; who = r; }
  int s_next = m > 0 ? ssize[0] : 0;
  for (int k = 0; k < m; ++k) {
    const int s = s_next;
    if (k + 1 < m) s_next = ssize[k + 1];
    if ((long long)s <= best) {
      sdest[k] = who;
#pragma unroll
      for (int r = 0; r < RP; ++r) fr[r] -= r == who ? (long long)s : 0;
      best = fr[0]; who = 0;
#pragma unroll
      for (int r = 1; r < RP; ++r) if (fr[r] > best) { best = fr[r]; who = r; }
    } else {
      sdest[k] = -1;
    }
  }
#pragma unroll
  for (int r = 0; r < RP; ++r) if (r < n_replicas) free_out[r] = fr[r];
}

// The same walk for up to 8 replicas with capacities below 2^27 pages (the usual case: 2^27 pages of
// 2 MiB are 256 TiB): each replica is ONE 32-bit key, free * 8 + (7 - r), so a plain integer maximum
// over 8 registers yields the largest capacity AND, among equals, the lowest replica index.  The
// loop-carried chain per admitted candidate is compare -> select -> a three-level max: ~20 cycles,
// against ~100 for the warp-wide redux + ballot, and nothing at all for one that does not fit.
__device__ __forceinline__ void bfd_walk_packed8(int m, const int32_t* ssize, int32_t* sdest, int n_replicas,
                                                 const long long* __restrict__ free_pages,
                                                 long long* __restrict__ free_out) {
  int key[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) key[r] = r < n_replicas ? (int)free_pages[r] * 8 + (7 - r) : -1;
  int best = max(max(max(key[0], key[1]), max(key[2], key[3])), max(max(key[4], key[5]), max(key[6], key[7])));
  // One step.  "fits" is best >= 8 s (the low three bits are below 8); the keys are unique, so
  // "key == best" names the winner without decoding its index, and the destination (7 - (best & 7))
  // is computed off the loop-carried chain  best -> compare -> subtract -> max.  A candidate that
  // does not fit costs one compare (measured: the branch-free form of this step is 1.5x slower on
  // queues where a third of the candidates do not fit).
  auto step = [&](int k, int s) {
    const int s8 = s > (1 << 27) ? 0x7FFFFFFF : s * 8;
    if (best >= s8) {
      sdest[k] = 7 - (best & 7);
#pragma unroll
      for (int r = 0; r < 8; ++r) key[r] -= key[r] == best ? s8 : 0;
      best = max(max(max(key[0], key[1]), max(key[2], key[3])), max(max(key[4], key[5]), max(key[6], key[7])));
    } else {
      sdest[k] = -1;
    }
  };
  int k = 0;
  for (; k + 4 <= m; k += 4) {                                       // sizes read four ahead of the chain
    const int s0 = ssize[k], s1 = ssize[k + 1], s2 = ssize[k + 2], s3 = ssize[k + 3];
    step(k, s0); step(k + 1, s1); step(k + 2, s2); step(k + 3, s3);
  }
  for (; k < m; ++k) step(k, ssize[k]);
#pragma unroll
  for (int r = 0; r < 8; ++r) if (r < n_replicas) free_out[r] = key[r] >> 3;
}

__global__ void __launch_bounds__(kRankMaxThreads, 1)
bfd_assign_kernel(int m, const int32_t* __restrict__ size, const float* __restrict__ idleness,
                  const uint8_t* __restrict__ flags, int n_replicas, const long long* __restrict__ free_pages,
                  int32_t* __restrict__ replica, long long* __restrict__ free_out,
                  int32_t* __restrict__ order, unsigned int* __restrict__ ticket) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ulonglong2* keys = reinterpret_cast<ulonglong2*>(smem_raw);        // [m] (x = low half, y = high half)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  for (int i = tid; i < m; i += blockDim.x) {
    const int s = size[i] > 0 ? size[i] : 0;
    keys[i] = make_ulonglong2(((unsigned long long)idleness_key(idleness[i]) << 32) | (uint32_t)i,   // least idle, then index
                              ((unsigned long long)(~(uint32_t)s) << 1) | ((flags[i] & 4) ? 1u : 0u));  // size descending, then class
  }
  __syncthreads();
  if (!rank_by_counting128(m, keys, order, ticket)) return;

  // ---- last CTA: sizes in packing order into shared memory, then the one-warp walk ---------------
  int32_t* ssize = reinterpret_cast<int32_t*>(keys);                 // [m] (keys are dead)
  int32_t* sdest = ssize + m;                                        // [m]
  __syncthreads();
  for (int k = tid; k < m; k += blockDim.x) {
    const int s = size[__ldcg(order + k)];
    ssize[k] = s > 0 ? s : 0;
  }
  __syncthreads();
  bool small = true;                                                  // every capacity fits an int?
  for (int r = 0; r < n_replicas; ++r) small = small && free_pages[r] <= 0x7FFFFFFFll;
  bool packed = true;                                                 // every capacity below 2^27 pages?
  for (int r = 0; r < n_replicas; ++r) packed = packed && free_pages[r] < (1ll << 27);
  if (packed && n_replicas <= 8) {
    if (tid == 0) bfd_walk_packed8(m, ssize, sdest, n_replicas, free_pages, free_out);
  } else if (small) {
    // 32-bit capacities (the usual case): warp 0, lane r = replica r; the maximum comes from one
    // redux.sync, the winner from a ballot of "equals the maximum" (lowest set bit).
    if (warp == 0) {
      int fr = lane < n_replicas ? (int)free_pages[lane] : -1;
      int best = __reduce_max_sync(0xFFFFFFFFu, fr);
      int who = __ffs(__ballot_sync(0xFFFFFFFFu, fr == best)) - 1;
      for (int k = 0; k < m; ++k) {
        const int s = ssize[k];                                       // broadcast read
        const bool fits = s <= best;
        if (lane == 0) sdest[k] = fits ? who : -1;
        if (fits) {
          if (lane == who) fr -= s;
          best = __reduce_max_sync(0xFFFFFFFFu, fr);
          who = __ffs(__ballot_sync(0xFFFFFFFFu, fr == best)) - 1;
        }
      }
      if (lane < n_replicas) free_out[lane] = fr;
    }
  } else if (tid == 0) {
    if (n_replicas <= 8) bfd_walk<8>(m, ssize, sdest, n_replicas, free_pages, free_out);
    else if (n_replicas <= 16) bfd_walk<16>(m, ssize, sdest, n_replicas, free_pages, free_out);
    else bfd_walk<32>(m, ssize, sdest, n_replicas, free_pages, free_out);
  }
  __syncthreads();
  for (int k = tid; k < m; k += blockDim.x) replica[__ldcg(order + k)] = sdest[k];
}

}  // namespace mori
