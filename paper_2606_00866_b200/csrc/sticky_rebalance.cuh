// sticky_rebalance.cuh -- NEXT-1: the paper's sticky, status-aware tier management (section
// 4.3.1) in ONE launch (sm_100a).  Declared in include/mori.h (mori_sticky_rebalance).
//
//   Demotion from GPU: only while the GPU queue exceeds its capacity; victims are Acting
//     programs before Reasoning ones, the most idle first; Reasoning victims are flagged lazy;
//     each victim goes to the CPU queue if it fits there, else to Waiting.
//   Promotion to GPU: while it fits, in priority order (1) CPU-queue programs waiting
//     for inference, (2) returning Waiting-queue programs, (3) new arrivals smallest context
//     first; the least idle first inside a class.
//   Everything else stays where it is.
//
// The paper's one-victim-at-a-time / one-candidate-at-a-time loops become one ordering and two
// prefix cuts.  Every program gets a unique 128-bit key (group, status | size, idleness, index)
// that sorts victims first (in victim order), then the promotion candidates (in priority order),
// then everybody else.  Positions come from ranking by counting on every SM (keys in shared
// memory, one warp per program); the last CTA to finish (atomic ticket) cuts the victim prefix
// ("usage minus what the earlier victims free still exceeds the capacity" is monotone) and the
// candidate prefix ("inclusive size sum fits the free capacity" is monotone) with block scans.
// The only sequential step is the paper's per-victim "CPU if it fits, else Waiting": skipped when
// all of them fit, else walked by one warp, 32 victims per round (the room only shrinks).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "rank_partition.cuh"

namespace mori {

constexpr int kFlagActing = 1, kFlagReady = 2, kFlagNew = 4;

// group: 0 GPU-queue program (victim order), 1..3 promotion classes, 7 not a candidate
__device__ __forceinline__ int sticky_group(int prev, int fl) {
  if (prev == 0) return 0;
  if (!(fl & kFlagReady)) return 7;
  if (prev == 1) return 1;
  return (fl & kFlagNew) ? 3 : 2;
}

__device__ __forceinline__ void sticky_key(int p, float iota, int s, int prev, int fl, unsigned long long& hi,
                                           unsigned long long& lo) {
  const uint32_t ik = idleness_key(iota);
  const int g = sticky_group(prev, fl);
  if (g == 0) {                       // Acting first, then most idle first (later in the total order)
    hi = (uint64_t)((fl & kFlagActing) ? 0 : 1) << 32;
    lo = ((uint64_t)(~ik) << 32) | (uint32_t)(~(uint32_t)p);
  } else {                            // least idle first; class 3: smallest context first
    hi = ((uint64_t)g << 33) | (g == 3 ? (uint32_t)(s > 0 ? s : 0) : 0u);
    lo = ((uint64_t)ik << 32) | (uint32_t)p;
  }
}

template <int IPT>
__global__ void __launch_bounds__(kRankMaxThreads, 1)
sticky_rebalance_kernel(int n, const float* __restrict__ idleness, const int32_t* __restrict__ kv_pages,
                        const uint8_t* __restrict__ prev_tier, const uint8_t* __restrict__ flags,
                        long long cap_gpu, long long cap_cpu, uint8_t* __restrict__ tier,
                        uint8_t* __restrict__ lazy, long long* __restrict__ used,
                        int32_t* __restrict__ lists, int32_t* __restrict__ list_counts,
                        int32_t* __restrict__ order, unsigned int* __restrict__ ticket) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ulonglong2* keys = reinterpret_cast<ulonglong2*>(smem_raw);        // [n] (x = low half, y = high half)
  uint64_t* warp_tot = reinterpret_cast<uint64_t*>(keys + n);        // [3][33]
  long long* bcast = reinterpret_cast<long long*>(warp_tot + 99);    // [4]
  // the per-program inputs, kept for the last CTA's tail: there they are read in RANK order, which
  // from global memory is a scattered gather (one transaction per program) and from here is free
  int32_t* s_kv = reinterpret_cast<int32_t*>(bcast + 4);             // [n]
  uint8_t* s_prev = reinterpret_cast<uint8_t*>(s_kv + n);            // [n]
  uint8_t* s_fl = s_prev + n;                                        // [n]
  const int tid = threadIdx.x;

  for (int p = tid; p < n; p += blockDim.x) {
    const int pv = prev_tier[p], kvp = kv_pages[p], flg = flags[p];
    s_kv[p] = kvp; s_prev[p] = (uint8_t)pv; s_fl[p] = (uint8_t)flg;
    unsigned long long hi64, lo64;
    sticky_key(p, idleness[p], kvp, pv == 0 ? 0 : (pv == 1 ? 1 : 2), flg, hi64, lo64);
    keys[p] = make_ulonglong2(lo64, hi64);
  }
  __syncthreads();
  // ---- position of every program = number of smaller 128-bit keys; the last CTA goes on ---------
  if (!rank_by_counting128(n, keys, order, ticket)) return;

  // ---- this thread's positions ------------------------------------------------------------------
  int32_t* vsize = reinterpret_cast<int32_t*>(keys);                 // [n] victims' sizes, by position
  uint8_t* vdest = reinterpret_cast<uint8_t*>(vsize + n);            // [n] 1 = CPU queue, 2 = Waiting
  uint8_t* s_tier = vdest + n;                                       // [n] per-PROGRAM outputs, staged (flush_bytes)
  uint8_t* s_lazy = s_tier + n;                                      // [n]
  int prog[IPT], grp[IPT], was[IPT], fl[IPT];
  long long sz[IPT];
  long long sum_g = 0, sum_c = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    const int r = tid * IPT + i;
    prog[i] = -1; grp[i] = 7; was[i] = 2; fl[i] = 0; sz[i] = 0;
    if (r < n) {
      const int p = __ldcg(order + r);
      const int pv = s_prev[p];
      prog[i] = p;
      was[i] = pv == 0 ? 0 : (pv == 1 ? 1 : 2);
      fl[i] = s_fl[p];
      grp[i] = sticky_group(was[i], fl[i]);
      const int s = s_kv[p];
      sz[i] = s > 0 ? s : 0;
      if (was[i] == 0) sum_g += sz[i];
      if (was[i] == 1) sum_c += sz[i];
    }
  }
  __syncthreads();                                                   // keys are dead: smem is reused below

  // ---- demotion: victims = the prefix of group 0 whose predecessors do not free enough ----------
  uint64_t tot;
  uint64_t sc2[2] = {(uint64_t)sum_g, (uint64_t)sum_c}, tt2[2];
  block_excl_scan_n<2>(sc2, warp_tot, tt2);                          // one set of barriers for both sums
  long long run = (long long)sc2[0];                                 // freed BEFORE this thread
  const long long usage_gpu0 = (long long)tt2[0], usage_cpu0 = (long long)tt2[1];
  bool victim[IPT];
  int n_v = 0;
  long long freed_mine = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    victim[i] = grp[i] == 0 && usage_gpu0 - run > cap_gpu;           // group 0 sits at positions [0, nG)
    if (grp[i] == 0) run += sz[i];
    if (victim[i]) {
      ++n_v; freed_mine += sz[i];
      vsize[tid * IPT + i] = (int32_t)sz[i];
    }
  }
  uint64_t vf2[2] = {(uint64_t)n_v, (uint64_t)freed_mine};
  block_excl_scan_n<2>(vf2, warp_tot, tt2);
  const int v = (int)tt2[0];                                         // victims are positions [0, v)
  const long long freed = (long long)tt2[1];

  // ---- each victim: CPU queue if it fits, else Waiting, in victim order -----------------
  if (usage_cpu0 + freed <= cap_cpu) {                               // all of them fit
#pragma unroll
    for (int i = 0; i < IPT; ++i) if (victim[i]) vdest[tid * IPT + i] = 1;
    if (tid == 0) bcast[0] = usage_cpu0 + freed;
  } else if (tid < 32) {
    // The paper's walk is sequential ("each victim, in that order, goes to the CPU queue if it
    // still fits"), but the room only ever shrinks, which one warp exploits 32 victims at a time:
    //   (1) a victim larger than the room that is left can never fit -> Waiting, whatever precedes it;
    //   (2) of the others, in order, the longest prefix whose summed size fits is taken at once;
    //   (3) the one right after that prefix is then larger than the new room -> step (1) again.
    // Every round decides at least one victim of the chunk and usually all 32.
    const int lane = tid;
    long long room = cap_cpu - usage_cpu0;
    for (int k0 = 0; k0 < v; k0 += 32) {
      const int k = k0 + lane;
      const long long s = k < v ? (long long)vsize[k] : 0;
      unsigned undecided = __ballot_sync(0xFFFFFFFFu, k < v);
      int dest = 0;
      while (undecided) {
        const bool mine = (undecided >> lane) & 1u;
        const unsigned miss = __ballot_sync(0xFFFFFFFFu, mine && s > room);
        if ((miss >> lane) & 1u) dest = 2;
        undecided &= ~miss;
        if (!undecided) break;
        const bool still = (undecided >> lane) & 1u;
        long long incl = still ? s : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const long long o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
          if (lane >= d) incl += o;
        }
        const unsigned fit = __ballot_sync(0xFFFFFFFFu, still && incl <= room);   // a prefix of the undecided ones
        if ((fit >> lane) & 1u) dest = 1;
        const long long taken = __shfl_sync(0xFFFFFFFFu, incl, fit ? 31 - __clz(fit) : 0);
        room -= fit ? taken : 0;
        undecided &= ~fit;
      }
      if (k < v) vdest[k] = (uint8_t)dest;
    }
    if (lane == 0) bcast[0] = cap_cpu - room;
  }
  __syncthreads();
  const long long usage_cpu1 = bcast[0];

  // ---- promotion: the longest prefix of the candidates (positions [nG, nG + nC)) that fits -------
  const long long free_gpu = cap_gpu - (usage_gpu0 - freed);
  long long cand_mine = 0;
#pragma unroll
  for (int i = 0; i < IPT; ++i) if (grp[i] >= 1 && grp[i] <= 3) cand_mine += sz[i];
  long long crun = (long long)block_excl_scan((uint64_t)cand_mine, warp_tot, &tot);
  bool promoted[IPT];
  long long up_g = 0, down_c = 0;
  uint64_t packed = 0;                                               // 16-bit counters: demote | promote | drop | admit
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    promoted[i] = false;
    if (grp[i] >= 1 && grp[i] <= 3) {
      crun += sz[i];
      promoted[i] = crun <= free_gpu;
      if (promoted[i]) {
        up_g += sz[i];
        if (was[i] == 1) { down_c += sz[i]; packed += 1ull << 16; } else packed += 1ull << 48;
      }
    }
    if (victim[i]) packed += vdest[tid * IPT + i] == 1 ? 1ull : (1ull << 32);
  }
  uint64_t pud[3] = {packed, (uint64_t)up_g, (uint64_t)down_c}, tt3[3];
  block_excl_scan_n<3>(pud, warp_tot, tt3);
  uint64_t pex = pud[0];
  const uint64_t ptot = tt3[0];
  const long long promoted_pages = (long long)tt3[1];
  const long long promoted_from_cpu = (long long)tt3[2];

  // ---- outputs ----------------------------------------------------------------------------------
#pragma unroll
  for (int i = 0; i < IPT; ++i) {
    if (prog[i] < 0) continue;
    int now = was[i], row = -1;
    if (victim[i]) { now = vdest[tid * IPT + i]; row = now == 1 ? 0 : 2; }
    else if (promoted[i]) { now = 0; row = was[i] == 1 ? 1 : 3; }
    s_tier[prog[i]] = (uint8_t)now;
    s_lazy[prog[i]] = (uint8_t)(victim[i] && !(fl[i] & kFlagActing));
    if (row >= 0) {
      const int pos = (int)((pex >> (16 * row)) & 0xFFFF);
      pex += 1ull << (16 * row);
      lists[(size_t)row * n + pos] = prog[i];
    }
  }
  flush_bytes(s_tier, tier, n);
  flush_bytes(s_lazy, lazy, n);
  if (tid < 4) list_counts[tid] = (int)((ptot >> (16 * tid)) & 0xFFFF);
  if (tid == 4) list_counts[4] = 0;
  if (tid == 0) {
    used[0] = usage_gpu0 - freed + promoted_pages;
    used[1] = usage_cpu1 - promoted_from_cpu;
  }
}

}  // namespace mori
