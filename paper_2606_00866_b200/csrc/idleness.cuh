// idleness.cuh -- NEXT-2: the windowed idleness metric of Eq. (1) kept and evaluated
// on the device, so that iota goes straight into the rankers with no per-tick host computation.
// Declared in include/mori.h (mori_idleness_update / mori_idleness_eval).
//
//   iota = T_acting^(k) / (T_reasoning^(k) + T_acting^(k)) over the last k cycles, the unfinished
//   cycle included with its elapsed time, gated time never reported.
//
// State (library-owned, per program): a ring of the last k completed (reasoning, acting) pairs
// and the number of cycles pushed since the slot was reset.  Arithmetic is fixed so that the
// result is reproducible bit for bit: double sums, oldest cycle first, the open cycle last, one
// IEEE division, one rounding to float (explicit __dadd_rn / __ddiv_rn: no contraction).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mori {

constexpr int kIdlenessThreads = 256;
constexpr int kIdlenessTile = 1024;   // events staged in shared memory per pass

// One thread per program applies that program's events in list order; programs are independent.
// The event list is staged in shared memory and scanned by whole warps, 32 events per ballot.
__global__ void __launch_bounds__(kIdlenessThreads)
idleness_update_kernel(int n, int k, double* __restrict__ ring_r, double* __restrict__ ring_a,
                       int32_t* __restrict__ pushed, long long m, const int32_t* __restrict__ prog,
                       const uint8_t* __restrict__ kind, const double* __restrict__ reasoning,
                       const double* __restrict__ acting) {
  __shared__ int32_t s_prog[kIdlenessTile];
  __shared__ uint8_t s_kind[kIdlenessTile];
  const int p = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
  int cnt = p < n ? pushed[p] : 0;
  for (long long base = 0; base < m; base += kIdlenessTile) {
    const int len = (int)min((long long)kIdlenessTile, m - base);
    __syncthreads();
    for (int i = threadIdx.x; i < len; i += blockDim.x) { s_prog[i] = prog[base + i]; s_kind[i] = kind[base + i]; }
    __syncthreads();
    // 32 events at a time: one ballot tells the warp which of them belong to its 32 programs,
    // and only those are visited (in list order), so a thread does m/32 + (its own events) steps
    const int wp0 = p - lane;
    for (int i0 = 0; i0 < len; i0 += 32) {
      const int ep = i0 + lane < len ? s_prog[i0 + lane] : -1;
      unsigned hit = __ballot_sync(0xFFFFFFFFu, ep >= wp0 && ep < wp0 + 32);
      while (hit) {
        const int i = i0 + __ffs(hit) - 1;
        hit &= hit - 1;
        if (s_prog[i] != p || p >= n) continue;
        if (s_kind[i] == 1) { cnt = 0; continue; }               // slot taken by a fresh program
        const int slot = cnt % k;                                 // overwrites the oldest when full
        ring_r[(size_t)p * k + slot] = reasoning[base + i];
        ring_a[(size_t)p * k + slot] = acting[base + i];
        ++cnt;
      }
    }
  }
  if (p < n) pushed[p] = cnt;
}

__global__ void __launch_bounds__(kIdlenessThreads)
idleness_eval_kernel(int n, int k, const double* __restrict__ ring_r, const double* __restrict__ ring_a,
                     const int32_t* __restrict__ pushed, const double* __restrict__ open_r,
                     const double* __restrict__ open_a, float* __restrict__ iota) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const double o_r = open_r ? open_r[p] : 0.0, o_a = open_a ? open_a[p] : 0.0;
  const bool open = __dadd_rn(o_r, o_a) > 0.0;
  const int cnt = pushed[p];
  const int stored = min(cnt, k);
  const int take = min(open ? k - 1 : k, stored);                 // the open cycle is one of the k
  double tr = 0.0, ta = 0.0;
  for (int i = stored - take; i < stored; ++i) {                  // chronological: oldest first
    const int slot = (cnt - stored + i) % k;
    tr = __dadd_rn(tr, ring_r[(size_t)p * k + slot]);
    ta = __dadd_rn(ta, ring_a[(size_t)p * k + slot]);
  }
  if (open) { tr = __dadd_rn(tr, o_r); ta = __dadd_rn(ta, o_a); }
  const double den = __dadd_rn(tr, ta);
  iota[p] = den == 0.0 ? __int_as_float(0x7FC00000) : __double2float_rn(__ddiv_rn(ta, den));
}

}  // namespace mori
