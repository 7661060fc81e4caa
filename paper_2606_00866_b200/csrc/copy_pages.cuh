// copy_pages.cuh -- steps a5/a6: move whole KV pages between the paged device pool and a
// page-major linear buffer (device staging, or the mapped pinned host arena).  sm_100a.
//
//   pool    [L][P][chunk]    address of (layer l, page g)  = pool + (l*P + g) * chunk
//   linear  [*][L][chunk]    address of (entry e, layer l) = lin  + (e*L + l) * chunk
//   GATHER : lin(e_k, l) <- pool(l, g_k)        SCATTER : pool(l, g_k) <- lin(e_k, l)
//   with g_k = gpu_pages[k] and e_k = lin_idx ? lin_idx[k] : k, for k in [0, n_pages).
// (include/mori.h: mori_demote / mori_promote / mori_gather_pages / mori_scatter_pages;
//  offload to CPU DRAM and reload over PCIe.)
//
// Pure data movement: the bound is HBM (device staging) or the host link (mapped arena), so the
// design goal is bytes in flight, not arithmetic.  Work is cut into "pieces": a contiguous run
// of <= piece_bytes inside one chunk, contiguous on BOTH sides (the bulk-copy kernel uses whole
// 64 KiB chunks as pieces; the LD/ST kernel 16 KiB).
//
// Three implementations:
//   copy_pages_tma   two threads per CTA drive the SM's bulk-copy engine: a loader issues
//                    cp.async.bulk global->shared (mbarrier complete_tx) into a ring of stages
//                    and publishes each stage's destination; a storer issues cp.async.bulk
//                    shared->global (bulk_group) and hands stages back.  No registers, no LSU
//                    instructions per byte; the rings of the CTAs resident on an SM take up to
//                    192 KiB.  Chunks are handed out dynamically (one atomic per chunk, fetched
//                    one chunk ahead) so that no SM idles while a slower one finishes a static
//                    share; one page-table load per chunk.
//   copy_pages_ldst  256 threads, 4 x 16-byte ld.global.nc.L1::no_allocate per thread issued
//                    before the 4 st.global: 16 KiB in flight per CTA, 8 CTAs per SM; piece w
//                    maps to (k, l, c) = (w / (L*ppc), (w / ppc) % L, w % ppc).
//   copy_pages_small the LD/ST body with the page / slot ids passed BY VALUE in the kernel
//                    parameters: a move of a few pages (cfg 1: KiBs per epoch) is one launch --
//                    no index upload, no staging, no DMA -- straight to / from the mapped arena.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mori {

struct CopyArgs {
  unsigned char* pool;
  unsigned char* lin;
  const int32_t* gpu_pages;   // [n_pages] device
  const int32_t* lin_idx;     // [n_pages] device, or nullptr for identity
  long long n_pages;
  long long pool_pages;       // P
  int n_layers;               // L
  int chunk_bytes;            // multiple of 16
  int piece_bytes;            // multiple of 16, <= chunk_bytes
  int pieces_per_chunk;       // ceil(chunk / piece)
  int stages;                 // bulk-copy kernel: ring depth (2 .. 24)
  int store_lag;              // bulk-copy kernel: 1 or 2 (< stages)
  unsigned int* sched;        // bulk-copy kernel: [2] zeroed words (next chunk, CTAs done) for dynamic
                              // chunk hand-out, or nullptr: CTA b takes chunks b, b + grid, ...
};

template <bool kGather>
__device__ __forceinline__ void piece_addresses(const CopyArgs& a, long long w, const unsigned char*& src,
                                                unsigned char*& dst, int& bytes) {
  const int ppc = a.pieces_per_chunk;
  const long long per_page = (long long)a.n_layers * ppc;
  const long long k = w / per_page;
  const int rem = (int)(w - k * per_page);
  const int l = rem / ppc, c = rem - l * ppc;
  const long long g = a.gpu_pages[k];
  const long long e = a.lin_idx ? (long long)a.lin_idx[k] : k;
  const long long off = (long long)c * a.piece_bytes;
  bytes = min(a.piece_bytes, a.chunk_bytes - (int)off);
  unsigned char* pp = a.pool + ((long long)l * a.pool_pages + g) * a.chunk_bytes + off;
  unsigned char* lp = a.lin + (e * a.n_layers + l) * a.chunk_bytes + off;
  if (kGather) { src = pp; dst = lp; } else { src = lp; dst = pp; }
}

// ------------------------------------------------------------------------------------------
// LD/ST implementation
// ------------------------------------------------------------------------------------------
constexpr int kLdstThreads = 256;
constexpr int kLdstUnroll = 4;   // 256 thr * 4 * 16 B = 16 KiB per CTA iteration

__device__ __forceinline__ int4 ld_stream(const int4* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(int4* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

template <bool kGather>
__global__ void __launch_bounds__(kLdstThreads) copy_pages_ldst(const CopyArgs a) {
  const long long n_pieces = a.n_pages * a.n_layers * a.pieces_per_chunk;
  for (long long w = blockIdx.x; w < n_pieces; w += gridDim.x) {
    const unsigned char* src; unsigned char* dst; int bytes;
    piece_addresses<kGather>(a, w, src, dst, bytes);
    const int4* s = reinterpret_cast<const int4*>(src);
    int4* d = reinterpret_cast<int4*>(dst);
    const int n_vec = bytes >> 4;
    for (int v0 = 0; v0 < n_vec; v0 += kLdstThreads * kLdstUnroll) {
      int4 r[kLdstUnroll];
#pragma unroll
      for (int u = 0; u < kLdstUnroll; ++u) {
        const int v = v0 + u * kLdstThreads + threadIdx.x;
        if (v < n_vec) r[u] = ld_stream(s + v);
      }
#pragma unroll
      for (int u = 0; u < kLdstUnroll; ++u) {
        const int v = v0 + u * kLdstThreads + threadIdx.x;
        if (v < n_vec) st_stream(d + v, r[u]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// TMA (1-D bulk copy) implementation
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
               :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
// Every byte is touched exactly once, so both halves of a copy carry an L2 evict-first hint: it
// keeps the stream from displacing what else lives in the 126 MB L2 and measures 1.5-2.5 % faster
// next to the copy engines' DMA traffic.
__device__ __forceinline__ uint64_t l2_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
      :: "r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(l2_evict_first()) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               :: "l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes), "l"(l2_evict_first()) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int kPending>
__device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(kPending) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}

constexpr int kTmaThreads = 64;   // warp 0 lane 0 = load issuer, warp 1 lane 0 = store issuer

// Addresses of chunk w = (page k, layer l): one page-table load and one division per CHUNK;
// the pieces of a chunk are consecutive on both sides.
template <bool kGather>
__device__ __forceinline__ void chunk_addresses(const CopyArgs& a, long long w, const unsigned char*& src,
                                                unsigned char*& dst) {
  const long long k = w / a.n_layers;
  const int l = (int)(w - k * a.n_layers);
  const long long g = a.gpu_pages[k];
  const long long e = a.lin_idx ? (long long)a.lin_idx[k] : k;
  unsigned char* pp = a.pool + ((long long)l * a.pool_pages + g) * a.chunk_bytes;
  unsigned char* lp = a.lin + (e * a.n_layers + l) * a.chunk_bytes;
  if (kGather) { src = pp; dst = lp; } else { src = lp; dst = pp; }
}

// Shared memory: a.stages stage buffers of a.piece_bytes each, then a.stages "full" and a.stages
// "empty" mbarriers, then per stage the destination address and byte count the loader publishes.
// Two single-thread roles so that neither waits for the other's latency:
//   loader  (warp 0): takes the next chunk (statically b, b + grid, ..., or dynamically from
//                     a.sched, fetched one chunk ahead so the atomic's latency is hidden); for
//                     every piece: wait until its stage is empty, publish (dst, bytes),
//                     expect_tx + bulk load.  After the last piece it publishes bytes = 0.
//   storer  (warp 1): wait until the stage is full, bulk store to the published address, commit;
//                     once the store issued `lag` groups ago has finished READING shared memory,
//                     hand its stage back to the loader (lag = 2 on a deep ring, 1 on a ring of a
//                     few large stages).  Stops at the bytes = 0 stage.
// Stage index and mbarrier phase are carried incrementally (no division per piece).
template <bool kGather>
__global__ void __launch_bounds__(kTmaThreads) copy_pages_tma(const CopyArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int stages = a.stages;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)stages * a.piece_bytes);
  uint64_t* empty = full + stages;
  unsigned char** st_dst = reinterpret_cast<unsigned char**>(empty + stages);
  uint32_t* st_bytes = reinterpret_cast<uint32_t*>(st_dst + stages);
  if (threadIdx.x == 0) {
    for (int s = 0; s < stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if ((threadIdx.x & 31) != 0) return;

  if (threadIdx.x == 0) {
    // ---------------- loader ----------------
    const long long n_chunks = a.n_pages * a.n_layers;
    const int ppc = a.pieces_per_chunk;
    unsigned int* sched = a.sched;
    int st = 0; uint32_t phase = 0; bool wrapped = false;          // phase of the NEXT wait on empty[st]
    long long w = blockIdx.x;
    long long w_next = sched ? (long long)gridDim.x + atomicAdd(&sched[0], 1u) : w + gridDim.x;
    while (w < n_chunks) {
      const unsigned char* src; unsigned char* dst;
      chunk_addresses<kGather>(a, w, src, dst);
      for (int c = 0; c < ppc; ++c) {
        const int off = c * a.piece_bytes;
        const uint32_t bytes = (uint32_t)min(a.piece_bytes, a.chunk_bytes - off);
        if (wrapped) mbar_wait(&empty[st], phase);
        st_dst[st] = dst + off;
        st_bytes[st] = bytes;
        mbar_expect_tx(&full[st], bytes);                           // release: the storer sees (dst, bytes)
        bulk_g2s(smem + (size_t)st * a.piece_bytes, src + off, bytes, &full[st]);
        if (++st == stages) { st = 0; if (wrapped) phase ^= 1; wrapped = true; }
      }
      w = w_next;
      w_next = sched ? (long long)gridDim.x + atomicAdd(&sched[0], 1u) : w + gridDim.x;
    }
    if (wrapped) mbar_wait(&empty[st], phase);
    st_bytes[st] = 0;                                               // end marker for the storer
    mbar_arrive(&full[st]);
    // the last CTA to stop taking chunks re-arms the two words for the next launch that uses them
    if (sched && atomicAdd(&sched[1], 1u) == gridDim.x - 1) { sched[0] = 0; sched[1] = 0; }
  } else {
    // ---------------- storer ----------------
    const int lag = a.store_lag;
    int st = 0; uint32_t phase = 0;                                 // stage / phase of the piece being stored
    int rel = 0; long long issued = 0;                              // next stage to hand back
    for (;;) {
      mbar_wait(&full[st], phase);
      const uint32_t bytes = st_bytes[st];
      if (bytes == 0) break;
      bulk_s2g(st_dst[st], smem + (size_t)st * a.piece_bytes, bytes);
      bulk_commit();
      if (++st == stages) { st = 0; phase ^= 1; }
      if (++issued > lag) {                                         // the group issued `lag` ago has left smem
        if (lag == 1) bulk_wait_read<1>(); else bulk_wait_read<2>();
        mbar_arrive(&empty[rel]);
        if (++rel == stages) rel = 0;
      }
    }
    bulk_wait_all();   // writes complete before the CTA exits
  }
}

// Shared-memory bytes of one copy_pages_tma CTA.
__host__ __device__ inline size_t tma_smem_bytes(int stages, int piece_bytes) {
  return (size_t)stages * piece_bytes + (size_t)stages * (2 * sizeof(uint64_t) + sizeof(void*) + sizeof(uint32_t));
}

// ------------------------------------------------------------------------------------------
// Small moves: ids by value in the kernel parameters (no index upload), 4 KiB pieces so that even
// a few pages spread over many SMs (the move is latency-bound: what matters is requests in
// flight on the link, not per-SM efficiency).
// ------------------------------------------------------------------------------------------
constexpr int kSmallMaxPages = 448;                                 // 3.5 KiB of ids: the 4 KiB parameter space
constexpr int kSmallFewPages = 64;                                  // a shorter parameter block launches faster
constexpr int kSmallPiece = kLdstThreads * 16;
template <int kCap> struct SmallIds { int32_t gpu[kCap]; int32_t lin[kCap]; };

template <bool kGather, int kCap>
__global__ void __launch_bounds__(kLdstThreads) copy_pages_small(const CopyArgs a, const SmallIds<kCap> ids) {
  const int ppc = a.pieces_per_chunk;                               // pieces of kSmallPiece bytes
  const int per_page = a.n_layers * ppc;
  const int n_pieces = (int)a.n_pages * per_page;
  for (int w = blockIdx.x; w < n_pieces; w += gridDim.x) {
    const int k = w / per_page, rem = w - k * per_page;
    const int l = rem / ppc, c = rem - l * ppc;
    const int off = c * kSmallPiece;
    const unsigned char* pp = a.pool + ((long long)l * a.pool_pages + ids.gpu[k]) * a.chunk_bytes + off;
    const unsigned char* lp = a.lin + ((long long)ids.lin[k] * a.n_layers + l) * a.chunk_bytes + off;
    const int v = threadIdx.x;
    if (v * 16 < a.chunk_bytes - off) {
      const int4* s = reinterpret_cast<const int4*>(kGather ? pp : lp) + v;
      int4* d = reinterpret_cast<int4*>(const_cast<unsigned char*>(kGather ? lp : pp)) + v;
      st_stream(d, ld_stream(s));
    }
  }
}

}  // namespace mori
