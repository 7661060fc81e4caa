// mori.cu -- libmori.so: context, streams, staging and the C ABI of include/mori.h.
// Every step of the hot path runs in the kernels of rank_partition.cuh / copy_pages.cuh or on
// the GPU's copy engines; the host code here only marshals arguments and orders streams.
#include "../../include/mori.h"

#include <cuda_runtime.h>

#include <sys/mman.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <mutex>
#include <thread>
#include <utility>
#include <cstring>
#include <string>
#include <vector>

#include "copy_pages.cuh"
#include "rank_partition.cuh"
#include "sticky_rebalance.cuh"
#include "idleness.cuh"
#include "eviction_order.cuh"
#include "bfd_assign.cuh"

namespace {

thread_local std::string g_create_error;
std::mutex g_host_mu;
std::map<void*, std::pair<void*, size_t>> g_host_allocs;   // mori_host_alloc: aligned ptr -> (mmap base, length)

constexpr int kTicketRing = 4096;
// Last-CTA tickets of the rankers and chunk counters of the copy kernel: one entry per launch,
// taken round-robin and re-armed by the launch's own last CTA.  An entry is in use only while its
// kernel is RESIDENT, and a device runs at most 128 grids at once, so 256 entries cannot collide.
constexpr int kRankTickets = 256;
constexpr int kSchedRing = 256;
constexpr int kPieceBytesDefault = 64 * 1024;   // bytes per bulk copy = stage size (whole 64 KiB chunks)
constexpr int kRingBytesDefault = 192 * 1024;   // shared memory the rings of one SM's CTAs may take
constexpr int kMaxTmaStages = 24;
constexpr long long kAutoMinRunBytes = 6LL << 20;   // AUTO: below this mean slot-run length, ZEROCOPY
constexpr long long kRampBytes = 512LL << 20;        // STAGED: size of a call's first (demote) / last (promote) segment
constexpr long long kSmallMaxBytes = 4LL << 20;     // calls up to this size (and kSmallMaxPages) take the one-launch path

// Tuning overrides for experiments (read once per mori_create): MORI_PIECE_KIB, MORI_RING_KIB,
// MORI_CTAS_PER_SM, MORI_SCHED (0 static, 1 dynamic), MORI_STAGING_MIB, MORI_EVICT_MULTI (1: the
// general multi-kernel eviction sort at every size).  Unset = the defaults.
long long env_ll(const char* name, long long dflt) {
  const char* v = std::getenv(name);
  if (!v || !*v) return dflt;
  char* end = nullptr;
  const long long x = std::strtoll(v, &end, 10);
  return end && *end == 0 ? x : dflt;
}

struct ProfSpan { cudaEvent_t a, b; long long bytes; int kind; };   // kind 0: gather/scatter/zero-copy kernel, 1: DMA segment
struct TimelineRow { int kind; double t0_ms, t1_ms; long long bytes; };

struct Direction {
  int path = 0;
  bool auto_path = false;                        // AUTO: STAGED or ZEROCOPY per call, by slot-run length
  cudaStream_t kern = nullptr, copy = nullptr;   // kernel stream, DMA stream (STAGED only)
  unsigned char* staging[2] = {nullptr, nullptr};
  cudaEvent_t kern_done[2] = {nullptr, nullptr}, copy_done[2] = {nullptr, nullptr};
  int buf = 0;
  bool copy_busy = false;                        // DMAs enqueued on `copy` since the last join
  bool kern_busy = false;                        // anything enqueued on `kern` since the last join
  // index ring: pinned host (written by the CPU, read by the upload kernel) + device copy
  int32_t* idx_host = nullptr; int32_t* idx_host_dev = nullptr; int32_t* idx_dev = nullptr;
  long long idx_cap = 0, idx_used = 0;
  std::vector<cudaEvent_t> tickets;              // ring
  long long next_ticket = 1;
  std::vector<ProfSpan> spans;
  std::vector<TimelineRow> timeline;            // mori_profile(ctx, 2): every span, on one clock
  double prof_ms = 0; long long prof_launches = 0, prof_bytes = 0;
};

}  // namespace

struct mori_ctx {
  mori_config cfg;
  int device = 0, sm_count = 148;
  long long chunk = 0, page_bytes = 0, staging_bytes = 0, max_pages = 0;
  int copy_kernel = MORI_KERNEL_TMA;
  int piece = kPieceBytesDefault, ppc = 1, tma_stages = 3, tma_lag = 1, ctas_per_sm = 1;
  int link_ctas = 32;
  size_t tma_smem = 0;
  unsigned int* sched = nullptr;                 // [kSchedRing][2] chunk counters of the copy kernel (nullptr: static)
  mutable unsigned long long sched_seq = 0;
  bool debug = false;                            // MORI_DEBUG=1: duplicate-id validation
  std::vector<uint8_t> dbg_seen;                 // scratch bitmap of the host-side duplicate check
  int* dbg_flag = nullptr; unsigned int* dbg_bitmap = nullptr;   // device-side check of gather/scatter ids
  int* dbg_flag_host = nullptr;
  unsigned char* arena_dev = nullptr;            // device-side alias of the pinned arena
  bool arena_is_device = false;                  // arena lives in (this or a peer GPU's) HBM
  unsigned int* rank_tickets = nullptr;          // [kRankTickets] last-CTA counters of the multi-CTA ranker
  unsigned long long rank_seq = 0;
  int idl_k = 5;                                 // window of Eq. (1)
  double* idl_r = nullptr; double* idl_a = nullptr; int32_t* idl_pushed = nullptr;   // [max_programs][k], [max_programs]
  // the sequence of mori_eviction_order, captured once per (tier, argument set) and replayed
  cudaGraphExec_t evict_exec[2] = {nullptr, nullptr}; cudaStream_t evict_cap_stream = nullptr;
  struct EvictKey { int n_programs; long long n_pages; const void *owner, *ptier, *last; void *victims, *nres; } evict_key[2]{};
  unsigned int* evict_max_last = nullptr;
  int32_t* evict_perm[2] = {nullptr, nullptr}; int32_t* evict_table = nullptr; long long evict_cap = 0;   // scratch, grown on demand
  bool evict_multi_kernel = false;               // MORI_EVICT_MULTI=1: force the general (multi-kernel) sort
  int evict_cluster_want = 16;
  int evict_cluster = 8;                         // CTAs of the one-launch eviction sort's cluster (8, or 16 where allowed)
  int32_t* sticky_order = nullptr;               // [kRankTickets][max_programs] positions scratch
  Direction dir[2];                              // 0 demote, 1 promote
  std::vector<cudaEvent_t> free_events;
  // mori_after_stream is lazy: the caller-stream event is kept here and each of the four library
  // streams waits on it only when it next gets work (an epoch that only demotes a few pages never
  // touches the promote streams or the DMA streams).  streams_left: bit 2*dir = kernel stream,
  // bit 2*dir+1 = DMA stream.  Entries whose event has completed are dropped at mori_sync.
  struct PendingAfter { cudaEvent_t ev; int streams_left; };
  std::vector<PendingAfter> pending_after;
  std::vector<cudaEvent_t> free_timing_events;   // profiling spans reuse their events (creating one costs microseconds)
  bool profiling = false;
  bool timeline = false; cudaEvent_t prof_base = nullptr;   // mori_profile(ctx, 2)
  mutable long long launches = 0;                // kernels launched by this context
  int sticky = MORI_OK;
  mutable std::string err;
};

namespace {

int fail(const mori_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}

#define CK(ctx, call)                                                                         \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      if (ctx) (ctx)->sticky = MORI_ERR_CUDA;                                                 \
      return fail(ctx, MORI_ERR_CUDA,                                                         \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                        \
    }                                                                                         \
  } while (0)

__global__ void upload_idx_kernel(const int32_t* __restrict__ src, int32_t* __restrict__ dst, long long n) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x)
    dst[i] = src[i];
}

// MORI_DEBUG: range (and, for destinations, duplicate) check of a DEVICE id table.  flag: bit 0 =
// out of range, bit 1 = duplicate.  The bitmap is left clean (second pass clears what was set).
__global__ void validate_ids_kernel(const int32_t* __restrict__ ids, long long n, long long id_space,
                                    unsigned int* __restrict__ bitmap, int check_dup, int clear, int* flag) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int id = ids[i];
    if (id < 0 || id >= id_space) { if (!clear) atomicOr(flag, 1); continue; }
    if (!check_dup) continue;
    const unsigned int bit = 1u << (id & 31);
    if (clear) atomicAnd(&bitmap[id >> 5], ~bit);
    else if (atomicOr(&bitmap[id >> 5], bit) & bit) atomicOr(flag, 2);
  }
}

mori::CopyArgs make_args(const mori_ctx* c, unsigned char* lin, const int32_t* gpu_pages,
                         const int32_t* lin_idx, long long n_pages) {
  mori::CopyArgs a;
  a.pool = static_cast<unsigned char*>(c->cfg.gpu_pool);
  a.lin = lin;
  a.gpu_pages = gpu_pages;
  a.lin_idx = lin_idx;
  a.n_pages = n_pages;
  a.pool_pages = c->cfg.gpu_pool_pages;
  a.n_layers = c->cfg.n_layers;
  a.chunk_bytes = (int)c->chunk;
  a.piece_bytes = c->piece;
  a.pieces_per_chunk = c->ppc;
  a.stages = c->tma_stages;
  a.store_lag = c->tma_lag;
  a.sched = nullptr;
  return a;
}

// One launch of the page-copy kernel.  `link` = the linear side is host memory behind PCIe:
// a small grid saturates the link and leaves the SMs to everything else.
template <bool kGather>
cudaError_t launch_copy(const mori_ctx* c, const mori::CopyArgs& a, cudaStream_t s, bool link) {
  const long long n_pieces = a.n_pages * a.n_layers * a.pieces_per_chunk;
  if (n_pieces == 0) return cudaSuccess;
  c->launches += 1;
  if (c->copy_kernel == MORI_KERNEL_TMA) {
    const long long max_grid = link ? c->link_ctas : (long long)c->sm_count * c->ctas_per_sm;  // smem-bound residency
    const int grid = (int)std::min<long long>(a.n_pages * a.n_layers, max_grid);   // CTAs take whole chunks
    mori::CopyArgs b = a;
    if (c->sched && grid > 1) b.sched = c->sched + 2 * (c->sched_seq++ % kSchedRing);
    mori::copy_pages_tma<kGather><<<grid, mori::kTmaThreads, c->tma_smem, s>>>(b);
  } else {
    mori::CopyArgs b = a;                                        // LD/ST works in 16 KiB pieces
    b.piece_bytes = (int)std::min<long long>(16 * 1024, a.chunk_bytes);
    b.pieces_per_chunk = (a.chunk_bytes + b.piece_bytes - 1) / b.piece_bytes;
    const long long n_ldst = a.n_pages * a.n_layers * b.pieces_per_chunk;
    const long long max_grid = link ? 2 * c->link_ctas : (long long)c->sm_count * 8;
    const int grid = (int)std::min<long long>(n_ldst, max_grid);
    mori::copy_pages_ldst<kGather><<<grid, mori::kLdstThreads, 0, s>>>(b);
  }
  return cudaGetLastError();
}

// The one-launch path of a small move: ids by value in the kernel parameters, LD/ST straight
// between the pool and the (mapped or device) arena.
template <bool kGather, int kCap>
cudaError_t launch_small_cap(const mori_ctx* c, long long n, const int32_t* gpu_pages, const int32_t* host_slots,
                             cudaStream_t s) {
  mori::SmallIds<kCap> ids;
  std::memcpy(ids.gpu, gpu_pages, sizeof(int32_t) * n);
  std::memcpy(ids.lin, host_slots, sizeof(int32_t) * n);
  mori::CopyArgs a = make_args(c, c->arena_dev, nullptr, nullptr, n);
  a.pieces_per_chunk = (int)((c->chunk + mori::kSmallPiece - 1) / mori::kSmallPiece);
  const long long n_pieces = n * a.n_layers * a.pieces_per_chunk;
  const int grid = (int)std::min<long long>(n_pieces, (long long)c->sm_count * 4);
  c->launches += 1;
  mori::copy_pages_small<kGather, kCap><<<grid, mori::kLdstThreads, 0, s>>>(a, ids);
  return cudaGetLastError();
}
template <bool kGather>
cudaError_t launch_small(const mori_ctx* c, long long n, const int32_t* gpu_pages, const int32_t* host_slots,
                         cudaStream_t s) {
  return n <= mori::kSmallFewPages ? launch_small_cap<kGather, mori::kSmallFewPages>(c, n, gpu_pages, host_slots, s)
                                   : launch_small_cap<kGather, mori::kSmallMaxPages>(c, n, gpu_pages, host_slots, s);
}

// nullptr (and a latched MORI_ERR_CUDA) when the driver cannot create an event.
cudaEvent_t get_event(mori_ctx* c, bool timing) {
  cudaEvent_t e = nullptr;
  if (!timing && !c->free_events.empty()) { e = c->free_events.back(); c->free_events.pop_back(); return e; }
  if (timing && !c->free_timing_events.empty()) { e = c->free_timing_events.back(); c->free_timing_events.pop_back(); return e; }
  const cudaError_t rc = cudaEventCreateWithFlags(&e, timing ? cudaEventDefault : cudaEventDisableTiming);
  if (rc != cudaSuccess) {
    c->sticky = MORI_ERR_CUDA;
    c->err = std::string("cudaEventCreateWithFlags: ") + cudaGetErrorString(rc);
    return nullptr;
  }
  return e;
}

int check_ids(const mori_ctx* c, long long n, const int32_t* gpu_pages, const int32_t* host_slots) {
  for (long long j = 0; j < n; ++j) {
    if (gpu_pages[j] < 0 || gpu_pages[j] >= c->cfg.gpu_pool_pages)
      return fail(c, MORI_ERR_INVALID_ARG, "gpu page id out of range at index " + std::to_string(j));
    if (host_slots[j] < 0 || host_slots[j] >= c->cfg.host_arena_slots)
      return fail(c, MORI_ERR_INVALID_ARG, "host slot id out of range at index " + std::to_string(j));
  }
  return MORI_OK;
}

// MORI_DEBUG=1: a DESTINATION id listed twice in one call is undefined behaviour in release (two
// copies race for the same bytes); here it is found on the host before anything is enqueued.
int check_duplicates(mori_ctx* c, long long n, const int32_t* dst_ids, long long id_space, const char* what) {
  if ((long long)c->dbg_seen.size() < id_space) c->dbg_seen.assign((size_t)id_space, 0);
  int rc = MORI_OK;
  long long j = 0;
  for (; j < n; ++j) {
    if (c->dbg_seen[dst_ids[j]]) { rc = MORI_ERR_INVALID_ARG; break; }
    c->dbg_seen[dst_ids[j]] = 1;
  }
  const long long bad = j;
  for (long long i = 0; i < (rc ? bad : n); ++i) c->dbg_seen[dst_ids[i]] = 0;
  if (rc) return fail(c, rc, std::string("MORI_DEBUG: duplicate destination ") + what + " " +
                             std::to_string(dst_ids[bad]) + " at index " + std::to_string(bad));
  return MORI_OK;
}

// Copies the two index arrays into the direction's pinned ring and launches the upload kernel
// on the kernel stream.  Returns device pointers.
int stage_indices(mori_ctx* c, Direction& d, long long n, const int32_t* a0, const int32_t* a1,
                  const int32_t** d0, const int32_t** d1) {
  if (2 * n > d.idx_cap) return fail(c, MORI_ERR_CAPACITY, "more pages in one call than max_pages_per_call");
  if (d.idx_used + 2 * n > d.idx_cap) {           // ring full: drain this direction, start over
    CK(c, cudaStreamSynchronize(d.kern));
    if (d.copy) CK(c, cudaStreamSynchronize(d.copy));
    d.idx_used = 0;
  }
  int32_t* h = d.idx_host + d.idx_used;
  std::memcpy(h, a0, sizeof(int32_t) * n);
  std::memcpy(h + n, a1, sizeof(int32_t) * n);
  const int grid = (int)std::min<long long>((2 * n + 255) / 256, 64);
  upload_idx_kernel<<<grid, 256, 0, d.kern>>>(d.idx_host_dev + d.idx_used, d.idx_dev + d.idx_used, 2 * n);
  CK(c, cudaGetLastError());
  c->launches += 1;
  *d0 = d.idx_dev + d.idx_used;
  *d1 = d.idx_dev + d.idx_used + n;
  d.idx_used += 2 * n;
  return MORI_OK;
}

int wait_ticket(mori_ctx* c, Direction& other, long long ticket, cudaStream_t s) {
  if (ticket <= 0) return MORI_OK;
  if (ticket >= other.next_ticket) return fail(c, MORI_ERR_INVALID_ARG, "ticket was never issued");
  // a ticket older than the ring has been overwritten by a LATER event of the same stream:
  // waiting on that one is conservative and still correct.
  CK(c, cudaStreamWaitEvent(s, other.tickets[ticket % kTicketRing], 0));
  return MORI_OK;
}

int issue_ticket(mori_ctx* c, Direction& d, cudaStream_t s, int64_t* out) {
  if (!out) return MORI_OK;                       // nobody will wait on it: no event, no number
  const long long t = d.next_ticket++;
  CK(c, cudaEventRecord(d.tickets[t % kTicketRing], s));
  if (out) *out = t;
  return MORI_OK;
}

void prof_begin(mori_ctx* c, Direction& d, cudaStream_t s, long long bytes, int kind = 0) {
  if (!c->profiling || (kind != 0 && !c->timeline)) return;
  ProfSpan sp{get_event(c, true), get_event(c, true), bytes, kind};
  if (!sp.a || !sp.b) { if (sp.a) cudaEventDestroy(sp.a); if (sp.b) cudaEventDestroy(sp.b); sp.a = sp.b = nullptr; }
  if (sp.a) cudaEventRecord(sp.a, s);
  d.spans.push_back(sp);
}
void prof_end(mori_ctx* c, Direction& d, cudaStream_t s, int kind = 0) {
  if (!c->profiling || (kind != 0 && !c->timeline) || d.spans.empty() || !d.spans.back().b) return;
  cudaEventRecord(d.spans.back().b, s);
}
void prof_collect(mori_ctx* c, Direction& d) {
  for (auto& sp : d.spans) {
    float ms = 0;
    if (!sp.a) continue;
    if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) {
      if (sp.kind == 0) { d.prof_ms += ms; d.prof_launches += 1; d.prof_bytes += sp.bytes; }
      float t0 = 0;
      if (c && c->timeline && c->prof_base && cudaEventElapsedTime(&t0, c->prof_base, sp.a) == cudaSuccess)
        d.timeline.push_back({sp.kind, (double)t0, (double)t0 + ms, sp.bytes});
    }
    if (c) { c->free_timing_events.push_back(sp.a); c->free_timing_events.push_back(sp.b); }
    else { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  }
  cudaGetLastError();
  d.spans.clear();
}

template <int IPT>
cudaError_t launch_rank(int threads, size_t smem, cudaStream_t s, int n, int n_pad, const float* idl,
                        const int32_t* kv, const uint8_t* prev, long long cg, long long cc, int32_t* order,
                        uint8_t* tier, int32_t* bounds, long long* used, int32_t* lists, int32_t* counts) {
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(mori::rank_partition_kernel<IPT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  mori::rank_partition_kernel<IPT><<<1, threads, smem, s>>>(n, n_pad, idl, kv, prev, cg, cc, order, tier,
                                                            bounds, used, lists, counts);
  return cudaGetLastError();
}

template <int IPT>
cudaError_t launch_rank_multi(int grid, size_t smem, cudaStream_t s, int n, const float* idl, const int32_t* kv,
                              const uint8_t* prev, long long cg, long long cc, int32_t* order, uint8_t* tier,
                              int32_t* bounds, long long* used, int32_t* lists, int32_t* counts,
                              int32_t* scratch_order, unsigned int* ticket) {
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(mori::rank_partition_multi_kernel<IPT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  mori::rank_partition_multi_kernel<IPT><<<grid, mori::kRankMaxThreads, smem, s>>>(
      n, idl, kv, prev, cg, cc, order, tier, bounds, used, lists, counts, scratch_order, ticket);
  return cudaGetLastError();
}

template <int IPT>
cudaError_t launch_tiers(int grid, size_t smem, cudaStream_t s, int n, const float* idl, const int32_t* kv,
                         const mori::TierCaps& caps, const uint8_t* prev, int32_t* order, uint8_t* tier,
                         int32_t* bounds, long long* used, int32_t* moves, int32_t* move_counts,
                         int32_t* scratch_order, unsigned int* ticket) {
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(mori::rank_tiers_kernel<IPT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  mori::rank_tiers_kernel<IPT><<<grid, mori::kRankMaxThreads, smem, s>>>(n, idl, kv, caps, prev, order, tier, bounds,
                                                                        used, moves, move_counts, scratch_order, ticket);
  return cudaGetLastError();
}

template <int IPT>
cudaError_t launch_sticky(int grid, size_t smem, cudaStream_t s, int n, const float* idl, const int32_t* kv,
                                 const uint8_t* prev, const uint8_t* flags, long long cg, long long cc,
                                 uint8_t* tier, uint8_t* lazy, long long* used, int32_t* lists, int32_t* counts,
                                 int32_t* order, unsigned int* ticket) {
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(mori::sticky_rebalance_kernel<IPT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  mori::sticky_rebalance_kernel<IPT><<<grid, mori::kRankMaxThreads, smem, s>>>(
      n, idl, kv, prev, flags, cg, cc, tier, lazy, used, lists, counts, order, ticket);
  return cudaGetLastError();
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// mori_eviction_order_noalloc: the sort scratch of the one-launch eviction order as a file-scope
// array, so that the entry point never allocates.  2 buffers of MORI_NOALLOC_MAX_PAGES 64-bit
// items = 1 MiB, held by every GPU that loads the library until the process exits.  In HOST code
// this name is a stand-in, not a device address: the address comes from cudaGetSymbolAddress, once
// per device with that device current (noalloc_setup below).
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned long long g_noalloc_evict_scratch[2 * MORI_NOALLOC_MAX_PAGES];

namespace {
constexpr int kNoallocMaxDevices = 64;
struct NoallocDev { bool ready = false; unsigned long long* scratch = nullptr; int cluster = 8; };
NoallocDev g_noalloc_dev[kNoallocMaxDevices];
std::mutex g_noalloc_mu;

// Once per device, with that device current.  No allocation: a symbol lookup, a function attribute
// and an occupancy query.  -> static error string, or nullptr when the device is ready.
const char* noalloc_setup(int dev) {
  NoallocDev& d = g_noalloc_dev[dev];
  if (d.ready) return nullptr;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { cudaGetLastError(); return "cudaGetDeviceProperties failed"; }
  if (prop.major != 10) return "libmori is built for sm_100a (B200) only";
  unsigned long long* ptr = nullptr;
  if (cudaGetSymbolAddress((void**)&ptr, g_noalloc_evict_scratch) != cudaSuccess || ptr == nullptr) {
    cudaGetLastError();
    return "cudaGetSymbolAddress(g_noalloc_evict_scratch) failed";
  }
  // cluster of 16 CTAs where the device can co-schedule that non-portable size, else the portable 8
  bool ok = true;
  const void* ks[] = {(const void*)mori::evict_order_cluster_kernel<2>, (const void*)mori::evict_order_cluster_kernel<4>,
                      (const void*)mori::evict_order_cluster_kernel<8>, (const void*)mori::evict_order_cluster_kernel<16>};
  for (const void* k : ks) ok = ok && cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
  if (ok) {
    cudaLaunchConfig_t lc{};
    lc.gridDim = dim3(16); lc.blockDim = dim3(1024);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 16; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.attrs = at; lc.numAttrs = 1;
    int n_clusters = 0;
    ok = cudaOccupancyMaxActiveClusters(&n_clusters, mori::evict_order_cluster_kernel<8>, &lc) == cudaSuccess && n_clusters >= 1;
  }
  cudaGetLastError();
  d.cluster = ok ? 16 : 8;
  d.scratch = ptr;
  d.ready = true;
  return nullptr;
}
}  // namespace

extern "C" {

int mori_eviction_order_noalloc(void* stream, int32_t which_tier, int64_t n_pages, const int32_t* page_owner,
                                int32_t n_programs, const uint8_t* program_tier, const uint32_t* last_access,
                                int32_t* victims, int32_t* n_resident, const char** why) {
  const char* dummy;
  const char*& msg = why ? *why : dummy;
  msg = "";
  if (which_tier != MORI_TIER_GPU && which_tier != MORI_TIER_CPU) { msg = "which_tier must be MORI_TIER_GPU or MORI_TIER_CPU"; return MORI_ERR_INVALID_ARG; }
  if (n_pages < 0 || n_programs < 0) { msg = "n_pages / n_programs is negative"; return MORI_ERR_INVALID_ARG; }
  if (n_pages > MORI_NOALLOC_MAX_PAGES) {
    msg = "n_pages exceeds MORI_NOALLOC_MAX_PAGES (65536): the static scratch of this entry point is 1 MiB; "
          "use mori_eviction_order for larger pools";
    return MORI_ERR_CAPACITY;
  }
  if (n_pages > 0 && (!page_owner || !last_access || !victims || !n_resident || (n_programs > 0 && !program_tier))) {
    msg = "NULL array"; return MORI_ERR_INVALID_ARG;
  }
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); msg = "no current CUDA device"; return MORI_ERR_CUDA; }
  if (dev < 0 || dev >= kNoallocMaxDevices) { msg = "device ordinal beyond 63"; return MORI_ERR_UNSUPPORTED; }
  {
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (const char* e = noalloc_setup(dev)) { msg = e; return e[0] == 'l' ? MORI_ERR_UNSUPPORTED : MORI_ERR_CUDA; }
  }
  const NoallocDev& d = g_noalloc_dev[dev];
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (n_pages == 0) {
    if (n_resident && cudaMemsetAsync(n_resident, 0, sizeof(int32_t), s) != cudaSuccess) {
      cudaGetLastError(); msg = "cudaMemsetAsync(n_resident) failed"; return MORI_ERR_CUDA;
    }
    return MORI_OK;
  }
  mori::EvictArgs a{n_pages, n_programs, which_tier == MORI_TIER_GPU ? 0 : 1, 0, page_owner, program_tier, last_access};
  const int csize = d.cluster;
  const long long seg = ((n_pages + csize - 1) / csize + 1023) / 1024 * 1024;
  const int rounds = (int)(seg / 1024);                              // <= 8 at the maximum with a cluster of 8
  uint64_t* b0 = reinterpret_cast<uint64_t*>(d.scratch);             // the DEVICE address, not the symbol
  uint64_t* b1 = b0 + MORI_NOALLOC_MAX_PAGES;
  cudaLaunchConfig_t lc{};
  lc.gridDim = dim3(csize); lc.blockDim = dim3(1024); lc.dynamicSmemBytes = 0; lc.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = csize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lc.attrs = at; lc.numAttrs = 1;
  cudaError_t le;
  if (rounds <= 2) le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<2>, a, b0, b1, victims, n_resident);
  else if (rounds <= 4) le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<4>, a, b0, b1, victims, n_resident);
  else if (rounds <= 8) le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<8>, a, b0, b1, victims, n_resident);
  else le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<16>, a, b0, b1, victims, n_resident);
  if (le != cudaSuccess) { cudaGetLastError(); msg = "launch of the eviction-order kernel failed"; return MORI_ERR_CUDA; }
  return MORI_OK;
}

const char* mori_last_error(const mori_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int mori_create(const mori_config* cfg, mori_ctx** out) {
  if (out) *out = nullptr;
  if (!cfg || !out) return fail(nullptr, MORI_ERR_INVALID_ARG, "cfg/out is NULL");
  if (cfg->n_layers <= 0 || cfg->n_kv_heads <= 0 || cfg->head_dim <= 0 || cfg->page_tokens <= 0 ||
      cfg->elem_bytes <= 0)
    return fail(nullptr, MORI_ERR_INVALID_ARG, "KV shape fields must be positive");
  if (!cfg->gpu_pool || cfg->gpu_pool_pages <= 0) return fail(nullptr, MORI_ERR_INVALID_ARG, "gpu_pool missing");
  if (cfg->gpu_pool_pages > INT32_MAX || cfg->host_arena_slots > INT32_MAX || cfg->host_arena_slots < 0)
    return fail(nullptr, MORI_ERR_INVALID_ARG, "page/slot counts must fit int32");
  if (cfg->max_programs < 1 || cfg->max_programs > MORI_MAX_PROGRAMS)
    return fail(nullptr, MORI_ERR_INVALID_ARG, "max_programs must be 1..8192");
  const long long chunk = 2LL * cfg->n_kv_heads * cfg->page_tokens * cfg->head_dim * cfg->elem_bytes;
  if (chunk % 16 != 0 || chunk > (1LL << 30)) return fail(nullptr, MORI_ERR_INVALID_ARG, "chunk must be a multiple of 16 bytes");
  if (((uintptr_t)cfg->gpu_pool & 15) || ((uintptr_t)cfg->host_arena & 15))
    return fail(nullptr, MORI_ERR_INVALID_ARG, "gpu_pool and host_arena must be 16-byte aligned");
  for (int p : {cfg->path_demote, cfg->path_promote})
    if (p < MORI_PATH_AUTO || p > MORI_PATH_COPYENGINE) return fail(nullptr, MORI_ERR_INVALID_ARG, "bad path");
  if (cfg->copy_kernel < MORI_KERNEL_AUTO || cfg->copy_kernel > MORI_KERNEL_TMA)
    return fail(nullptr, MORI_ERR_INVALID_ARG, "bad copy_kernel");
  if (cfg->staging_bytes < 0 || cfg->max_pages_per_call < 0) return fail(nullptr, MORI_ERR_INVALID_ARG, "negative size");
  if (cfg->zerocopy_ctas < 0 || cfg->zerocopy_ctas > 1024 || cfg->idleness_window < 0 || cfg->idleness_window > 64) return fail(nullptr, MORI_ERR_INVALID_ARG, "bad zerocopy_ctas / idleness_window");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(nullptr, MORI_ERR_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(e));
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) return fail(nullptr, MORI_ERR_CUDA, cudaGetErrorString(e));
  if (prop.major != 10) return fail(nullptr, MORI_ERR_UNSUPPORTED, "libmori is built for sm_100a (B200) only");

  mori_ctx* c = new mori_ctx();
  c->cfg = *cfg;
  c->device = dev;
  c->sm_count = prop.multiProcessorCount;
  c->chunk = chunk;
  if (cfg->zerocopy_ctas > 0) c->link_ctas = cfg->zerocopy_ctas;
  c->page_bytes = chunk * cfg->n_layers;
  // Ring geometry of the bulk-copy kernel: `ctas_per_sm` CTAs share an SM's ring budget, each with
  // as many stages of `piece` bytes as fit (DESIGN.md section 5.2 has the measurements behind the
  // defaults).
  c->ctas_per_sm = (int)std::max<long long>(1, std::min<long long>(8, env_ll("MORI_CTAS_PER_SM", 1)));
  const long long ring_bytes = std::max<long long>(16, std::min<long long>(200, env_ll("MORI_RING_KIB", kRingBytesDefault >> 10))) << 10;
  const long long piece_max = std::max<long long>(1, std::min<long long>(128, env_ll("MORI_PIECE_KIB", kPieceBytesDefault >> 10))) << 10;
  c->piece = (int)std::min<long long>(piece_max, chunk);
  c->ppc = (int)((chunk + c->piece - 1) / c->piece);
  c->copy_kernel = cfg->copy_kernel == MORI_KERNEL_AUTO ? MORI_KERNEL_TMA : cfg->copy_kernel;
  c->tma_stages = (int)std::max<long long>(2, std::min<long long>(kMaxTmaStages, ring_bytes / c->ctas_per_sm / c->piece));
  c->tma_lag = c->tma_stages >= 6 ? 2 : 1;
  c->tma_smem = mori::tma_smem_bytes(c->tma_stages, c->piece);
  if (c->tma_smem > (size_t)prop.sharedMemPerBlockOptin) {
    delete c;
    return fail(nullptr, MORI_ERR_INVALID_ARG, "copy-kernel ring does not fit shared memory (chunk too large for 2 stages)");
  }
  c->debug = env_ll("MORI_DEBUG", 0) != 0;
  c->evict_multi_kernel = env_ll("MORI_EVICT_MULTI", 0) != 0;
  c->evict_cluster_want = (int)env_ll("MORI_EVICT_CLUSTER", 16);
  c->max_pages = cfg->max_pages_per_call ? cfg->max_pages_per_call
                                          : std::max<long long>(cfg->gpu_pool_pages, cfg->host_arena_slots);
  // Staging: the gather / scatter kernels run one launch per segment, and a launch pays ~15 us of
  // ramp and tail whatever its size, so segments are as large as HBM comfortably allows: 2 GiB
  // (4 buffers = 8 GiB; in-step 0.99 of the measured HBM copy rate) when >= 32 GiB are free, 1 GiB
  // (0.93) when >= 12 GiB are, else 256 MiB.  DESIGN.md section 7.
  long long staging_default = 256LL << 20;
  {
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
      if (free_b >= (32ULL << 30)) staging_default = 2048LL << 20;
      else if (free_b >= (12ULL << 30)) staging_default = 1024LL << 20;
    } else {
      cudaGetLastError();
    }
  }
  c->staging_bytes = cfg->staging_bytes ? cfg->staging_bytes : (env_ll("MORI_STAGING_MIB", staging_default >> 20) << 20);
  c->staging_bytes = std::min(c->staging_bytes, c->max_pages * c->page_bytes);   // never more than one call can fill
  c->staging_bytes = std::max(c->staging_bytes, c->page_bytes);
  c->staging_bytes -= c->staging_bytes % c->page_bytes;
  // AUTO: see DESIGN.md section 6 for the measurements behind this choice.
  c->dir[0].path = cfg->path_demote == MORI_PATH_AUTO ? MORI_PATH_STAGED : cfg->path_demote;
  c->dir[1].path = cfg->path_promote == MORI_PATH_AUTO ? MORI_PATH_STAGED : cfg->path_promote;
  c->dir[0].auto_path = cfg->path_demote == MORI_PATH_AUTO;
  c->dir[1].auto_path = cfg->path_promote == MORI_PATH_AUTO;
  *out = c;   // from here on mori_destroy cleans up

#define CKC(call)                                                                             \
  do {                                                                                        \
    cudaError_t e2_ = (call);                                                                 \
    if (e2_ != cudaSuccess) {                                                                 \
      g_create_error = std::string(#call) + ": " + cudaGetErrorString(e2_);                   \
      mori_destroy(c); *out = nullptr; return MORI_ERR_CUDA;                                  \
    }                                                                                         \
  } while (0)

  // CUDA loads kernels lazily, on their first launch (tens of microseconds each): touch the hot
  // path's kernels now so that no epoch pays for it -- a small move is a single ~10 us launch.
  {
    cudaFuncAttributes fa;
    const void* hot[] = {(const void*)mori::copy_pages_small<true, mori::kSmallFewPages>,
                         (const void*)mori::copy_pages_small<false, mori::kSmallFewPages>,
                         (const void*)mori::copy_pages_small<true, mori::kSmallMaxPages>,
                         (const void*)mori::copy_pages_small<false, mori::kSmallMaxPages>,
                         (const void*)mori::copy_pages_tma<true>, (const void*)mori::copy_pages_tma<false>,
                         (const void*)mori::copy_pages_ldst<true>, (const void*)mori::copy_pages_ldst<false>,
                         (const void*)upload_idx_kernel, (const void*)mori::rank_partition_kernel<1>,
                         (const void*)mori::rank_partition_multi_kernel<2>, (const void*)mori::rank_partition_multi_kernel<4>,
                         (const void*)mori::rank_partition_multi_kernel<8>};
    for (const void* f : hot) CKC(cudaFuncGetAttributes(&fa, f));
    // ... and the one-launch movers really run once, on nothing (n_pages = 0): the first launch of a
    // kernel costs tens of microseconds more than the next, which for a 272 KiB move is the move
    mori::CopyArgs z{};
    z.n_layers = 1; z.chunk_bytes = 16; z.piece_bytes = 16; z.pieces_per_chunk = 1; z.stages = 2; z.store_lag = 1;
    mori::copy_pages_small<true, mori::kSmallFewPages><<<1, mori::kLdstThreads>>>(z, mori::SmallIds<mori::kSmallFewPages>{});
    mori::copy_pages_small<false, mori::kSmallFewPages><<<1, mori::kLdstThreads>>>(z, mori::SmallIds<mori::kSmallFewPages>{});
    mori::copy_pages_small<true, mori::kSmallMaxPages><<<1, mori::kLdstThreads>>>(z, mori::SmallIds<mori::kSmallMaxPages>{});
    mori::copy_pages_small<false, mori::kSmallMaxPages><<<1, mori::kLdstThreads>>>(z, mori::SmallIds<mori::kSmallMaxPages>{});
    CKC(cudaGetLastError());
    CKC(cudaDeviceSynchronize());
  }
  auto warm_streams = [&]() -> cudaError_t {      // first use of a stream / an event costs microseconds too
    mori::CopyArgs z{};
    z.n_layers = 1; z.chunk_bytes = 16; z.piece_bytes = 16; z.pieces_per_chunk = 1; z.stages = 2; z.store_lag = 1;
    for (int i = 0; i < 2; ++i) {
      Direction& d = c->dir[i];
      if (!d.kern) continue;
      mori::copy_pages_small<true, mori::kSmallFewPages><<<1, mori::kLdstThreads, 0, d.kern>>>(z, mori::SmallIds<mori::kSmallFewPages>{});
      cudaEventRecord(d.tickets[0], d.kern);
      cudaStreamWaitEvent(d.copy, d.tickets[0], 0);
    }
    cudaError_t e = cudaGetLastError();
    return e != cudaSuccess ? e : cudaDeviceSynchronize();
  };
  // The attribute is per function and PROCESS-wide: every context sets it to the device's opt-in
  // maximum, so contexts with different ring sizes never lower it under one another.
  CKC(cudaFuncSetAttribute(mori::copy_pages_tma<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin));
  CKC(cudaFuncSetAttribute(mori::copy_pages_tma<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin));
  CKC(cudaMalloc((void**)&c->rank_tickets, sizeof(unsigned int) * kRankTickets));
  CKC(cudaMemset(c->rank_tickets, 0, sizeof(unsigned int) * kRankTickets));
  if (c->evict_cluster_want >= 16) {
    // a cluster of 16 CTAs is a non-portable size: allowed per kernel, and only if the device can
    // co-schedule it (cudaOccupancyMaxActiveClusters); otherwise the portable 8
    bool ok = true;
    const void* ks[] = {(const void*)mori::evict_order_cluster_kernel<2>, (const void*)mori::evict_order_cluster_kernel<4>,
                        (const void*)mori::evict_order_cluster_kernel<8>, (const void*)mori::evict_order_cluster_kernel<16>};
    for (const void* k : ks) ok = ok && cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
    if (ok) {
      cudaLaunchConfig_t lc{};
      lc.gridDim = dim3(16); lc.blockDim = dim3(1024);
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = 16; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      lc.attrs = at; lc.numAttrs = 1;
      int n_clusters = 0;
      ok = cudaOccupancyMaxActiveClusters(&n_clusters, mori::evict_order_cluster_kernel<8>, &lc) == cudaSuccess && n_clusters >= 1;
    }
    cudaGetLastError();
    c->evict_cluster = ok ? 16 : 8;
  }
  if (env_ll("MORI_SCHED", 1) != 0) {
    CKC(cudaMalloc((void**)&c->sched, sizeof(unsigned int) * 2 * kSchedRing));
    CKC(cudaMemset(c->sched, 0, sizeof(unsigned int) * 2 * kSchedRing));
  }
  if (c->debug) {
    const long long ids = std::max<long long>(cfg->gpu_pool_pages, cfg->host_arena_slots);
    CKC(cudaMalloc((void**)&c->dbg_bitmap, sizeof(unsigned int) * (size_t)((ids + 31) / 32)));
    CKC(cudaMemset(c->dbg_bitmap, 0, sizeof(unsigned int) * (size_t)((ids + 31) / 32)));
    CKC(cudaHostAlloc((void**)&c->dbg_flag_host, sizeof(int), cudaHostAllocMapped));
    *c->dbg_flag_host = 0;
    CKC(cudaHostGetDevicePointer((void**)&c->dbg_flag, c->dbg_flag_host, 0));
  }
  c->idl_k = cfg->idleness_window ? cfg->idleness_window : 5;
  CKC(cudaMalloc((void**)&c->idl_r, sizeof(double) * (size_t)cfg->max_programs * c->idl_k));
  CKC(cudaMalloc((void**)&c->idl_a, sizeof(double) * (size_t)cfg->max_programs * c->idl_k));
  CKC(cudaMalloc((void**)&c->idl_pushed, sizeof(int32_t) * (size_t)cfg->max_programs));
  CKC(cudaMemset(c->idl_pushed, 0, sizeof(int32_t) * (size_t)cfg->max_programs));
  CKC(cudaMalloc((void**)&c->evict_max_last, sizeof(unsigned int)));
  CKC(cudaMalloc((void**)&c->sticky_order, sizeof(int32_t) * kRankTickets * (size_t)cfg->max_programs));
  if (cfg->host_arena) {
    // The arena may also be DEVICE memory -- a second pool in this GPU's HBM, or a peer GPU's HBM
    // mapped over NVLink (the intermediate tier of P:L347): then there is no host link to stage
    // for, and both directions are the one-kernel path at full grid.
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, cfg->host_arena) == cudaSuccess && at.type == cudaMemoryTypeDevice) {
      if (at.device != dev) {
        // a peer GPU's HBM: this GPU's SMs reach it over NVLink once peer access is on
        int can = 0;
        CKC(cudaDeviceCanAccessPeer(&can, dev, at.device));
        if (!can) {
          g_create_error = "host_arena is memory of GPU " + std::to_string(at.device) + ", which GPU " +
                           std::to_string(dev) + " cannot access as a peer";
          mori_destroy(c); *out = nullptr; return MORI_ERR_UNSUPPORTED;
        }
        const cudaError_t pe = cudaDeviceEnablePeerAccess(at.device, 0);
        if (pe != cudaSuccess && pe != cudaErrorPeerAccessAlreadyEnabled) CKC(pe);
        cudaGetLastError();
      }
      c->arena_is_device = true;
      c->arena_dev = static_cast<unsigned char*>(cfg->host_arena);
      for (int i = 0; i < 2; ++i) { c->dir[i].path = MORI_PATH_ZEROCOPY; c->dir[i].auto_path = false; }
    } else {
      cudaGetLastError();
      void* dp = nullptr;
      CKC(cudaHostGetDevicePointer(&dp, cfg->host_arena, 0));
      c->arena_dev = static_cast<unsigned char*>(dp);
    }
  }
  for (int i = 0; i < 2; ++i) {
    Direction& d = c->dir[i];
    CKC(cudaStreamCreateWithFlags(&d.kern, cudaStreamNonBlocking));
    CKC(cudaStreamCreateWithFlags(&d.copy, cudaStreamNonBlocking));
    d.tickets.resize(kTicketRing);
    for (auto& ev : d.tickets) CKC(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    if (cfg->host_arena) {
      d.idx_cap = std::max<long long>(4 * c->max_pages, 1 << 16);
      CKC(cudaHostAlloc((void**)&d.idx_host, sizeof(int32_t) * d.idx_cap, cudaHostAllocMapped));
      CKC(cudaHostGetDevicePointer((void**)&d.idx_host_dev, d.idx_host, 0));
      CKC(cudaMalloc((void**)&d.idx_dev, sizeof(int32_t) * d.idx_cap));
      if (d.path == MORI_PATH_STAGED) {
        for (int b = 0; b < 2; ++b) {
          CKC(cudaMalloc((void**)&d.staging[b], c->staging_bytes));
          CKC(cudaEventCreateWithFlags(&d.kern_done[b], cudaEventDisableTiming));
          CKC(cudaEventCreateWithFlags(&d.copy_done[b], cudaEventDisableTiming));
        }
      }
    }
  }
  CKC(warm_streams());
#undef CKC
  return MORI_OK;
}

int mori_destroy(mori_ctx* c) {
  if (!c) return MORI_OK;
  cudaDeviceSynchronize();
  for (int i = 0; i < 2; ++i) {
    Direction& d = c->dir[i];
    prof_collect(c, d);
    for (int b = 0; b < 2; ++b) {
      if (d.staging[b]) cudaFree(d.staging[b]);
      if (d.kern_done[b]) cudaEventDestroy(d.kern_done[b]);
      if (d.copy_done[b]) cudaEventDestroy(d.copy_done[b]);
    }
    if (d.idx_host) cudaFreeHost(d.idx_host);
    if (d.idx_dev) cudaFree(d.idx_dev);
    for (auto ev : d.tickets) if (ev) cudaEventDestroy(ev);
    if (d.kern) cudaStreamDestroy(d.kern);
    if (d.copy) cudaStreamDestroy(d.copy);
  }
  for (auto& p : c->pending_after) cudaEventDestroy(p.ev);
  for (auto ev : c->free_events) cudaEventDestroy(ev);
  for (auto ev : c->free_timing_events) cudaEventDestroy(ev);
  if (c->prof_base) cudaEventDestroy(c->prof_base);
  if (c->rank_tickets) cudaFree(c->rank_tickets);
  if (c->sched) cudaFree(c->sched);
  if (c->dbg_bitmap) cudaFree(c->dbg_bitmap);
  if (c->dbg_flag_host) cudaFreeHost(c->dbg_flag_host);
  if (c->sticky_order) cudaFree(c->sticky_order);
  for (int t = 0; t < 2; ++t) if (c->evict_exec[t]) cudaGraphExecDestroy(c->evict_exec[t]);
  if (c->evict_cap_stream) cudaStreamDestroy(c->evict_cap_stream);
  for (int b = 0; b < 2; ++b) if (c->evict_perm[b]) cudaFree(c->evict_perm[b]);
  if (c->evict_table) cudaFree(c->evict_table);
  if (c->evict_max_last) cudaFree(c->evict_max_last);
  if (c->idl_r) cudaFree(c->idl_r);
  if (c->idl_a) cudaFree(c->idl_a);
  if (c->idl_pushed) cudaFree(c->idl_pushed);
  delete c;
  return MORI_OK;
}

int mori_rank_partition(mori_ctx* c, void* stream, int32_t n, const float* idleness, const int32_t* kv_pages,
                        const uint8_t* prev_tier, int64_t gpu_cap, int64_t cpu_cap, int32_t* order,
                        uint8_t* tier, int32_t* bounds, int64_t* used, int32_t* lists, int32_t* counts) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (n < 0 || n > c->cfg.max_programs) return fail(c, MORI_ERR_INVALID_ARG, "n out of range (0..max_programs)");
  if (gpu_cap < 0 || cpu_cap < 0) return fail(c, MORI_ERR_INVALID_ARG, "negative capacity");
  if (!bounds || !used) return fail(c, MORI_ERR_INVALID_ARG, "bounds/used_pages is NULL");
  if (n > 0 && (!idleness || !kv_pages || !order || !tier)) return fail(c, MORI_ERR_INVALID_ARG, "NULL array");
  if (prev_tier && (!lists || !counts)) return fail(c, MORI_ERR_INVALID_ARG, "prev_tier given but lists/list_counts NULL");
  int n_pad = 64;                                  // the kernel's warp-local stages need >= 64
  while (n_pad < n) n_pad <<= 1;
  const int ipt = n_pad <= 1024 ? 1 : n_pad / 1024;
  const int threads = n_pad / ipt;
  if (n > mori::kRankMaxThreads) {
    // more than one CTA's worth: rank by counting on every SM, last CTA partitions
    const int grid = std::min(c->sm_count, (n + 7) / 8);
    const size_t smem_m = sizeof(uint64_t) * ((size_t)n + 66) + 2 * sizeof(long long) + 5 * (size_t)n;   // keys, scan scratch, staged sizes and tiers
    const unsigned long long slot_m = c->rank_seq++ % kRankTickets;
    unsigned int* tk = c->rank_tickets + slot_m;
    int32_t* so = c->sticky_order + slot_m * (size_t)c->cfg.max_programs;
    cudaStream_t sm = static_cast<cudaStream_t>(stream);
    long long* um = reinterpret_cast<long long*>(used);
    cudaError_t em;
#define LM(I) launch_rank_multi<I>(grid, smem_m, sm, n, idleness, kv_pages, prev_tier, gpu_cap, cpu_cap, order, tier, bounds, um, lists, counts, so, tk)
    switch (ipt) {
      case 2: em = LM(2); break;
      case 4: em = LM(4); break;
      default: em = LM(8); break;
    }
#undef LM
    CK(c, em);
    c->launches += 1;
    return MORI_OK;
  }
  const size_t smem = sizeof(uint64_t) * (n_pad + 66) + 2 * sizeof(long long);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaError_t e;
  long long* u = reinterpret_cast<long long*>(used);
  e = launch_rank<1>(threads, smem, s, n, n_pad, idleness, kv_pages, prev_tier, gpu_cap, cpu_cap, order, tier, bounds, u, lists, counts);
  CK(c, e);
  c->launches += 1;
  return MORI_OK;
}

int mori_sticky_rebalance(mori_ctx* c, void* stream, int32_t n, const float* idleness, const int32_t* kv_pages,
                          const uint8_t* prev_tier, const uint8_t* flags, int64_t gpu_cap, int64_t cpu_cap,
                          uint8_t* tier, uint8_t* lazy, int64_t* used, int32_t* lists, int32_t* counts) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (n < 0 || n > c->cfg.max_programs) return fail(c, MORI_ERR_INVALID_ARG, "n out of range (0..max_programs)");
  if (gpu_cap < 0 || cpu_cap < 0) return fail(c, MORI_ERR_INVALID_ARG, "negative capacity");
  if (!used || !counts) return fail(c, MORI_ERR_INVALID_ARG, "used_pages/list_counts is NULL");
  if (n > 0 && (!idleness || !kv_pages || !prev_tier || !flags || !tier || !lazy || !lists))
    return fail(c, MORI_ERR_INVALID_ARG, "NULL array");
  int n_pad = 1024;
  while (n_pad < n) n_pad <<= 1;
  const int grid = std::max(1, std::min(c->sm_count, (n + 7) / 8));
  const size_t smem = sizeof(uint64_t) * (2 * (size_t)n + 99) + 4 * sizeof(long long) + 6 * (size_t)n;   // keys, scan scratch, staged inputs
  const unsigned long long slot = c->rank_seq++ % kRankTickets;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  long long* u = reinterpret_cast<long long*>(used);
  int32_t* ord = c->sticky_order + slot * (size_t)c->cfg.max_programs;
  unsigned int* tk = c->rank_tickets + slot;
  cudaError_t e;
#define LS(I) launch_sticky<I>(grid, smem, s, n, idleness, kv_pages, prev_tier, flags, gpu_cap, cpu_cap, tier, lazy, u, lists, counts, ord, tk)
  switch (n_pad / 1024) {
    case 1: e = LS(1); break;
    case 2: e = LS(2); break;
    case 4: e = LS(4); break;
    default: e = LS(8); break;
  }
#undef LS
  CK(c, e);
  c->launches += 1;
  return MORI_OK;
}

int mori_rank_partition_tiers(mori_ctx* c, void* stream, int32_t n, const float* idleness, const int32_t* kv_pages,
                              int32_t n_tiers, const int64_t* cap_pages, const uint8_t* prev_tier, int32_t* order,
                              uint8_t* tier, int32_t* bounds, int64_t* used, int32_t* moves, int32_t* move_counts) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (n < 0 || n > c->cfg.max_programs) return fail(c, MORI_ERR_INVALID_ARG, "n out of range (0..max_programs)");
  if (n_tiers < 1 || n_tiers > mori::kMaxTiers || !cap_pages) return fail(c, MORI_ERR_INVALID_ARG, "n_tiers must be 1..8");
  if (!bounds || !used || (n > 0 && (!idleness || !kv_pages || !order || !tier))) return fail(c, MORI_ERR_INVALID_ARG, "NULL array");
  if (prev_tier && (!moves || !move_counts)) return fail(c, MORI_ERR_INVALID_ARG, "prev_tier given but moves/move_counts NULL");
  mori::TierCaps caps{};
  caps.n_tiers = n_tiers;
  for (int t = 0; t < n_tiers; ++t) {
    if (cap_pages[t] < 0) return fail(c, MORI_ERR_INVALID_ARG, "negative capacity");
    caps.cap[t] = cap_pages[t];
  }
  int n_pad = 1024;
  while (n_pad < n) n_pad <<= 1;
  const int grid = std::max(1, std::min(c->sm_count, (n + 7) / 8));
  const size_t smem = sizeof(uint64_t) * ((size_t)n + 33) + 2 * sizeof(long long);
  const unsigned long long slot_t = c->rank_seq++ % kRankTickets;
  unsigned int* tk = c->rank_tickets + slot_t;
  int32_t* so = c->sticky_order + slot_t * (size_t)c->cfg.max_programs;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  long long* u = reinterpret_cast<long long*>(used);
  cudaError_t e;
#define LT(I) launch_tiers<I>(grid, smem, s, n, idleness, kv_pages, caps, prev_tier, order, tier, bounds, u, moves, move_counts, so, tk)
  switch (n_pad / 1024) {
    case 1: e = LT(1); break;
    case 2: e = LT(2); break;
    case 4: e = LT(4); break;
    default: e = LT(8); break;
  }
#undef LT
  CK(c, e);
  c->launches += 1;
  return MORI_OK;
}

int mori_bfd_assign(mori_ctx* c, void* stream, int32_t m, const int32_t* size, const float* idleness,
                    const uint8_t* flags, int32_t n_replicas, const int64_t* free_pages, int32_t* replica,
                    int64_t* free_out) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (m < 0 || m > c->cfg.max_programs) return fail(c, MORI_ERR_INVALID_ARG, "m out of range (0..max_programs)");
  if (n_replicas < 1 || n_replicas > mori::kBfdMaxReplicas) return fail(c, MORI_ERR_UNSUPPORTED, "n_replicas must be 1..32");
  if (!free_pages || !free_out || (m > 0 && (!size || !idleness || !flags || !replica)))
    return fail(c, MORI_ERR_INVALID_ARG, "NULL array");
  const int grid = std::max(1, std::min(c->sm_count, (m + 7) / 8));
  const size_t smem = sizeof(uint64_t) * 2 * (size_t)std::max(m, 1);
  const unsigned long long slot = c->rank_seq++ % kRankTickets;
  if (smem > 48 * 1024)
    CK(c, cudaFuncSetAttribute(mori::bfd_assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  mori::bfd_assign_kernel<<<grid, mori::kRankMaxThreads, smem, static_cast<cudaStream_t>(stream)>>>(
      m, size, idleness, flags, n_replicas, reinterpret_cast<const long long*>(free_pages), replica,
      reinterpret_cast<long long*>(free_out), c->sticky_order + slot * (size_t)c->cfg.max_programs,
      c->rank_tickets + slot);
  CK(c, cudaGetLastError());
  c->launches += 1;
  return MORI_OK;
}

int mori_eviction_order(mori_ctx* c, void* stream, int32_t which_tier, int64_t n_pages, const int32_t* page_owner,
                        int32_t n_programs, const uint8_t* program_tier, const uint32_t* last_access,
                        int32_t* victims, int32_t* n_resident) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (which_tier != MORI_TIER_GPU && which_tier != MORI_TIER_CPU) return fail(c, MORI_ERR_INVALID_ARG, "which_tier must be GPU or CPU");
  const long long limit = which_tier == MORI_TIER_GPU ? c->cfg.gpu_pool_pages : c->cfg.host_arena_slots;
  if (n_pages < 0 || n_pages > limit) return fail(c, MORI_ERR_INVALID_ARG, "n_pages exceeds the pool");
  if (n_programs < 0 || !n_resident) return fail(c, MORI_ERR_INVALID_ARG, "bad n_programs / n_resident");
  if (n_pages > 0 && (!page_owner || !last_access || !victims || (n_programs > 0 && !program_tier)))
    return fail(c, MORI_ERR_INVALID_ARG, "NULL array");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (n_pages == 0) { CK(c, cudaMemsetAsync(n_resident, 0, sizeof(int32_t), s)); return MORI_OK; }
  const int tiles = (int)((n_pages + mori::kEvictTile - 1) / mori::kEvictTile);
  if (n_pages > c->evict_cap) {                    // first use / larger pool: (re)allocate scratch
    CK(c, cudaStreamSynchronize(s));
    for (int t = 0; t < 2; ++t) if (c->evict_exec[t]) { cudaGraphExecDestroy(c->evict_exec[t]); c->evict_exec[t] = nullptr; }
    for (int b = 0; b < 2; ++b) { if (c->evict_perm[b]) cudaFree(c->evict_perm[b]); c->evict_perm[b] = nullptr; }
    if (c->evict_table) cudaFree(c->evict_table);
    c->evict_table = nullptr; c->evict_cap = 0;
    for (int b = 0; b < 2; ++b) CK(c, cudaMalloc((void**)&c->evict_perm[b], sizeof(uint64_t) * (size_t)n_pages));   // int32 order, or 64-bit items
    CK(c, cudaMalloc((void**)&c->evict_table, sizeof(int32_t) * 256 * (size_t)tiles));
    c->evict_cap = n_pages;
  }
  mori::EvictArgs a{n_pages, n_programs, which_tier == MORI_TIER_GPU ? 0 : 1, tiles, page_owner, program_tier, last_access};
  if (n_pages <= (long long)c->evict_cluster * 1024 * 16 && n_pages <= 2 * mori::kEvictClusterMaxPages && !c->evict_multi_kernel) {
    // every BASELINE.json pool: ONE launch, a cluster of 8 CTAs, passes separated by cluster barriers
    const int csize = c->evict_cluster;
    const long long seg = ((n_pages + csize - 1) / csize + 1023) / 1024 * 1024;
    const int rounds = (int)(seg / 1024);
    uint64_t* b0 = reinterpret_cast<uint64_t*>(c->evict_perm[0]);
    uint64_t* b1 = reinterpret_cast<uint64_t*>(c->evict_perm[1]);
    cudaLaunchConfig_t lc{};
    lc.gridDim = dim3(csize); lc.blockDim = dim3(1024); lc.dynamicSmemBytes = 0; lc.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = csize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.attrs = at; lc.numAttrs = 1;
    cudaError_t le;
    if (rounds <= 2) le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<2>, a, b0, b1, victims, n_resident);
    else if (rounds <= 4) le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<4>, a, b0, b1, victims, n_resident);
    else if (rounds <= 8) le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<8>, a, b0, b1, victims, n_resident);
    else le = cudaLaunchKernelEx(&lc, mori::evict_order_cluster_kernel<16>, a, b0, b1, victims, n_resident);
    CK(c, le);
    CK(c, cudaGetLastError());
    c->launches += 1;
    return MORI_OK;
  }
  auto enqueue = [&](cudaStream_t q) -> cudaError_t {
    cudaError_t e = cudaMemsetAsync(n_resident, 0, sizeof(int32_t), q);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(c->evict_max_last, 0, sizeof(unsigned int), q);
    if (e != cudaSuccess) return e;
    const int32_t* in = nullptr;                   // pass 0 reads the pages in id order
    for (int pass = 0; pass < mori::kEvictPasses; ++pass) {
      int32_t* out = pass == mori::kEvictPasses - 1 ? victims : c->evict_perm[pass & 1];
      mori::evict_hist_kernel<<<tiles, mori::kEvictTile, 0, q>>>(a, pass, in, c->evict_table, n_resident, c->evict_max_last);
      mori::evict_scan_kernel<<<1, mori::kRankMaxThreads, 0, q>>>(c->evict_table, 256 * tiles, pass, c->evict_max_last);
      mori::evict_scatter_kernel<<<tiles, mori::kEvictTile, 0, q>>>(a, pass, in, c->evict_table, out, c->evict_max_last);
      in = out;
    }
    return cudaGetLastError();
  };
  // Launch-bound (15 small kernels + a memset): captured once into a CUDA graph per (tier,
  // argument set) -- an engine passes the same tables every time, and alternating between the two
  // tiers keeps both graphs -- and replayed with one cudaGraphLaunch.  The scratch is shared, so
  // calls must be enqueued on one stream at a time (include/mori.h).
  const int gi = which_tier == MORI_TIER_GPU ? 0 : 1;
  cudaGraphExec_t& exec = c->evict_exec[gi];
  mori_ctx::EvictKey& key = c->evict_key[gi];
  const bool same = exec && key.n_programs == n_programs && key.n_pages == n_pages && key.owner == page_owner &&
                    key.ptier == program_tier && key.last == last_access && key.victims == victims &&
                    key.nres == n_resident;
  if (!same) {
    if (exec) { cudaGraphExecDestroy(exec); exec = nullptr; }
    if (!c->evict_cap_stream) cudaStreamCreateWithFlags(&c->evict_cap_stream, cudaStreamNonBlocking);
    cudaGraph_t g = nullptr;
    if (c->evict_cap_stream &&
        cudaStreamBeginCapture(c->evict_cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      const cudaError_t e1 = enqueue(c->evict_cap_stream);
      const cudaError_t e2 = cudaStreamEndCapture(c->evict_cap_stream, &g);
      if (e1 == cudaSuccess && e2 == cudaSuccess && g && cudaGraphInstantiate(&exec, g, 0) != cudaSuccess)
        exec = nullptr;
      if (e1 != cudaSuccess || e2 != cudaSuccess) exec = nullptr;
      if (g) cudaGraphDestroy(g);
    }
    cudaGetLastError();                            // a failed capture falls back to plain launches
    key = {n_programs, n_pages, page_owner, program_tier, last_access, victims, n_resident};
  }
  if (exec) CK(c, cudaGraphLaunch(exec, s));
  else CK(c, enqueue(s));
  c->launches += 3 * mori::kEvictPasses;
  return MORI_OK;
}

int mori_idleness_update(mori_ctx* c, void* stream, int64_t m, const int32_t* prog, const uint8_t* kind,
                         const double* reasoning, const double* acting) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (m < 0 || (m > 0 && (!prog || !kind || !reasoning || !acting))) return fail(c, MORI_ERR_INVALID_ARG, "bad event list");
  if (m == 0) return MORI_OK;
  const int n = c->cfg.max_programs;
  mori::idleness_update_kernel<<<(n + mori::kIdlenessThreads - 1) / mori::kIdlenessThreads, mori::kIdlenessThreads, 0,
                                 static_cast<cudaStream_t>(stream)>>>(n, c->idl_k, c->idl_r, c->idl_a, c->idl_pushed, m,
                                                                      prog, kind, reasoning, acting);
  CK(c, cudaGetLastError());
  c->launches += 1;
  return MORI_OK;
}

int mori_idleness_eval(mori_ctx* c, void* stream, int32_t n, const double* open_r, const double* open_a, float* out) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (n < 0 || n > c->cfg.max_programs) return fail(c, MORI_ERR_INVALID_ARG, "n out of range (0..max_programs)");
  if (n > 0 && !out) return fail(c, MORI_ERR_INVALID_ARG, "idleness_out is NULL");
  if (n == 0) return MORI_OK;
  mori::idleness_eval_kernel<<<(n + mori::kIdlenessThreads - 1) / mori::kIdlenessThreads, mori::kIdlenessThreads, 0,
                               static_cast<cudaStream_t>(stream)>>>(n, c->idl_k, c->idl_r, c->idl_a, c->idl_pushed,
                                                                    open_r, open_a, out);
  CK(c, cudaGetLastError());
  c->launches += 1;
  return MORI_OK;
}

// MORI_DEBUG only: validates a DEVICE page table on `stream` and waits for the verdict.
static int debug_validate(mori_ctx* c, cudaStream_t s, long long n, const int32_t* ids, bool check_dup) {
  if (!c->debug || n == 0) return MORI_OK;
  *c->dbg_flag_host = 0;
  const int grid = (int)std::min<long long>((n + 255) / 256, 1024);
  validate_ids_kernel<<<grid, 256, 0, s>>>(ids, n, c->cfg.gpu_pool_pages, c->dbg_bitmap, check_dup ? 1 : 0, 0, c->dbg_flag);
  if (check_dup)
    validate_ids_kernel<<<grid, 256, 0, s>>>(ids, n, c->cfg.gpu_pool_pages, c->dbg_bitmap, 1, 1, c->dbg_flag);
  CK(c, cudaGetLastError());
  CK(c, cudaStreamSynchronize(s));
  const int f = *c->dbg_flag_host;
  if (f & 1) return fail(c, MORI_ERR_INVALID_ARG, "MORI_DEBUG: gpu page id out of range in a device page table");
  if (f & 2) return fail(c, MORI_ERR_INVALID_ARG, "MORI_DEBUG: duplicate destination gpu page in a device page table");
  return MORI_OK;
}

int mori_gather_pages(mori_ctx* c, void* stream, int64_t n_pages, const int32_t* gpu_pages, void* dst) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (n_pages < 0 || (n_pages > 0 && (!gpu_pages || !dst))) return fail(c, MORI_ERR_INVALID_ARG, "bad gather arguments");
  if (int rc = debug_validate(c, static_cast<cudaStream_t>(stream), n_pages, gpu_pages, false)) return rc;
  mori::CopyArgs a = make_args(c, static_cast<unsigned char*>(dst), gpu_pages, nullptr, n_pages);
  CK(c, launch_copy<true>(c, a, static_cast<cudaStream_t>(stream), false));
  return MORI_OK;
}

int mori_scatter_pages(mori_ctx* c, void* stream, int64_t n_pages, const int32_t* gpu_pages, const void* src) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (n_pages < 0 || (n_pages > 0 && (!gpu_pages || !src))) return fail(c, MORI_ERR_INVALID_ARG, "bad scatter arguments");
  if (int rc = debug_validate(c, static_cast<cudaStream_t>(stream), n_pages, gpu_pages, true)) return rc;
  mori::CopyArgs a = make_args(c, static_cast<unsigned char*>(const_cast<void*>(src)), gpu_pages, nullptr, n_pages);
  CK(c, launch_copy<false>(c, a, static_cast<cudaStream_t>(stream), false));
  return MORI_OK;
}

// Enqueues the waits that earlier mori_after_stream calls owe the streams of direction `di` that
// are about to get work, and recycles the events no stream needs any more.
static int consume_pending_after(mori_ctx* c, int di, bool kern, bool copy) {
  if (c->pending_after.empty()) return MORI_OK;
  Direction& d = c->dir[di];
  const int bit_k = 1 << (2 * di), bit_c = 1 << (2 * di + 1);
  for (auto& p : c->pending_after) {
    if (kern && (p.streams_left & bit_k)) { CK(c, cudaStreamWaitEvent(d.kern, p.ev, 0)); p.streams_left &= ~bit_k; }
    if (copy && (p.streams_left & bit_c)) { CK(c, cudaStreamWaitEvent(d.copy, p.ev, 0)); p.streams_left &= ~bit_c; }
  }
  size_t keep = 0;
  for (auto& p : c->pending_after) {
    if (p.streams_left) c->pending_after[keep++] = p;
    else c->free_events.push_back(p.ev);
  }
  c->pending_after.resize(keep);
  return MORI_OK;
}

// Drops the pending entries whose caller-stream event has already completed: the dependency holds.
static void prune_pending_after(mori_ctx* c) {
  size_t keep = 0;
  for (auto& p : c->pending_after) {
    if (cudaEventQuery(p.ev) == cudaSuccess) c->free_events.push_back(p.ev);
    else c->pending_after[keep++] = p;
  }
  cudaGetLastError();                              // cudaErrorNotReady is not an error
  c->pending_after.resize(keep);
}

// Shared body of mori_demote (dir 0) and mori_promote (dir 1).
//   wait_pool   ticket of the OTHER direction after which this call may touch the POOL
//   wait_arena  ticket of the OTHER direction after which this call may touch the ARENA
// (mori_demote passes the same ticket twice.)  On every path both hold for every byte of the call.
static int migrate(mori_ctx* c, int di, long long total, const int32_t* gpu_pages, const int32_t* host_slots,
                   long long wait_pool, long long wait_arena, int64_t* ticket_out) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!c->cfg.host_arena) return fail(c, MORI_ERR_STATE, "context was created without a host arena");
  if (total < 0 || (total > 0 && (!gpu_pages || !host_slots))) return fail(c, MORI_ERR_INVALID_ARG, "bad page table");
  if (total > c->max_pages) return fail(c, MORI_ERR_CAPACITY, "total_pages exceeds max_pages_per_call");
  if (int rc = check_ids(c, total, gpu_pages, host_slots)) return rc;
  Direction& d = c->dir[di];
  Direction& other = c->dir[1 - di];
  const bool demote = di == 0;
  if (c->debug) {
    const int rc = demote ? check_duplicates(c, total, host_slots, c->cfg.host_arena_slots, "host slot")
                          : check_duplicates(c, total, gpu_pages, c->cfg.gpu_pool_pages, "gpu page");
    if (rc) return rc;
  }
  for (long long t : {wait_pool, wait_arena})
    if (t > 0 && t >= other.next_ticket) return fail(c, MORI_ERR_INVALID_ARG, "ticket was never issued");
  unsigned char* pool = static_cast<unsigned char*>(c->cfg.gpu_pool);
  unsigned char* arena = static_cast<unsigned char*>(c->cfg.host_arena);
  const long long pb = c->page_bytes;

  // AUTO: a few pages -> the one-launch path.  Otherwise a DMA per run of
  // consecutive slots costs ~4.3 us of copy-engine set-up, so short runs (2 MiB: 89 % of the link
  // peak, 4 MiB: 94 %) lose to SM-driven zero-copy (92 % whatever the run length); long runs
  // (>= 8 MiB: 97-100 %) win.
  int path = d.path;
  bool small = false;
  if (d.auto_path && total > 0) {
    small = total <= mori::kSmallMaxPages && total * pb <= kSmallMaxBytes;
    long long runs = 1;
    for (long long j = 1; j < total; ++j) runs += host_slots[j] != host_slots[j - 1] + 1;
    path = (small || total * pb / runs < kAutoMinRunBytes) ? MORI_PATH_ZEROCOPY : MORI_PATH_STAGED;
  }

  if (int rc = consume_pending_after(c, di, true, path == MORI_PATH_STAGED)) return rc;
  d.kern_busy = true;
  // one stream carries the whole call on every path but STAGED: it waits for both tickets
  auto wait_both = [&](cudaStream_t s) -> int {
    if (int rc = wait_ticket(c, other, wait_pool, s)) return rc;
    if (wait_arena != wait_pool) if (int rc = wait_ticket(c, other, wait_arena, s)) return rc;
    return MORI_OK;
  };

  if (path == MORI_PATH_ZEROCOPY) {
    if (int rc = wait_both(d.kern)) return rc;
    // Calls of one direction take effect in issue order.  An earlier STAGED demote of this
    // direction may still have DMAs in flight on the copy stream: this kernel must not overtake
    // them (same-stream order covers every other combination of paths).
    if (demote && d.copy_busy)
      for (int b = 0; b < 2; ++b)
        if (d.copy_done[b]) CK(c, cudaStreamWaitEvent(d.kern, d.copy_done[b], 0));
    if (total > 0) {
      prof_begin(c, d, d.kern, total * pb);
      if (small) {
        CK(c, demote ? launch_small<true>(c, total, gpu_pages, host_slots, d.kern)
                     : launch_small<false>(c, total, gpu_pages, host_slots, d.kern));
      } else {
        const int32_t *dg, *dh;
        if (int rc = stage_indices(c, d, total, gpu_pages, host_slots, &dg, &dh)) return rc;
        mori::CopyArgs a = make_args(c, c->arena_dev, dg, dh, total);
        CK(c, demote ? launch_copy<true>(c, a, d.kern, !c->arena_is_device) : launch_copy<false>(c, a, d.kern, !c->arena_is_device));
      }
      prof_end(c, d, d.kern);
    }
    return issue_ticket(c, d, d.kern, ticket_out);
  }

  if (path == MORI_PATH_COPYENGINE) {
    if (int rc = wait_both(d.kern)) return rc;
    const size_t dpitch = (size_t)c->cfg.gpu_pool_pages * c->chunk;   // layer stride in the pool
    for (long long j = 0; j < total; ++j) {
      unsigned char* dev = pool + (long long)gpu_pages[j] * c->chunk;
      unsigned char* hst = arena + (long long)host_slots[j] * pb;
      if (demote) CK(c, cudaMemcpy2DAsync(hst, c->chunk, dev, dpitch, c->chunk, c->cfg.n_layers, cudaMemcpyDeviceToHost, d.kern));
      else        CK(c, cudaMemcpy2DAsync(dev, dpitch, hst, c->chunk, c->chunk, c->cfg.n_layers, cudaMemcpyHostToDevice, d.kern));
    }
    return issue_ticket(c, d, d.kern, ticket_out);
  }

  // STAGED.  demote:  kern stream: gather -> staging[b]      copy stream: staging[b] -> arena
  //          promote: copy stream: arena -> staging[b]       kern stream: staging[b] -> scatter
  // Double-buffered with events so the DMA of segment i overlaps the kernel of segment i+1.
  // demote : the gather (pool reads) is first in the pipeline and every DMA follows a gather, so
  //          both tickets gate the kernel stream.
  // promote: the DMAs read the ARENA -> the copy stream waits for wait_arena; the scatters write
  //          the POOL -> the kernel stream waits for wait_pool.  A promotion into pages that a
  //          demotion is still vacating therefore streams its bytes over the link meanwhile.
  const long long seg_pages = c->staging_bytes / pb;
  const int32_t* dg = nullptr; const int32_t* dh = nullptr;
  if (demote) { if (int rc = wait_both(d.kern)) return rc; }
  else {
    if (int rc = wait_ticket(c, other, wait_arena, d.copy)) return rc;
    if (int rc = wait_ticket(c, other, wait_pool, d.kern)) return rc;
  }
  if (total > 0)
    if (int rc = stage_indices(c, d, total, gpu_pages, host_slots, &dg, &dh)) return rc;
  if (total > 0) d.copy_busy = true;
  // The pipeline's ramp: a demotion's first DMA waits for its first gather and a promotion's last
  // scatter runs after its last DMA, so those two segments are short (<= 512 MiB: ~0.17 ms of kernel
  // instead of ~0.65 ms for a 2 GiB segment); every other kernel hides under a DMA.
  // The rest of the call is cut into EQUAL segments (6.1 GiB = ramp + 3 x 1.95 GiB, not ramp + 2 + 2 +
  // 1.85 + a 0.1 GiB tail whose launch would be all ramp and tail).
  const long long ramp_pages = std::max<long long>(1, std::min<long long>(seg_pages, kRampBytes / pb));
  const long long ramp = total > 2 * ramp_pages ? ramp_pages : 0;
  const long long body = total - ramp;
  const long long n_body = (body + seg_pages - 1) / seg_pages;              // segments of the body
  long long seg_i = 0;
  for (long long a0 = 0, cnt = 0; a0 < total; a0 += cnt, ++seg_i) {
    const long long bi = demote ? seg_i - (ramp ? 1 : 0) : seg_i;           // index within the body, or outside it
    if (bi < 0 || bi >= n_body) cnt = ramp;                                 // the ramp: first (demote) / last (promote)
    else cnt = body / n_body + (bi < body % n_body ? 1 : 0);
    const int b = d.buf; d.buf ^= 1;
    unsigned char* stg = d.staging[b];
    mori::CopyArgs a = make_args(c, stg, dg + a0, nullptr, cnt);
    auto dma = [&](cudaStream_t s) -> int {
      for (long long i = 0; i < cnt;) {                      // one DMA per run of consecutive slots
        long long r = 1;
        while (i + r < cnt && host_slots[a0 + i + r] == host_slots[a0 + i] + r) ++r;
        unsigned char* h = arena + (long long)host_slots[a0 + i] * pb;
        if (demote) CK(c, cudaMemcpyAsync(h, stg + i * pb, r * pb, cudaMemcpyDeviceToHost, s));
        else        CK(c, cudaMemcpyAsync(stg + i * pb, h, r * pb, cudaMemcpyHostToDevice, s));
        i += r;
      }
      return MORI_OK;
    };
    if (demote) {
      CK(c, cudaStreamWaitEvent(d.kern, d.copy_done[b], 0));       // staging[b] drained
      prof_begin(c, d, d.kern, cnt * pb);
      CK(c, launch_copy<true>(c, a, d.kern, false));
      prof_end(c, d, d.kern);
      CK(c, cudaEventRecord(d.kern_done[b], d.kern));
      CK(c, cudaStreamWaitEvent(d.copy, d.kern_done[b], 0));
      prof_begin(c, d, d.copy, cnt * pb, 1);
      if (int rc = dma(d.copy)) return rc;
      prof_end(c, d, d.copy, 1);
      CK(c, cudaEventRecord(d.copy_done[b], d.copy));
    } else {
      CK(c, cudaStreamWaitEvent(d.copy, d.kern_done[b], 0));       // staging[b] scattered
      prof_begin(c, d, d.copy, cnt * pb, 1);
      if (int rc = dma(d.copy)) return rc;
      prof_end(c, d, d.copy, 1);
      CK(c, cudaEventRecord(d.copy_done[b], d.copy));
      CK(c, cudaStreamWaitEvent(d.kern, d.copy_done[b], 0));
      prof_begin(c, d, d.kern, cnt * pb);
      CK(c, launch_copy<false>(c, a, d.kern, false));
      prof_end(c, d, d.kern);
      CK(c, cudaEventRecord(d.kern_done[b], d.kern));
    }
  }
  // the ticket marks the end of the LAST stage of the pipeline
  if (demote) {
    // copy stream finishes last; it already follows the kernel stream, so one event on it covers
    // the call
    return issue_ticket(c, d, d.copy, ticket_out);
  }
  // promote: the kernel stream finishes last; an EMPTY call has put nothing on it that follows the
  // copy stream's wait for wait_arena, so fold that in for the ticket to cover both waits
  if (total == 0 && wait_arena > 0 && wait_arena != wait_pool)
    if (int rc = wait_ticket(c, other, wait_arena, d.kern)) return rc;
  return issue_ticket(c, d, d.kern, ticket_out);
}

int mori_demote(mori_ctx* c, int64_t total, const int32_t* gpu_pages, const int32_t* host_slots,
                int64_t wait_promote_ticket, int64_t* ticket_out) {
  return migrate(c, 0, total, gpu_pages, host_slots, wait_promote_ticket, wait_promote_ticket, ticket_out);
}

int mori_promote(mori_ctx* c, int64_t total, const int32_t* host_slots, const int32_t* gpu_pages,
                 int64_t pages_after_demote, int64_t slots_after_demote, int64_t* ticket_out) {
  return migrate(c, 1, total, gpu_pages, host_slots, pages_after_demote, slots_after_demote, ticket_out);
}

int mori_sync(mori_ctx* c, int32_t which) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (which < 1 || which > 3) return fail(c, MORI_ERR_INVALID_ARG, "which must be 1, 2 or 3");
  for (int i = 0; i < 2; ++i) {
    if (!(which & (1 << i))) continue;
    Direction& d = c->dir[i];
    cudaError_t e1 = cudaStreamSynchronize(d.kern);
    cudaError_t e2 = cudaStreamSynchronize(d.copy);
    if (e1 != cudaSuccess || e2 != cudaSuccess) {
      c->sticky = MORI_ERR_CUDA;
      return fail(c, MORI_ERR_CUDA, std::string("asynchronous failure: ") + cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
    }
    d.idx_used = 0;
    d.copy_busy = false;
    d.kern_busy = false;
    prof_collect(c, d);
  }
  prune_pending_after(c);
  return c->sticky;
}

int mori_after_stream(mori_ctx* c, int32_t which, void* stream) {
  if (!c || which < 1 || which > 3) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (c->pending_after.size() >= 16) {             // a caller that never joins: settle the old ones now
    prune_pending_after(c);
    for (int i = 0; i < 2 && !c->pending_after.empty(); ++i)
      if (int rc = consume_pending_after(c, i, true, true)) return rc;
  }
  cudaEvent_t ev = get_event(c, false);
  if (!ev) return c->sticky;
  CK(c, cudaEventRecord(ev, static_cast<cudaStream_t>(stream)));
  int left = 0;
  for (int i = 0; i < 2; ++i)
    if (which & (1 << i)) left |= 3 << (2 * i);    // the direction's kernel and DMA streams
  c->pending_after.push_back({ev, left});          // waited on when those streams next get work
  return MORI_OK;
}

int mori_stream_wait(mori_ctx* c, void* stream, int32_t which) {
  if (!c || which < 1 || which > 3) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  for (int i = 0; i < 2; ++i)
    if (which & (1 << i))
      for (cudaStream_t s : {c->dir[i].kern, c->dir[i].copy}) {
        if (s == c->dir[i].copy && !c->dir[i].copy_busy) continue;   // nothing enqueued there since the last join
        if (s == c->dir[i].kern && !c->dir[i].kern_busy) continue;
        cudaEvent_t ev = get_event(c, false);
        if (!ev) return c->sticky;
        CK(c, cudaEventRecord(ev, s));
        CK(c, cudaStreamWaitEvent(static_cast<cudaStream_t>(stream), ev, 0));
        c->free_events.push_back(ev);
      }
  return MORI_OK;
}

int mori_profile(mori_ctx* c, int32_t enable) {
  if (!c) return MORI_ERR_INVALID_ARG;
  c->profiling = enable != 0;
  c->timeline = enable == 2;
  if (c->timeline) {
    if (!c->prof_base) CK(c, cudaEventCreate(&c->prof_base));
    CK(c, cudaEventRecord(c->prof_base, c->dir[0].kern));           // time zero of the timeline
    CK(c, cudaEventSynchronize(c->prof_base));
    for (int i = 0; i < 2; ++i) c->dir[i].timeline.clear();
  }
  return MORI_OK;
}

int mori_profile_timeline(mori_ctx* c, int32_t which, int64_t max_rows, int32_t* kind, double* start_ms,
                          double* end_ms, int64_t* bytes, int64_t* n_rows) {
  if (!c || (which != MORI_DEMOTE && which != MORI_PROMOTE) || !n_rows || max_rows < 0) return MORI_ERR_INVALID_ARG;
  const auto& tl = c->dir[which - 1].timeline;
  *n_rows = (int64_t)tl.size();
  for (int64_t i = 0; i < std::min<int64_t>(max_rows, (int64_t)tl.size()); ++i) {
    if (kind) kind[i] = tl[i].kind;
    if (start_ms) start_ms[i] = tl[i].t0_ms;
    if (end_ms) end_ms[i] = tl[i].t1_ms;
    if (bytes) bytes[i] = tl[i].bytes;
  }
  return MORI_OK;
}

int mori_profile_read(mori_ctx* c, int32_t which, double* ms, int64_t* launches, int64_t* bytes) {
  if (!c || (which != MORI_DEMOTE && which != MORI_PROMOTE)) return MORI_ERR_INVALID_ARG;
  Direction& d = c->dir[which - 1];
  if (ms) *ms = d.prof_ms;
  if (launches) *launches = d.prof_launches;
  if (bytes) *bytes = d.prof_bytes;
  d.prof_ms = 0; d.prof_launches = 0; d.prof_bytes = 0;
  return MORI_OK;
}

__global__ void noop_kernel() {}

int mori_noop(mori_ctx* c, void* stream) {
  if (!c) return MORI_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  noop_kernel<<<1, 32, 0, static_cast<cudaStream_t>(stream)>>>();
  CK(c, cudaGetLastError());
  c->launches += 1;
  return MORI_OK;
}

int mori_launch_count(const mori_ctx* c, int64_t* out) {
  if (!c || !out) return MORI_ERR_INVALID_ARG;
  *out = c->launches;
  return MORI_OK;
}

int mori_host_alloc(int64_t bytes, void** out) {
  if (out) *out = nullptr;
  if (!out || bytes <= 0) return fail(nullptr, MORI_ERR_INVALID_ARG, "mori_host_alloc: bad arguments");
  // Anonymous memory backed by transparent huge pages, faulted in by a few threads, then
  // page-locked and mapped with cudaHostRegister: ~2.5x faster than cudaHostAlloc for the
  // 100+ GiB arenas of this workload, same DMA bandwidth (measured).
  constexpr size_t kHuge = 2u << 20;
  const size_t len = ((size_t)bytes + kHuge - 1) / kHuge * kHuge + kHuge;
  void* raw = mmap(nullptr, len, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
  if (raw != MAP_FAILED) {
    unsigned char* p = reinterpret_cast<unsigned char*>(((uintptr_t)raw + kHuge - 1) & ~(uintptr_t)(kHuge - 1));
    madvise(p, (size_t)bytes, MADV_HUGEPAGE);
    const int nt = (int)std::max<long long>(1, std::min<long long>(8, bytes / (1LL << 30)));
    std::vector<std::thread> th;
    for (int t = 0; t < nt; ++t)
      th.emplace_back([=] {
        const size_t lo = (size_t)bytes / nt * t, hi = t == nt - 1 ? (size_t)bytes : (size_t)bytes / nt * (t + 1);
        for (size_t o = lo; o < hi; o += 4096) p[o] = 0;
      });
    for (auto& t : th) t.join();
    cudaError_t e = cudaHostRegister(p, (size_t)bytes, cudaHostRegisterMapped | cudaHostRegisterPortable);
    if (e == cudaSuccess) {
      std::lock_guard<std::mutex> lk(g_host_mu);
      g_host_allocs[p] = {raw, len};
      *out = p;
      return MORI_OK;
    }
    cudaGetLastError();
    munmap(raw, len);
  }
  void* p = nullptr;
  cudaError_t e = cudaHostAlloc(&p, (size_t)bytes, cudaHostAllocMapped | cudaHostAllocPortable);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(nullptr, MORI_ERR_CUDA, std::string("cudaHostRegister and cudaHostAlloc failed: ") + cudaGetErrorString(e));
  }
  *out = p;
  return MORI_OK;
}

int mori_host_free(void* p) {
  if (!p) return MORI_OK;
  {
    std::lock_guard<std::mutex> lk(g_host_mu);
    auto it = g_host_allocs.find(p);
    if (it != g_host_allocs.end()) {
      const cudaError_t e = cudaHostUnregister(p);
      munmap(it->second.first, it->second.second);
      g_host_allocs.erase(it);
      return e == cudaSuccess ? MORI_OK : MORI_ERR_CUDA;
    }
  }
  return cudaFreeHost(p) == cudaSuccess ? MORI_OK : MORI_ERR_CUDA;
}

int mori_path(const mori_ctx* c, int32_t which) {
  if (!c || (which != MORI_DEMOTE && which != MORI_PROMOTE)) return MORI_ERR_INVALID_ARG;
  return c->dir[which - 1].path;
}

int mori_copy_kernel(const mori_ctx* c) { return c ? c->copy_kernel : MORI_ERR_INVALID_ARG; }

}  // extern "C"
