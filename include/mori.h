/*
 * mori.h -- C ABI of libmori.so: the data-parallel hot path under MORI's idleness-ranked
 * two-tier KV placement (arxiv/paper_2606_00866), hand-written for NVIDIA B200 (sm_100a).
 *
 * Citations "P:Lnnn" are lines of the paper text; "R<k>" are the readings listed in DESIGN.md
 * section 3 for points the paper leaves open.
 *
 * Conventions
 *   - Every function returns a mori_status (0 = OK, negative = error) unless stated otherwise.
 *   - Argument checks are synchronous: on MORI_ERR_INVALID_ARG nothing has been enqueued.
 *   - Asynchronous CUDA failures surface at mori_sync() as MORI_ERR_CUDA and are sticky.
 *   - "DEVICE" pointers are device memory of the context's GPU; "HOST" pointers are ordinary
 *     host memory read before the call returns (the caller may reuse them at once);
 *     "PINNED" is page-locked host memory mapped into the device address space
 *     (cudaHostAlloc / cudaHostRegister; what torch's pin_memory gives).
 *   - The caller owns the pool, the arena, the page allocator and every array it passes in;
 *     the library owns the context, its streams, events, staging and index buffers.
 *   - One context per GPU; calls on one context must come from one host thread at a time.
 *   - The placement entry points (mori_rank_partition, mori_rank_partition_tiers,
 *     mori_sticky_rebalance, mori_bfd_assign, mori_eviction_order, mori_idleness_*) take a caller
 *     stream and share per-context scratch (last-CTA tickets, order buffers, the eviction sort's
 *     tables): enqueue them on ONE stream at a time; if two streams are used, the caller orders
 *     them (event or join) so that two such launches are never in flight together.
 *   - MORI_DEBUG=1 in the environment of mori_create turns on validation that release builds
 *     leave to the caller: duplicate destination ids (see mori_demote / mori_scatter_pages).
 *   - There is no CPU fallback: without a usable sm_100a device mori_create fails.
 *
 * Layouts (BASELINE.json north_star; the paper only says the cache is paged)
 *   chunk      = 2 (K,V) * n_kv_heads * page_tokens * head_dim * elem_bytes   contiguous bytes
 *                of one (layer, physical page); must be a multiple of 16
 *   gpu_pool   [n_layers][gpu_pool_pages][K/V][kv_heads][page_tokens][head_dim]
 *              byte address of (layer l, page g)  = gpu_pool + (l * gpu_pool_pages + g) * chunk
 *   host_arena [host_arena_slots][n_layers][K/V][kv_heads][page_tokens][head_dim]   (R7)
 *              byte address of (slot h, layer l)  = host_arena + (h * n_layers + l) * chunk
 *   Byte offsets are 64-bit; page ids and slot ids are int32.
 */
#ifndef MORI_H_
#define MORI_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mori_ctx mori_ctx; /* opaque, library-owned */

typedef enum {
  MORI_OK = 0,
  MORI_ERR_INVALID_ARG = -1,
  MORI_ERR_CUDA = -2,
  MORI_ERR_CAPACITY = -3, /* more pages in one call than the context was sized for */
  MORI_ERR_STATE = -4,
  MORI_ERR_UNSUPPORTED = -5
} mori_status;

enum { MORI_TIER_GPU = 0, MORI_TIER_CPU = 1, MORI_TIER_WAIT = 2 };
enum { MORI_DEMOTE = 1, MORI_PROMOTE = 2, MORI_BOTH = 3 };
enum { MORI_LIST_DEMOTE = 0, MORI_LIST_PROMOTE = 1, MORI_LIST_DROP = 2, MORI_LIST_ADMIT = 3,
       MORI_LIST_RESERVE = 4, MORI_N_LISTS = 5 };
/* How KV bytes cross the host link.
 *   ZEROCOPY   one kernel: SMs load pool chunks and store them straight into the mapped arena
 *              (demote), or load from the arena and store into the pool (promote).
 *   STAGED     gather kernel pool -> contiguous device staging at HBM speed, then large
 *              cudaMemcpyAsync DMAs staging -> arena on a copy stream, double-buffered
 *              (promote: DMA arena -> staging, then scatter kernel staging -> pool).
 *   COPYENGINE no kernel: one strided cudaMemcpy2DAsync per logical page (baseline).
 *   AUTO       chosen per call from the slot table: a call of at most 448
 *              pages and 4 MiB is ONE launch of a kernel that carries the page and slot ids in its
 *              parameters and copies straight between the pool and the mapped arena (no index
 *              upload, no staging, no DMA); otherwise STAGED when the runs of consecutive host slots
 *              average >= 6 MiB (large DMAs reach 97-100 % of the measured link peak), ZEROCOPY
 *              below that (a DMA per 2 MiB run reaches 89 %, SM-driven zero-copy 92 % whatever the
 *              fragmentation).  mori_path() reports STAGED. */
enum { MORI_PATH_AUTO = 0, MORI_PATH_ZEROCOPY = 1, MORI_PATH_STAGED = 2, MORI_PATH_COPYENGINE = 3 };
/* Device copy kernel used by STAGED paths and by mori_gather_pages / mori_scatter_pages. */
enum { MORI_KERNEL_AUTO = 0, MORI_KERNEL_LDST = 1, MORI_KERNEL_TMA = 2 };

#define MORI_MAX_PROGRAMS 8192 /* the keys of all programs fit one CTA's shared memory */

typedef struct {
  int32_t n_layers, n_kv_heads, head_dim, page_tokens, elem_bytes; /* bf16 -> elem_bytes 2 */
  void*   gpu_pool;          /* DEVICE, caller-owned, 16-byte aligned */
  int64_t gpu_pool_pages;
  void*   host_arena;        /* PINNED, caller-owned, 16-byte aligned; may be NULL if neither
                                mori_demote nor mori_promote is used.  May instead be DEVICE
                                memory (this GPU's, or a peer GPU's -- mori_create turns peer
                                access on, or fails with MORI_ERR_UNSUPPORTED if the two GPUs are
                                not peers: the intermediate tier of P:L347): both directions then
                                run as one full-grid kernel, path_* are ignored.  A DEVICE arena
                                described as a pool of ONE layer (n_layers = 1, n_kv_heads = L * H:
                                a slot is then one chunk) can in turn be the gpu_pool of a second
                                context whose host_arena is pinned memory: the arena <-> arena
                                mover of a three-tier hierarchy */
  int64_t host_arena_slots;
  int32_t max_programs;      /* 1 .. MORI_MAX_PROGRAMS */
  int32_t path_demote;       /* MORI_PATH_* */
  int32_t path_promote;      /* MORI_PATH_* */
  int32_t copy_kernel;       /* MORI_KERNEL_* */
  int64_t staging_bytes;     /* per staging buffer (2 per direction); 0 -> 2 GiB when the device has
                                >= 32 GiB free at mori_create, 1 GiB when >= 12 GiB, else 256 MiB */
  int64_t max_pages_per_call;/* 0 -> max(gpu_pool_pages, host_arena_slots) */
  int32_t zerocopy_ctas;     /* grid of a ZEROCOPY kernel (it is link-bound, a few CTAs saturate
                                PCIe and the rest of the SMs stay free); 0 -> library default */
  int32_t idleness_window;   /* k of Eq. (1); 0 -> 5 ("we use k=5 in all experiments"); <= 64 */
} mori_config;

/* Creates a context on the CURRENT CUDA device.  *out is NULL on failure. */
int mori_create(const mori_config* cfg, mori_ctx** out);
/* Joins all outstanding work, then frees everything the library owns. */
int mori_destroy(mori_ctx* ctx);

/*
 * Steps a1-a4 of the hot path: rank all active programs by idleness, prefix-sum their KV
 * footprints in rank order, cut the ranking at the GPU and CPU capacities, label the rest
 * WAITING, and list who moves.  One kernel launch on `stream` (a cudaStream_t; NULL = the
 * legacy default stream); returns without waiting.  All pointers are DEVICE pointers.
 *
 *   Order      ascending idleness, rank 0 = busiest (the busier programs
 *              are prioritised for HBM, the most idle go to CPU DRAM).  Equal scores (as floats,
 *              so -0 == +0) rank by program index; NaN ranks after every number (R2, R11, R12).
 *   GPU tier   ranks [0, b_gpu): the longest prefix whose summed kv_pages is <= gpu_cap_pages
 *              ("does not exceed GPU memory capacity"; "filling from the busiest
 *              end of the ranking until local capacity is reached").
 *   CPU tier   ranks [b_gpu, b_cpu): the longest following run whose sum is <= cpu_cap_pages
 *              ("enforced analogously").
 *   WAITING    ranks [b_cpu, n): admitted to neither tier, KV discarded.
 *   Lists      from prev_tier -> tier, each in the order the paper moves programs:
 *                demote  (GPU -> CPU)      most idle first   ("highest idleness first")
 *                promote (CPU -> GPU)      least idle first  ("lowest idleness first")
 *                drop    (GPU|CPU -> WAIT) most idle first
 *                admit   (WAIT -> GPU)     least idle first
 *                reserve (WAIT -> CPU)     least idle first  (label only, no bytes: R9)
 *
 *   n            0 .. max_programs (0 is a valid no-op that still writes bounds/used/counts)
 *   idleness     [n] float32, any value
 *   kv_pages     [n] int32 >= 0 (negative values are treated as 0)
 *   prev_tier    [n] uint8 or NULL; values other than 0 and 1 mean WAITING.  NULL: lists and
 *                list_counts are not written (and may be NULL)
 *   order        [n] out: program at each rank
 *   tier         [n] out: MORI_TIER_* per program
 *   bounds       [2] out: b_gpu, b_cpu
 *   used_pages   [2] out: pages held by the GPU tier, by the CPU tier
 *   lists        [5][n] out: row MORI_LIST_*; entries past list_counts[row] are unspecified
 *   list_counts  [5] out
 * Every output array is written exactly once, by one CTA, and never read back, so the outputs
 * (not the inputs) may also be PINNED host memory: the placement then lands in host memory with
 * no copy, complete when `stream` has run the launch.  Worth it for small n (scattered 4-byte
 * stores cross PCIe one by one); for thousands of programs one device-to-host copy is faster.
 */
int mori_rank_partition(mori_ctx* ctx, void* stream, int32_t n, const float* idleness,
                        const int32_t* kv_pages, const uint8_t* prev_tier, int64_t gpu_cap_pages,
                        int64_t cpu_cap_pages, int32_t* order, uint8_t* tier, int32_t* bounds,
                        int64_t* used_pages, int32_t* lists, int32_t* list_counts);

/*
 * Step a5, demotion ("offloaded to CPU DRAM on the same node"): for every
 * j in [0, total_pages) and every layer l, copy chunk (l, gpu_pages[j]) of the pool to
 * (host_slots[j], l) of the arena.  Asynchronous, on the context's demote stream(s).
 *
 *   gpu_pages, host_slots  HOST int32[total_pages]; ids out of range -> MORI_ERR_INVALID_ARG.
 *                          A destination slot listed twice in one call is undefined behaviour
 *                          (two copies race for the same bytes); with MORI_DEBUG=1 in the
 *                          environment of mori_create it is found on the host before anything is
 *                          enqueued -> MORI_ERR_INVALID_ARG.
 *   wait_promote_ticket    0, or a ticket returned by mori_promote: no byte of this call is read
 *                          or written before that promote call has completed (device-side wait).
 *   ticket_out             receives this call's ticket (> 0, increasing); NULL: no ticket is issued
 *                          (and no event recorded) -- for calls nothing will ever wait on.
 * total_pages == 0 is a valid no-op that still yields a ticket.
 * Calls of one direction take effect in issue order (a later call that writes the same slots or
 * pages wins), whichever path each of them takes; the two directions are ordered only by tickets,
 * and a ticket means the same on every path (ZEROCOPY, STAGED, COPYENGINE, the one-launch path of
 * a small call): what it names has completed before what it gates starts.
 */
int mori_demote(mori_ctx* ctx, int64_t total_pages, const int32_t* gpu_pages,
                const int32_t* host_slots, int64_t wait_promote_ticket, int64_t* ticket_out);

/*
 * Step a6, promotion ("CPU-to-GPU transfer over PCIe"): the mirror image,
 * arena (host_slots[j], l) -> pool (l, gpu_pages[j]), on the promote stream(s), concurrently
 * with demotions.  A promotion touches two resources that a demotion may still be using, so it
 * takes two tickets of mori_demote (0 = none):
 *   pages_after_demote   no byte of the POOL is written before that demotion has completed (the
 *                        demotion that vacates the destination pages);
 *   slots_after_demote   no byte of the ARENA is read before that demotion has completed (a
 *                        demotion that wrote the source slots and has not been joined since).
 * Keeping them apart is what lets a STAGED promotion stream its bytes over the link while the
 * pages it will land in are still being vacated.  Duplicate destination PAGES: as for mori_demote.
 */
int mori_promote(mori_ctx* ctx, int64_t total_pages, const int32_t* host_slots,
                 const int32_t* gpu_pages, int64_t pages_after_demote, int64_t slots_after_demote,
                 int64_t* ticket_out);

/* Step a7: block the host until every demote (1), promote (2) or both (3) call has finished;
 * returns the first asynchronous error if there was one. */
int mori_sync(mori_ctx* ctx, int32_t which);

/* Device-side ordering against a caller stream (cudaStream_t), no host blocking:
 *   mori_after_stream   work enqueued later in direction(s) `which` starts after everything
 *                       now in `stream` (e.g. the inference step that last touched the pages);
 *                       costs one event record: each library stream waits on it only when it
 *                       next gets work, so a direction that stays idle is never touched;
 *   mori_stream_wait    work enqueued later in `stream` starts after everything now enqueued
 *                       in direction(s) `which`. */
int mori_after_stream(mori_ctx* ctx, int32_t which, void* stream);
int mori_stream_wait(mori_ctx* ctx, void* stream, int32_t which);

/*
 * The on-device halves of the STAGED paths, exposed because they are what the HBM roofline is
 * measured on: pool pages <-> a contiguous DEVICE buffer laid out [n_pages][n_layers][chunk].
 * gpu_pages is a DEVICE int32[n_pages].  One launch on `stream`; asynchronous.
 * Ids are device data and are not checked in release.  With MORI_DEBUG=1 a validation kernel
 * runs first on `stream` and the call waits for it (range; for scatter also duplicate pages):
 * a bad table -> MORI_ERR_INVALID_ARG with nothing else enqueued.
 */
int mori_gather_pages(mori_ctx* ctx, void* stream, int64_t n_pages, const int32_t* gpu_pages,
                      void* dst);
int mori_scatter_pages(mori_ctx* ctx, void* stream, int64_t n_pages, const int32_t* gpu_pages,
                       const void* src);

/* ------------------------------------------------------------------------------------------------
 * Beyond the hot path: the steps around it, each with its own oracle.
 * ---------------------------------------------------------------------------------------------- */

/*
 * NEXT-1: the paper's sticky, status-aware tier management, section 4.3.1, as an
 * alternative to mori_rank_partition for callers that track program status.  Nothing moves unless
 * capacity forces or allows it.  One kernel launch on `stream`; DEVICE pointers.
 *
 *   Demotion   only while the GPU queue's pages exceed gpu_cap_pages: Acting programs before
 *              Reasoning ones, the most idle first (equal scores: the later program in
 *              the ranking order of mori_rank_partition is the more idle).  A Reasoning victim
 *              is flagged lazy[p] = 1 ("finishes its current inference step before being
 *              moved").  Each victim, in that order, goes to the CPU queue if its pages still
 *              fit under cpu_cap_pages, else to Waiting.
 *   Promotion  then, while the next candidate fits the GPU (the first that does not fit stops
 *              it), in the priority order of P:L208: (1) CPU-queue programs that are READY,
 *              (2) READY Waiting-queue programs that are not NEW, (3) READY NEW programs smallest
 *              kv_pages first; the least idle first inside a class.  A program demoted by this
 *              call is not a candidate in the same call.
 *
 *   flags        [n] uint8: MORI_FLAG_ACTING (waiting on a tool call; else Reasoning),
 *                MORI_FLAG_READY (a request of it is waiting for inference), MORI_FLAG_NEW (never
 *                held KV: a new arrival)
 *   prev_tier    [n] required; the CPU queue must fit cpu_cap_pages on entry (its programs are
 *                gated and do not grow) -- not checked on the device
 *   tier         [n] out;  lazy [n] out;  used_pages [2] out (GPU queue, CPU queue)
 *   lists        [5][n] out, rows MORI_LIST_*: demote and drop in victim order, promote and admit
 *                in priority order, reserve always empty;  list_counts [5] out
 */
enum { MORI_FLAG_ACTING = 1, MORI_FLAG_READY = 2, MORI_FLAG_NEW = 4 };
int mori_sticky_rebalance(mori_ctx* ctx, void* stream, int32_t n, const float* idleness,
                          const int32_t* kv_pages, const uint8_t* prev_tier, const uint8_t* flags,
                          int64_t gpu_cap_pages, int64_t cpu_cap_pages, uint8_t* tier, uint8_t* lazy,
                          int64_t* used_pages, int32_t* lists, int32_t* list_counts);

/*
 * NEXT-2: the windowed idleness metric, Eq. (1), tracked on the device:
 *     iota = T_acting^(k) / (T_reasoning^(k) + T_acting^(k))   over the last k cycles.
 * The context keeps, per program slot 0 .. max_programs-1, the last k completed
 * (reasoning, acting) duration pairs.  Time a program spent gated by the scheduler is simply never
 * reported.  DEVICE pointers; one launch each on `stream`; asynchronous.
 *
 * mori_idleness_update applies m events in list order (events of one program keep their order):
 *   prog [m] int32 slot;  kind [m] uint8: 0 = a cycle completed with durations
 *   reasoning[e], acting[e] (seconds, double), 1 = the slot was taken by a new program (window
 *   cleared; durations ignored).  Slots out of 0 .. max_programs-1 are ignored.
 * mori_idleness_eval writes idleness_out[p] for p < n: the window is the last k cycles, the
 *   unfinished one -- elapsed open_reasoning[p] + open_acting[p] > 0 -- counted as the newest of
 *   them ("the ongoing tool call's elapsed time keeps increasing and soon dominates");
 *   either open array may be NULL (all zero).  Sums in double, oldest first, open cycle last, one
 *   division, one rounding to float; no time at all -> NaN (which the rankers place last).
 *   idleness_out can be handed to mori_rank_partition / mori_sticky_rebalance on the same stream.
 */
int mori_idleness_update(mori_ctx* ctx, void* stream, int64_t m, const int32_t* prog,
                         const uint8_t* kind, const double* reasoning, const double* acting);
int mori_idleness_eval(mori_ctx* ctx, void* stream, int32_t n, const double* open_reasoning,
                       const double* open_acting, float* idleness_out);

/*
 * NEXT-3: typed eviction order: "The engine's eviction policy remains LRU
 * at its core, but uses the type label as a higher-priority sort key ... the type priority order
 * is reversed between the two tiers":  GPU HBM evicts inactive first, then idle, then busy;
 * CPU DRAM evicts inactive first, then busy, then idle; "within each type, LRU breaks ties".
 * A page's type is its owner's placement: MORI_TIER_GPU busy, MORI_TIER_CPU idle,
 * anything else inactive.  Equal last_access inside a type: lower page id first.
 * DEVICE pointers; asynchronous on `stream`: ONE launch (a cluster of 16 CTAs, 8 where the device does not
 * allow that size) for pools of up to 262 144 (131 072) pages, a fixed sequence of kernels replayed as a CUDA
 * graph beyond that.
 *
 *   which_tier    MORI_TIER_GPU: n_pages <= gpu_pool_pages;  MORI_TIER_CPU: n_pages <= host_arena_slots
 *   page_owner    [n_pages] int32 program slot, or < 0 for a free page (free pages are not listed)
 *   program_tier  [n_programs] uint8 (e.g. the tier array mori_rank_partition wrote)
 *   last_access   [n_pages] uint32, any monotone counter; smaller = less recently used
 *   victims       [n_pages] out: the resident pages, first to evict first, in [0, *n_resident);
 *                 entries past that are the free pages (unspecified order)
 *   n_resident    [1] int32 out
 */
int mori_eviction_order(mori_ctx* ctx, void* stream, int32_t which_tier, int64_t n_pages,
                        const int32_t* page_owner, int32_t n_programs, const uint8_t* program_tier,
                        const uint32_t* last_access, int32_t* victims, int32_t* n_resident);

/*
 * The same order for callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no context, and no cudaMalloc / cudaFree / allocating
 * library routine on any call -- mori_eviction_order allocates its sort scratch on first use, this
 * entry point keeps it in a file-scope static __device__ array instead (2 x MORI_NOALLOC_MAX_PAGES
 * x 8 bytes = 1 MiB, held by every GPU that loads the library until the process exits).
 *
 *   Runs on the CURRENT device, one launch (the cluster kernel of mori_eviction_order) on `stream`;
 *   arguments, order and outputs exactly as mori_eviction_order (which_tier: MORI_TIER_GPU / _CPU).
 *   n_pages      0 .. MORI_NOALLOC_MAX_PAGES; more -> MORI_ERR_CAPACITY, nothing enqueued
 *   why          NULL, or receives a pointer to a static string that says what was wrong (valid for
 *                ever; "" on success)
 * The first call on a device looks the scratch up (cudaGetSymbolAddress) and picks the cluster
 * size: make it outside graph capture (n_pages = 0 does only that).  Every call on a device shares
 * the one scratch array, which keeps the previous call's contents: nothing in it needs to start at
 * zero (each pass overwrites every entry it later reads), but two calls that OVERLAP on the GPU --
 * different streams, no ordering between them -- race on it.  Calls on one stream are safe.
 */
#define MORI_NOALLOC_MAX_PAGES 65536 /* cfg 2's arena, the largest BASELINE.json pool */
int mori_eviction_order_noalloc(void* stream, int32_t which_tier, int64_t n_pages,
                                const int32_t* page_owner, int32_t n_programs,
                                const uint8_t* program_tier, const uint32_t* last_access,
                                int32_t* victims, int32_t* n_resident, const char** why);

/*
 * NEXT-4(i): which replica admits each Waiting-queue promotion: "Waiting-
 * queue promotions use Best-Fit-Decreasing bin packing across replicas, selecting the replica
 * with the most available capacity first" (CPU-queue promotions keep their replica and are not
 * packed).  Every replica runs this on the same inputs -- the shared Waiting queue and
 * the all-gathered free capacities -- and gets the same answer.  DEVICE pointers, one launch.
 *
 *   m            candidates, 0 .. max_programs
 *   size         [m] int32 KV pages;  idleness [m] float;  flags [m] uint8 (MORI_FLAG_NEW used)
 *   n_replicas   1 .. 32;  free_pages [n_replicas] int64 >= 0
 *   replica      [m] out: admitting replica, or -1 = stays in Waiting
 *   free_out     [n_replicas] out: free pages left (may alias free_pages)
 * Order: largest first; equal sizes: returning before new, then least idle, then index.  Each
 * candidate goes to the replica with the most free pages (ties: lowest index) if it fits there,
 * else nowhere; the packing continues with the next candidate.
 */
int mori_bfd_assign(mori_ctx* ctx, void* stream, int32_t m, const int32_t* size, const float* idleness,
                    const uint8_t* flags, int32_t n_replicas, const int64_t* free_pages,
                    int32_t* replica, int64_t* free_out);

/*
 * NEXT-4(ii): the ranking cut by n_tiers capacities instead of two, P:L339-351 ("the
 * design generalizes naturally to more hierarchies ... a second idleness threshold ... an
 * intermediate tier"; "filling from the busiest end of the ranking until local capacity is
 * reached").  Tier t (0 = GPU HBM, then e.g. peer HBM over NVLink, host DRAM, SSD ...) takes the
 * longest run of the ranking right after tier t-1 whose kv_pages fit cap_pages[t]; the rest is
 * Waiting, written as tier value n_tiers.  With n_tiers = 2 this is mori_rank_partition without
 * the move lists.  One launch on `stream`; array pointers are DEVICE pointers.
 *
 *   n_tiers      1 .. 8;  cap_pages  HOST int64[n_tiers], >= 0, read before the call returns
 *   prev_tier    [n] uint8 or NULL (values >= n_tiers mean Waiting); NULL: no move lists
 *   order [n], tier [n], bounds [n_tiers] (end rank of every tier), used_pages [n_tiers]: out
 *   moves        [2][n] out: row 0 the programs that go DOWN the hierarchy (to a slower tier or to
 *                Waiting) most idle first, row 1 those that go UP least idle first -- the order of
 *                P:L206 / L208; from and to are prev_tier[p] and tier[p].  move_counts [2] out
 */
int mori_rank_partition_tiers(mori_ctx* ctx, void* stream, int32_t n, const float* idleness,
                              const int32_t* kv_pages, int32_t n_tiers, const int64_t* cap_pages,
                              const uint8_t* prev_tier, int32_t* order, uint8_t* tier, int32_t* bounds,
                              int64_t* used_pages, int32_t* moves, int32_t* move_counts);

/* Kernel timing for the roofline: while enabled, every gather/scatter kernel launched by
 * mori_demote / mori_promote is bracketed by CUDA events on its stream.  mori_profile_read
 * (call after mori_sync) returns and clears the totals for one direction. */
int mori_profile(mori_ctx* ctx, int32_t enable);
/* enable == 2 additionally keeps a TIMELINE: every kernel (kind 0) and every staging segment's run
 * of DMAs (kind 1) of both directions as [start, end) in milliseconds since the mori_profile call,
 * all on one clock -- the evidence of what overlaps what inside an epoch.  Read it after mori_sync;
 * *n_rows receives the number of rows available (at most max_rows are copied out). */
int mori_profile_timeline(mori_ctx* ctx, int32_t which, int64_t max_rows, int32_t* kind, double* start_ms,
                          double* end_ms, int64_t* bytes, int64_t* n_rows);
int mori_profile_read(mori_ctx* ctx, int32_t which, double* kernel_ms, int64_t* launches,
                      int64_t* bytes);

/* Launches an EMPTY kernel on `stream`: the launch-latency floor that the latency-bound entry
 * points (the rankers, the eviction order, the Waiting-queue packing) are reported against. */
int mori_noop(mori_ctx* ctx, void* stream);

/* Number of CUDA kernels this context has launched since mori_create (rank/partition, index
 * upload, gather/scatter/zero-copy kernels); copy-engine DMAs are not kernels and not counted. */
int mori_launch_count(const mori_ctx* ctx, int64_t* out);

/* PINNED host memory for an arena when the caller has no allocator of its own: page-locked,
 * mapped into the device address space, exactly `bytes` long (no rounding), 2 MiB aligned,
 * zero-filled (transparent-huge-page backed where the kernel allows).
 * *out is NULL on failure (MORI_ERR_CUDA; mori_last_error(NULL) says why).  Free with
 * mori_host_free, after destroying every context that uses it. */
int mori_host_alloc(int64_t bytes, void** out);
int mori_host_free(void* p);

/* Resolved MORI_PATH_* for a direction (after AUTO), and resolved MORI_KERNEL_*. */
int mori_path(const mori_ctx* ctx, int32_t which);
int mori_copy_kernel(const mori_ctx* ctx);

/* Library-owned, NUL-terminated description of the last error on this context (or of the last
 * failed mori_create when ctx is NULL); valid until the next call. */
const char* mori_last_error(const mori_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MORI_H_ */
