/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU statement of what the MORI hot path computes
 * (arxiv/paper_2606_00866; citations "P:Lnnn" are lines of /root/reference/PAPER.md).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this.  It shares no source, header, helper or table with
 * paper_2606_00866_b200/csrc/ and never includes include/mori.h.
 *
 * The method reaches a plainly defined result (a capacity-constrained split of a sorted list,
 * and a byte permutation), so each function below is that definition written out:
 *
 *   oracle_rank_partition      P:L11, L45, L149-152 (rank by relative idleness, busiest -> GPU),
 *                              P:L176-177 (capacity invariants of both tiers),
 *                              P:L147, L178 (admission control; overflow -> Waiting, discarded),
 *                              P:L351 ("filling from the busiest end of the ranking until local
 *                              capacity is reached"), P:L206/L208 (order of the move lists).
 *   oracle_bruteforce_partition  the same result stated WITHOUT a sort or a prefix sum:
 *                              enumeration of all 3^n tier maps (pins the function above).
 *   oracle_demote / oracle_promote   P:L177 ("offloaded to CPU DRAM"), P:L182 ("CPU-to-GPU
 *                              transfer"), P:L184 (reload restores the cache): per-(page, layer)
 *                              memcpy between a paged pool and a page-major arena.
 *
 * Readings of the paper adopted where it is silent are listed in DESIGN.md section 3 (R1..R14);
 * the ones that matter here are repeated next to the code.
 *
 * Further down, each with its own header comment and its own pins file under tests/:
 *   oracle_sticky_rebalance      P:L206, L208 (section 4.3.1)       tests/test_oracle_sticky_pins.py
 *   oracle_idleness_update/eval  Eq. (1), P:L190-196                tests/test_oracle_idleness_pins.py
 *   oracle_eviction_order        P:L212-221 (section 4.3.2)         tests/test_oracle_eviction_pins.py
 *   oracle_bfd_assign            P:L208-210                         tests/test_oracle_bfd_pins.py
 *   oracle_rank_partition_tiers  P:L339-351 (section 7.1)           tests/test_oracle_tiers_pins.py
 *   oracle_move_slots            P:L339-351 (arena <-> arena)       tests/test_oracle_tiers_pins.py
 * Every function is pinned (none is "parity unpinned"); DESIGN.md sections 10 and 12-15 say by what.
 *
 * Pins (tests/test_oracle_pins.py): brute force on n <= 9, numpy stable argsort / cumsum /
 * searchsorted restatement, closed forms (equal sizes, zero and infinite capacity), the
 * ordering / capacity / maximality invariants, list set identities, and for the movers the
 * numpy fancy-index gather and the demote->promote round trip.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)

enum { TIER_GPU = 0, TIER_CPU = 1, TIER_WAIT = 2 };

/* Total order on programs (R1, R2, R11, R12):
 *   a before b  iff  iota_a < iota_b, or they compare equal as floats (so -0 == +0) and a < b.
 *   NaN is greater than every non-NaN; NaNs tie among themselves (then by index).
 * Rank 0 is the LEAST idle (busiest) program: it is the first to get GPU HBM. */
typedef struct { float iota; int32_t idx; } prog_key;

static int is_nan_f(float x) { return x != x; }

static int before(const prog_key *a, const prog_key *b) {
  int na = is_nan_f(a->iota), nb = is_nan_f(b->iota);
  if (na != nb) return nb;              /* the non-NaN one comes first */
  if (!na) {
    if (a->iota < b->iota) return 1;
    if (b->iota < a->iota) return 0;
  }
  return a->idx < b->idx;
}

static int cmp_keys(const void *pa, const void *pb) {
  const prog_key *a = (const prog_key *)pa, *b = (const prog_key *)pb;
  if (before(a, b)) return -1;
  if (before(b, a)) return 1;
  return 0;                              /* only for a == b: the order is total */
}

/*
 * Placement.  Inputs: iota[n] (any float), s[n] (KV footprint in pages, >= 0), prev_tier[n] or
 * NULL, capacities in pages (>= 0).  Outputs (each may be NULL except order/tier):
 *   order[r]      program at rank r
 *   tier[p]       0 GPU, 1 CPU, 2 WAIT, indexed by program
 *   bounds[2]     b_gpu, b_cpu: GPU tier = ranks [0,b_gpu), CPU tier = ranks [b_gpu,b_cpu)
 *   used[2]       pages held by the GPU tier and by the CPU tier
 *   lists[5*n]    row 0 demote  (prev GPU -> CPU)  most idle first  ("highest idleness first")
 *                 row 1 promote (prev CPU -> GPU)  least idle first ("lowest idleness first")
 *                 row 2 drop    (prev GPU|CPU -> WAIT) most idle first
 *                 row 3 admit   (prev WAIT -> GPU) least idle first
 *                 row 4 reserve (prev WAIT -> CPU) least idle first
 *   counts[5]     lengths of the rows.  prev_tier values other than 0 and 1 mean WAIT.
 */
int oracle_rank_partition(int32_t n, const float *iota, const int32_t *s, const uint8_t *prev_tier,
                          int64_t cap_gpu, int64_t cap_cpu, int32_t *order, uint8_t *tier,
                          int32_t *bounds, int64_t *used, int32_t *lists, int32_t *counts) {
  if (n < 0 || cap_gpu < 0 || cap_cpu < 0) return ORACLE_ERR_ARG;
  if (n > 0 && (!iota || !s || !order || !tier)) return ORACLE_ERR_ARG;
  for (int32_t p = 0; p < n; ++p) if (s[p] < 0) return ORACLE_ERR_ARG;

  /* step 1: sort by the total order (library routine; the comparator is total, so no
   * stability is needed) */
  prog_key *keys = (prog_key *)malloc(sizeof(prog_key) * (size_t)(n > 0 ? n : 1));
  if (!keys) return ORACLE_ERR_ARG;
  for (int32_t p = 0; p < n; ++p) { keys[p].iota = iota[p]; keys[p].idx = p; }
  qsort(keys, (size_t)n, sizeof(prog_key), cmp_keys);
  for (int32_t r = 0; r < n; ++r) order[r] = keys[r].idx;
  free(keys);

  /* step 2: GPU tier = the longest prefix of the ranking whose footprint does not exceed the
   * GPU capacity ("does not exceed" -> <=; P:L351 stop at the first that does not fit) */
  int32_t b_gpu = 0; int64_t sum_gpu = 0;
  while (b_gpu < n && sum_gpu + s[order[b_gpu]] <= cap_gpu) { sum_gpu += s[order[b_gpu]]; ++b_gpu; }

  /* step 3: CPU tier = the longest run after it that fits the CPU capacity ("enforced
   * analogously"; "CPU queue if CPU capacity permits, or to the Waiting queue otherwise") */
  int32_t b_cpu = b_gpu; int64_t sum_cpu = 0;
  while (b_cpu < n && sum_cpu + s[order[b_cpu]] <= cap_cpu) { sum_cpu += s[order[b_cpu]]; ++b_cpu; }

  /* step 4: the rest is not admitted anywhere */
  for (int32_t r = 0; r < n; ++r)
    tier[order[r]] = (uint8_t)(r < b_gpu ? TIER_GPU : (r < b_cpu ? TIER_CPU : TIER_WAIT));

  if (bounds) { bounds[0] = b_gpu; bounds[1] = b_cpu; }
  if (used) { used[0] = sum_gpu; used[1] = sum_cpu; }

  /* step 5: transition lists */
  if (prev_tier && lists && counts) {
    for (int k = 0; k < 5; ++k) counts[k] = 0;
    /* ascending rank = least idle first */
    for (int32_t r = 0; r < n; ++r) {
      int32_t p = order[r];
      int was = prev_tier[p] == 0 ? TIER_GPU : (prev_tier[p] == 1 ? TIER_CPU : TIER_WAIT);
      int now = tier[p];
      if (was == TIER_CPU && now == TIER_GPU) lists[1 * (size_t)n + counts[1]++] = p;
      if (was == TIER_WAIT && now == TIER_GPU) lists[3 * (size_t)n + counts[3]++] = p;
      if (was == TIER_WAIT && now == TIER_CPU) lists[4 * (size_t)n + counts[4]++] = p;
    }
    /* descending rank = most idle first */
    for (int32_t r = n - 1; r >= 0; --r) {
      int32_t p = order[r];
      int was = prev_tier[p] == 0 ? TIER_GPU : (prev_tier[p] == 1 ? TIER_CPU : TIER_WAIT);
      int now = tier[p];
      if (was == TIER_GPU && now == TIER_CPU) lists[0 * (size_t)n + counts[0]++] = p;
      if (was != TIER_WAIT && now == TIER_WAIT) lists[2 * (size_t)n + counts[2]++] = p;
    }
  }
  return ORACLE_OK;
}

/*
 * The same placement with no sort and no prefix sum (n <= 12).  Enumerate every map
 * t: programs -> {GPU, CPU, WAIT}; keep those with
 *   (i)   sum of s over t = GPU  <= cap_gpu
 *   (ii)  sum of s over t = CPU  <= cap_cpu
 *   (iii) t(a) < t(b)  =>  a is before b in the total order              (every
 *         GPU-tier program is busier than every CPU-tier program, and so on down)
 * and return the one that maximises (|GPU tier|, then |CPU tier|) -- "filling each tier to
 * capacity".  *n_best receives how many maps attain the maximum (must be 1).
 */
int oracle_bruteforce_partition(int32_t n, const float *iota, const int32_t *s, int64_t cap_gpu,
                                int64_t cap_cpu, uint8_t *tier, int32_t *bounds, int32_t *n_best) {
  if (n < 0 || n > 12 || cap_gpu < 0 || cap_cpu < 0) return ORACLE_ERR_ARG;
  long total = 1;
  for (int i = 0; i < n; ++i) total *= 3;
  int best_g = -1, best_c = -1, ties = 0;
  uint8_t t[12], best_t[12];
  memset(best_t, 0, sizeof best_t);
  for (long code = 0; code < total; ++code) {
    long c = code; int64_t sg = 0, sc = 0; int ng = 0, nc = 0;
    for (int p = 0; p < n; ++p) {
      t[p] = (uint8_t)(c % 3); c /= 3;
      if (t[p] == TIER_GPU) { sg += s[p]; ++ng; }
      if (t[p] == TIER_CPU) { sc += s[p]; ++nc; }
    }
    if (sg > cap_gpu || sc > cap_cpu) continue;
    int ok = 1;
    for (int a = 0; a < n && ok; ++a)
      for (int b = 0; b < n; ++b)
        if (t[a] < t[b]) {
          prog_key ka = { iota[a], a }, kb = { iota[b], b };
          if (!before(&ka, &kb)) { ok = 0; break; }
        }
    if (!ok) continue;
    if (ng > best_g || (ng == best_g && nc > best_c)) {
      best_g = ng; best_c = nc; ties = 1; memcpy(best_t, t, sizeof t);
    } else if (ng == best_g && nc == best_c) {
      ++ties;
    }
  }
  for (int p = 0; p < n; ++p) tier[p] = best_t[p];
  if (bounds) { bounds[0] = best_g; bounds[1] = best_g + best_c; }
  if (n_best) *n_best = ties;
  return ORACLE_OK;
}

/*
 * KV movement.  chunk = 2 (K,V) * kv_heads * page_tokens * head_dim * elem_bytes is the
 * contiguous run of one (layer, physical page) in the device pool, whose layout is
 * [layers][pool_pages][K/V][kv_heads][page_tokens][head_dim] (BASELINE.json north_star; the
 * paper only says the cache is paged).  The host arena is page-major:
 * [slots][layers][K/V][kv_heads][page_tokens][head_dim] (R7).
 *   pool  address of (layer l, page g)  = pool  + (l * pool_pages + g) * chunk
 *   arena address of (slot h, layer l)  = arena + (h * n_layers  + l) * chunk
 * Whole pages always move, all layers, K and V ("exactly one tier"; R8).
 */
int oracle_demote(int32_t n_layers, int64_t chunk, const uint8_t *pool, int64_t pool_pages,
                  uint8_t *arena, int64_t arena_slots, int64_t total_pages,
                  const int32_t *gpu_pages, const int32_t *host_slots) {
  if (n_layers <= 0 || chunk <= 0 || total_pages < 0) return ORACLE_ERR_ARG;
  for (int64_t j = 0; j < total_pages; ++j) {
    int64_t g = gpu_pages[j], h = host_slots[j];
    if (g < 0 || g >= pool_pages || h < 0 || h >= arena_slots) return ORACLE_ERR_ARG;
    for (int64_t l = 0; l < n_layers; ++l)
      memcpy(arena + (h * n_layers + l) * chunk, pool + (l * pool_pages + g) * chunk, (size_t)chunk);
  }
  return ORACLE_OK;
}

int oracle_promote(int32_t n_layers, int64_t chunk, uint8_t *pool, int64_t pool_pages,
                   const uint8_t *arena, int64_t arena_slots, int64_t total_pages,
                   const int32_t *host_slots, const int32_t *gpu_pages) {
  if (n_layers <= 0 || chunk <= 0 || total_pages < 0) return ORACLE_ERR_ARG;
  for (int64_t j = 0; j < total_pages; ++j) {
    int64_t g = gpu_pages[j], h = host_slots[j];
    if (g < 0 || g >= pool_pages || h < 0 || h >= arena_slots) return ORACLE_ERR_ARG;
    for (int64_t l = 0; l < n_layers; ++l)
      memcpy(pool + (l * pool_pages + g) * chunk, arena + (h * n_layers + l) * chunk, (size_t)chunk);
  }
  return ORACLE_OK;
}

/*
 * NEXT-4(ii): with "an intermediate tier" between GPU HBM and host DRAM a
 * program can also move between two page-major arenas.  A slot is one whole logical page (all
 * layers, K and V: page_bytes = n_layers * chunk, contiguous), so the move is one memcpy per page:
 *   dst + dst_slots[j] * page_bytes  <-  src + src_slots[j] * page_bytes.
 * Pinned by tests/test_oracle_tiers_pins.py (byte-by-byte loop, fancy-index restatement, and the
 * reduction of a three-pool epoch with an empty middle tier to the two-pool epochs).
 */
int oracle_move_slots(int64_t page_bytes, const uint8_t *src, int64_t src_slots_n, uint8_t *dst,
                      int64_t dst_slots_n, int64_t total_pages, const int32_t *src_slots,
                      const int32_t *dst_slots) {
  if (page_bytes <= 0 || total_pages < 0) return ORACLE_ERR_ARG;
  for (int64_t j = 0; j < total_pages; ++j) {
    int64_t a = src_slots[j], b = dst_slots[j];
    if (a < 0 || a >= src_slots_n || b < 0 || b >= dst_slots_n) return ORACLE_ERR_ARG;
    memcpy(dst + b * page_bytes, src + a * page_bytes, (size_t)page_bytes);
  }
  return ORACLE_OK;
}

/*
 * NEXT-1: the paper's sticky, status-aware tier management, section 4.3.1, followed
 * step by step in the paper's order.  Nothing moves unless capacity forces or allows it
 * ("programs are not eagerly reshuffled on every tick").
 *
 *   flags[p] bit 0  ACTING   the program waits on a tool call (else REASONING)
 *            bit 1  READY    a CPU- or Waiting-queue program whose request is waiting for inference
 *            bit 2  NEW      a Waiting-queue program that never held KV ("new arrival")
 *
 * Demotion from GPU: "When the aggregate KV cache of GPU-queue programs exceeds GPU
 *   memory capacity, the scheduler demotes programs until usage fits within the budget ...
 *   prioritizes demoting Acting programs ... over Reasoning programs ... Among programs of the
 *   same status, it selects the one with the highest idleness first ... If only Reasoning
 *   programs remain, the scheduler applies lazy demotion ... Demoted programs move to the CPU
 *   queue if CPU capacity permits, or to the Waiting queue otherwise."
 * Promotion to GPU: "When GPU capacity becomes available, the scheduler promotes
 *   programs in a priority order: (1) CPU-queue programs that have completed their tool call and
 *   are waiting for inference; (2) Waiting-queue programs that are waiting for inference, with
 *   returning programs preferred over new arrivals; (3) newly arrived programs, smallest context
 *   first.  Within each priority level ... the lowest idleness first."
 *
 * Readings (S1..S6): equal idleness resolves by the same total order as the ranking
 * (the later program in that order is "more idle"); class 3 orders by (size, then that order);
 * promotion stops at the first candidate that does not fit (head of line, like R3); a program
 * demoted in this tick is not a promotion candidate in the same tick; the CPU queue must fit
 * its capacity on entry (its programs are gated and do not grow) -- violated: ORACLE_ERR_ARG;
 * no Waiting -> CPU move exists in this mode.
 *
 * Outputs: tier[n]; lazy[n] (1 = Reasoning victim, moves after its current step); used[2];
 * lists[5*n] rows demote (GPU->CPU, victim order), promote (CPU->GPU, priority order),
 * drop (GPU->WAIT, victim order), admit (WAIT->GPU, priority order), reserve (always empty);
 * counts[5].
 */
enum { FLAG_ACTING = 1, FLAG_READY = 2, FLAG_NEW = 4 };

int oracle_sticky_rebalance(int32_t n, const float *iota, const int32_t *s, const uint8_t *prev_tier,
                            const uint8_t *flags, int64_t cap_gpu, int64_t cap_cpu, uint8_t *tier,
                            uint8_t *lazy, int64_t *used, int32_t *lists, int32_t *counts) {
  if (n < 0 || cap_gpu < 0 || cap_cpu < 0) return ORACLE_ERR_ARG;
  if (n > 0 && (!iota || !s || !prev_tier || !flags || !tier || !lazy || !lists)) return ORACLE_ERR_ARG;
  if (!counts || !used) return ORACLE_ERR_ARG;
  int64_t usage_gpu = 0, usage_cpu = 0;
  for (int32_t p = 0; p < n; ++p) {
    if (s[p] < 0) return ORACLE_ERR_ARG;
    tier[p] = (uint8_t)(prev_tier[p] == 0 ? TIER_GPU : (prev_tier[p] == 1 ? TIER_CPU : TIER_WAIT));
    lazy[p] = 0;
    if (tier[p] == TIER_GPU) usage_gpu += s[p];
    if (tier[p] == TIER_CPU) usage_cpu += s[p];
  }
  if (usage_cpu > cap_cpu) return ORACLE_ERR_ARG;
  for (int k = 0; k < 5; ++k) counts[k] = 0;

  /* ---- demotion from GPU, one victim at a time ---- */
  while (usage_gpu > cap_gpu) {
    int32_t v = -1;
    for (int32_t p = 0; p < n; ++p) {
      if (tier[p] != TIER_GPU) continue;
      if (v < 0) { v = p; continue; }
      int ap = (flags[p] & FLAG_ACTING) != 0, av = (flags[v] & FLAG_ACTING) != 0;
      if (ap != av) { if (ap) v = p; continue; }           /* Acting before Reasoning */
      prog_key kp = { iota[p], p }, kv = { iota[v], v };
      if (before(&kv, &kp)) v = p;                          /* highest idleness first */
    }
    if (v < 0) break;                                       /* nothing left to demote */
    if (!(flags[v] & FLAG_ACTING)) lazy[v] = 1;             /* only Reasoning remain: lazy demotion */
    usage_gpu -= s[v];
    if (usage_cpu + s[v] <= cap_cpu) {                      /* CPU queue if capacity permits */
      tier[v] = TIER_CPU; usage_cpu += s[v];
      lists[0 * (size_t)n + counts[0]++] = v;
    } else {                                                /* Waiting queue otherwise */
      tier[v] = TIER_WAIT;
      lists[2 * (size_t)n + counts[2]++] = v;
    }
  }

  /* ---- promotion to GPU, in priority order, while it fits ---- */
  uint8_t *seen = (uint8_t *)calloc((size_t)(n > 0 ? n : 1), 1);
  if (!seen) return ORACLE_ERR_ARG;
  for (;;) {
    int32_t c = -1; int cls_c = 0;
    for (int32_t p = 0; p < n; ++p) {
      if (seen[p] || !(flags[p] & FLAG_READY)) continue;
      int cls;
      if (prev_tier[p] == 1) cls = 1;                                   /* CPU queue, ready        */
      else if (prev_tier[p] != 0) cls = (flags[p] & FLAG_NEW) ? 3 : 2;  /* Waiting: returning, new */
      else continue;                                                    /* was on GPU this tick    */
      int better;
      if (c < 0) better = 1;
      else if (cls != cls_c) better = cls < cls_c;
      else {
        prog_key kp = { iota[p], p }, kc = { iota[c], c };
        if (cls == 3 && s[p] != s[c]) better = s[p] < s[c];             /* smallest context first  */
        else better = before(&kp, &kc);                                 /* lowest idleness first   */
      }
      if (better) { c = p; cls_c = cls; }
    }
    if (c < 0) break;
    seen[c] = 1;
    if (usage_gpu + s[c] > cap_gpu) break;                  /* head of line does not fit: stop */
    usage_gpu += s[c];
    if (cls_c == 1) { usage_cpu -= s[c]; lists[1 * (size_t)n + counts[1]++] = c; }
    else lists[3 * (size_t)n + counts[3]++] = c;
    tier[c] = TIER_GPU;
  }
  free(seen);
  used[0] = usage_gpu; used[1] = usage_cpu;
  return ORACLE_OK;
}

/*
 * NEXT-2: the windowed idleness metric, Eq. (1), P:L190-194:
 *     iota = T_acting^(k) / (T_reasoning^(k) + T_acting^(k))
 * "the total time spent in each status over the last k inference--tool-call cycles (we use k=5)".
 * Gated time never enters either sum: the caller simply does not report it.
 * The unfinished cycle counts with its elapsed time ("the ongoing tool call's elapsed time keeps
 * increasing and soon dominates the other terms in the window"): when it has any elapsed
 * time it is the newest of the k cycles (R19).
 *
 * State per program, kept here in the plainest form: hist_r / hist_a [n][k] hold the completed
 * cycles oldest first, cnt[n] how many (<= k).  A push on a full window drops the oldest.
 * Precision (the paper is silent; R20): sums in double, oldest cycle first, the open
 * cycle last; one division; one rounding to float.  No completed and no open time -> NaN.
 */
int oracle_idleness_update(int32_t k, double *hist_r, double *hist_a, int32_t *cnt, int32_t n,
                           int64_t m, const int32_t *prog, const uint8_t *kind,
                           const double *reasoning, const double *acting) {
  if (k <= 0 || n < 0 || m < 0) return ORACLE_ERR_ARG;
  for (int64_t e = 0; e < m; ++e) {
    int32_t p = prog[e];
    if (p < 0 || p >= n) return ORACLE_ERR_ARG;
    double *hr = hist_r + (size_t)p * k, *ha = hist_a + (size_t)p * k;
    if (kind[e] == 1) { cnt[p] = 0; continue; }             /* a fresh program took this slot */
    if (cnt[p] == k) {                                      /* window slides: oldest cycle leaves */
      memmove(hr, hr + 1, sizeof(double) * (size_t)(k - 1));
      memmove(ha, ha + 1, sizeof(double) * (size_t)(k - 1));
      cnt[p] = k - 1;
    }
    hr[cnt[p]] = reasoning[e]; ha[cnt[p]] = acting[e]; cnt[p] += 1;
  }
  return ORACLE_OK;
}

int oracle_idleness_eval(int32_t k, const double *hist_r, const double *hist_a, const int32_t *cnt,
                         int32_t n, const double *open_r, const double *open_a, float *iota) {
  if (k <= 0 || n < 0) return ORACLE_ERR_ARG;
  for (int32_t p = 0; p < n; ++p) {
    double orr = open_r ? open_r[p] : 0.0, oa = open_a ? open_a[p] : 0.0;
    int open = (orr + oa) > 0.0;
    int take = open ? k - 1 : k;                            /* the open cycle is one of the k */
    if (take > cnt[p]) take = cnt[p];
    double tr = 0.0, ta = 0.0;
    for (int32_t i = cnt[p] - take; i < cnt[p]; ++i) {
      tr += hist_r[(size_t)p * k + i];
      ta += hist_a[(size_t)p * k + i];
    }
    if (open) { tr += orr; ta += oa; }
    iota[p] = (tr + ta == 0.0) ? (float)(0.0 / 0.0) : (float)(ta / (tr + ta));
  }
  return ORACLE_OK;
}

/*
 * NEXT-3: typed eviction order.  "The engine's eviction policy remains
 * LRU at its core, but uses the type label as a higher-priority sort key.  Crucially, the type
 * priority order is reversed between the two tiers":
 *     GPU HBM : evicts inactive first, then idle, then busy
 *     CPU DRAM: evicts inactive first, then busy, then idle
 * "Within each type, LRU breaks ties."  The label of a page is its program's placement
 * (P:L214): GPU queue -> busy, CPU queue -> idle, Waiting queue -> inactive.
 *
 *   which_tier     0: order the pages of the GPU pool, 1: of the CPU pool
 *   page_owner[j]  program that owns physical page j, or -1 if the page is free (not listed)
 *   program_tier   [n_programs] 0 GPU / 1 CPU / anything else Waiting
 *   last_access[j] time of last use (any monotone counter); smaller = less recently used
 *   victims        out: the resident pages, first to evict first; *n_resident their number
 * Reading (E1): equal last_access inside a type -> lower page id first.
 */
typedef struct { int32_t prio; uint32_t last; int32_t page; } evict_key;

static int cmp_evict(const void *pa, const void *pb) {
  const evict_key *a = (const evict_key *)pa, *b = (const evict_key *)pb;
  if (a->prio != b->prio) return a->prio < b->prio ? -1 : 1;
  if (a->last != b->last) return a->last < b->last ? -1 : 1;
  return a->page < b->page ? -1 : (a->page > b->page ? 1 : 0);
}

int oracle_eviction_order(int32_t which_tier, int64_t n_pages, const int32_t *page_owner,
                          int32_t n_programs, const uint8_t *program_tier, const uint32_t *last_access,
                          int32_t *victims, int64_t *n_resident) {
  if ((which_tier != 0 && which_tier != 1) || n_pages < 0 || n_programs < 0 || !n_resident) return ORACLE_ERR_ARG;
  evict_key *keys = (evict_key *)malloc(sizeof(evict_key) * (size_t)(n_pages > 0 ? n_pages : 1));
  if (!keys) return ORACLE_ERR_ARG;
  int64_t r = 0;
  for (int64_t j = 0; j < n_pages; ++j) {
    int32_t o = page_owner[j];
    if (o < 0) continue;                                       /* free page */
    if (o >= n_programs) { free(keys); return ORACLE_ERR_ARG; }
    int t = program_tier[o];
    int busy = t == 0, idle = t == 1;                          /* else inactive */
    int prio;
    if (!busy && !idle) prio = 0;                              /* inactive goes first in both tiers */
    else if (which_tier == 0) prio = idle ? 1 : 2;             /* GPU HBM : idle, then busy */
    else prio = busy ? 1 : 2;                                  /* CPU DRAM: busy, then idle */
    keys[r].prio = prio; keys[r].last = last_access[j]; keys[r].page = (int32_t)j; ++r;
  }
  qsort(keys, (size_t)r, sizeof(evict_key), cmp_evict);
  for (int64_t i = 0; i < r; ++i) victims[i] = keys[i].page;
  free(keys);
  *n_resident = r;
  return ORACLE_OK;
}

/*
 * NEXT-4(i): placement of Waiting-queue promotions across replicas, P:L208-210:
 * "For multi-replica deployments, Waiting-queue promotions use Best-Fit-Decreasing bin packing
 * across replicas, selecting the replica with the most available capacity first, while
 * CPU-queue promotions preserve replica affinity" (so only Waiting-queue programs are packed;
 * the single Waiting queue is shared by all replicas).
 *
 *   size[m], iota[m], flags[m]   the READY Waiting-queue candidates (FLAG_NEW marks new arrivals)
 *   free_pages[R]                GPU pages each replica has free after its own demotions and
 *                                CPU-queue promotions (all-gathered from the replicas)
 *   replica[m] out               the replica that admits the candidate, or -1: stays in Waiting
 *   free_out[R] out              what is left
 * Readings (B1..B3): "decreasing" = by size, largest first; equal sizes keep the
 * promotion priority of P:L208 (returning before new, then the least idle, then the index);
 * the chosen replica is the one with the MOST free pages (ties: lowest replica index); a
 * candidate that does not fit there fits nowhere and stays in Waiting, and the packing goes on
 * with the next (smaller) candidate.
 */
typedef struct { int32_t size; int cls; float iota; int32_t idx; } bfd_key;

static int cmp_bfd(const void *pa, const void *pb) {
  const bfd_key *a = (const bfd_key *)pa, *b = (const bfd_key *)pb;
  if (a->size != b->size) return a->size > b->size ? -1 : 1;        /* decreasing size */
  if (a->cls != b->cls) return a->cls < b->cls ? -1 : 1;            /* returning before new */
  prog_key ka = { a->iota, a->idx }, kb = { b->iota, b->idx };
  if (before(&ka, &kb)) return -1;
  if (before(&kb, &ka)) return 1;
  return 0;
}

int oracle_bfd_assign(int32_t m, const int32_t *size, const float *iota, const uint8_t *flags,
                      int32_t n_replicas, const int64_t *free_pages, int32_t *replica, int64_t *free_out) {
  if (m < 0 || n_replicas < 1 || !free_pages || !free_out) return ORACLE_ERR_ARG;
  for (int32_t r = 0; r < n_replicas; ++r) { if (free_pages[r] < 0) return ORACLE_ERR_ARG; free_out[r] = free_pages[r]; }
  bfd_key *keys = (bfd_key *)malloc(sizeof(bfd_key) * (size_t)(m > 0 ? m : 1));
  if (!keys) return ORACLE_ERR_ARG;
  for (int32_t i = 0; i < m; ++i) {
    if (size[i] < 0) { free(keys); return ORACLE_ERR_ARG; }
    keys[i].size = size[i]; keys[i].cls = (flags[i] & FLAG_NEW) ? 1 : 0; keys[i].iota = iota[i]; keys[i].idx = i;
  }
  qsort(keys, (size_t)m, sizeof(bfd_key), cmp_bfd);
  for (int32_t k = 0; k < m; ++k) {
    int32_t best = 0;
    for (int32_t r = 1; r < n_replicas; ++r) if (free_out[r] > free_out[best]) best = r;   /* most available */
    if (keys[k].size <= free_out[best]) { replica[keys[k].idx] = best; free_out[best] -= keys[k].size; }
    else replica[keys[k].idx] = -1;
  }
  free(keys);
  return ORACLE_OK;
}

/*
 * NEXT-4(ii): more offloading tiers: "the design generalizes naturally to
 * more hierarchies ... introducing a second idleness threshold: programs with iota between the
 * two thresholds would be offloaded to [the next tier] ... treating remote DRAM as an
 * intermediate tier".  The same rule as oracle_rank_partition with T capacities instead of two:
 * tier t takes the longest run of the ranking, right after tier t-1, that fits cap[t]
 * ("filling from the busiest end of the ranking until local capacity is reached");
 * what is left is Waiting (tier value T).
 */
int oracle_rank_partition_tiers(int32_t n, const float *iota, const int32_t *s, int32_t n_tiers,
                                const int64_t *cap, const uint8_t *prev_tier, int32_t *order,
                                uint8_t *tier, int32_t *bounds, int64_t *used, int32_t *moves,
                                int32_t *move_counts) {
  if (n < 0 || n_tiers < 1 || n_tiers > 8 || !cap) return ORACLE_ERR_ARG;
  for (int t = 0; t < n_tiers; ++t) if (cap[t] < 0) return ORACLE_ERR_ARG;
  for (int32_t p = 0; p < n; ++p) if (s[p] < 0) return ORACLE_ERR_ARG;
  prog_key *keys = (prog_key *)malloc(sizeof(prog_key) * (size_t)(n > 0 ? n : 1));
  if (!keys) return ORACLE_ERR_ARG;
  for (int32_t p = 0; p < n; ++p) { keys[p].iota = iota[p]; keys[p].idx = p; }
  qsort(keys, (size_t)n, sizeof(prog_key), cmp_keys);
  for (int32_t r = 0; r < n; ++r) order[r] = keys[r].idx;
  free(keys);
  int32_t b = 0;
  for (int t = 0; t < n_tiers; ++t) {
    int64_t sum = 0;
    while (b < n && sum + s[order[b]] <= cap[t]) { sum += s[order[b]]; tier[order[b]] = (uint8_t)t; ++b; }
    bounds[t] = b; used[t] = sum;
  }
  for (int32_t r = b; r < n; ++r) tier[order[r]] = (uint8_t)n_tiers;
  /* move lists, the two-tier rule of P:L206 / L208 carried over: programs that go DOWN the
   * hierarchy (to a slower tier or to Waiting) most idle first, programs that go UP least idle
   * first; prev_tier values >= n_tiers mean Waiting. */
  if (prev_tier && moves && move_counts) {
    move_counts[0] = move_counts[1] = 0;
    for (int32_t r = n - 1; r >= 0; --r) {
      int32_t p = order[r]; int was = prev_tier[p] < n_tiers ? prev_tier[p] : n_tiers;
      if (tier[p] > was) moves[0 * (size_t)n + move_counts[0]++] = p;
    }
    for (int32_t r = 0; r < n; ++r) {
      int32_t p = order[r]; int was = prev_tier[p] < n_tiers ? prev_tier[p] : n_tiers;
      if (tier[p] < was) moves[1 * (size_t)n + move_counts[1]++] = p;
    }
  }
  return ORACLE_OK;
}
