// gq/detail/ring.cuh — the bounded inner ring of G-LFQ and of G-WFQ's fast path.
//
// PAPER.md §III-B (L88-89): "a ring of size 2n, a threshold check for empty ... Each slot is
// a single 64-bit word ... monotonically increasing Head and Tail counters, a Threshold used
// by empty dequeues, and the entry array itself."  Algorithm 1 (L143-211): TRYENQ, TRYDEQ.
// SLOT(t) = t mod 2N, CYCLE(t) = floor(t / 2N) mod 2^bc (L107).  The ring is sized by
// N = max(n, pow2ceil(k)) so that k <= N holds for any thread count (reading G1).
//
// sm_100a layout (reading G13): entries are dense 8-byte words with no cache remap, so the
// 32 consecutive tickets of one warp_faa batch touch 256 contiguous bytes (8 sectors, 2 lines)
// and are served by one coalesced L2 request per instruction; Head, Tail and Threshold each
// sit on their own 1 KiB-strided line so that the three hot words never share an L2 slice
// queue.  `slot_shift` spreads entries over 32 B / 128 B for the padding ablation.
#pragma once
#include "prim.cuh"

namespace gq {

struct RingView {
  uint64_t* entry;      // 2N slots, stride 8 << slot_shift bytes
  uint64_t* head;       // packed per format (counter << kCtrShift | ThrIdx)
  uint64_t* tail;
  int64_t*  threshold;  // signed; reset value 3N-1
  uint64_t* owner;      // G-WFQ only: Owner[2N] side table (reading W6); else nullptr
  void*     rec;        // G-WFQ only: WfqRecord[k] of this ring; else nullptr
  int64_t   thr_reset;  // 3N-1
  uint32_t  order;      // log2(2N)
  uint32_t  slot_shift; // 0 dense, 2 = 32 B, 4 = 128 B
  uint32_t  park_ns;    // D2: longest time a dequeuer waits on its own vacant slot (0 = never)
  uint32_t  park_limit; // D1: EMPTY without a ticket once Head is this far ahead of Tail
  uint32_t  park_nap;   // D2: longest single __nanosleep between two looks at the parked slot
  uint32_t  prefetch;   // > 0: rings too large to stay L2-resident: pull the slot `prefetch` tickets ahead into L2
  uint32_t  id;         // 0 = AQ (or the only ring), 1 = FQ: names the ring in traces and latency probes (debug.cuh)
  uint32_t  spin_ns;    // D2: a parked dequeuer re-reads its slot without any nap for this long, then backs off
  uint32_t  slow_nap;   // G-WFQ: longest nap of a thread that lost a SLOWFAA round, ns (<= 1024: Backoff's own ladder only)
  uint32_t  _pad0;
  detail::BlockFunnel* fhead;   // block-level ticket funnels of the calling block (shared memory; D11), or nullptr:
  detail::BlockFunnel* ftail;   // set by the kernel on its own copy of the view (with_funnels, queue.cuh)
};

namespace detail {

enum : int { RING_OK = 0, RING_EMPTY = 1, RING_RETRY = 2, RING_PENDING = 3 };
// A dequeue attempt that waits in line (D2) without blocking its caller: try_deq hands the wait back (RING_PENDING) with the
// ticket it holds, and the caller comes back later with the same record; the parking budget (park_ns) then runs in real
// time (%globaltimer) from the first look at the vacant slot.  The holder of a ticket MUST come back until the attempt ends
// otherwise: the enqueuer that draws the same ticket will install an item for it.
struct DeqWait {
  uint64_t ticket = 0;
  uint64_t since = 0;      // %globaltimer of the first look at the vacant slot; 0 = no attempt pending
  __device__ __forceinline__ bool pending() const { return since != 0; }
  __device__ __forceinline__ void clear() { since = 0; }
};
// GQ_F_* bits of gq.h that reach the device (kept numerically identical)
enum : uint32_t { kPerLaneFaa = 1u, kNoProbe = 2u, kNoDeqSpin = 4u, kNoOptCas = 8u, kPlainThrStore = 16u,
                  kThrFirst = 32u, kNoPairedFaa = 64u, kThrRedMax = 128u, kFencedPayload = 256u, kEagerEmpty = 512u, kNoCellPrefetch = 1024u, kNoFullTest = 2048u,
                  kNoRepair = 4096u,
                  kRelaxedInstall = 1u << 16 /* internal: this install needs no release edge */,
                  kPublicFlags = 0x1FFFu /* what gq_opts.flags may carry */ };
// event sites of GQ_SITE / GQ_TRACE (debug.cuh): why a ring attempt did not succeed at its first ticket
enum : uint32_t { SITE_ENQ_CAS_LOST = 0, SITE_ENQ_UNSAFE = 1, SITE_ENQ_SLOT_AHEAD = 2, SITE_ENQ_SLOT_OCCUPIED = 3,
                  SITE_DEQ_PARK_EXPIRED = 4, SITE_DEQ_NO_PARK = 5, SITE_DEQ_SLOT_OCCUPIED = 6, SITE_DEQ_THR_DEAD = 7,
                  SITE_DEQ_D1_EMPTY = 8, SITE_DEQ_THR_LOW = 9, SITE_DEQ_RETRY = 10, SITE_DEQ_EMPTY_CATCHUP = 11,
                  SITE_DEQ_EMPTY_THR = 12, SITE_DEQ_EMPTY_EARLY = 13, SITE_DEQ_EMPTY_PROBE = 14, SITE_DEQ_REPAIR = 15 };
// latency probe sites (GQ_TIC / GQ_TOC): + 5 * ring id for the first five
enum : uint32_t { LAT_HEAD_FAA = 0, LAT_SLOT_WAIT = 1, LAT_TAIL_FAA = 2, LAT_INSTALL_CAS = 3, LAT_THR_CHECK = 4,
                  LAT_PAYLOAD = 10, LAT_ENQUEUE = 11, LAT_DEQUEUE = 12,
                  LAT_STEP_PENDING_ENQ = 13, LAT_STEP_PENDING_DEQ = 14 /* enqueue_or_dequeue_step calls that handed the wait back */ };

// ---- G-LFQ entry word (Alg. 1 <c,1,x>):  [63:33] Cycle(31) | [32] Safe | [31:0] Index
struct LfqFmt {
  static constexpr int kCycBits = 31;
  static constexpr int kCtrShift = 0;                    // Head/Tail are plain counters
  static constexpr uint32_t kBotC = 0xFFFFFFFFu;         // consumed   (reading G3)
  static constexpr uint32_t kBot = 0xFFFFFFFEu;          // empty
  static constexpr uint64_t kIdxMask = 0xFFFFFFFFull;
  static constexpr uint64_t kSafeBit = 1ull << 32;
  static constexpr uint64_t kConsumeMask = kIdxMask;     // CONSUME = atomic OR of the index field
  static constexpr uint32_t kCycMask = 0x7FFFFFFFu;
  __device__ __host__ static uint32_t cycle(uint64_t e) { return (uint32_t)(e >> 33); }
  __device__ __host__ static uint32_t index(uint64_t e) { return (uint32_t)e; }
  __device__ __host__ static bool safe(uint64_t e) { return (e & kSafeBit) != 0; }
  __device__ __host__ static bool enq_visible(uint64_t) { return true; }
  __device__ __host__ static bool vacant(uint64_t e) { return index(e) >= kBot; }    // Index in {bot, botc}
  // <c, 1, x>
  __device__ __host__ static uint64_t installed(uint64_t, uint32_t c, uint32_t x) { return ((uint64_t)c << 33) | kSafeBit | x; }
  // <c, E.Safe, bot>
  __device__ __host__ static uint64_t advanced(uint64_t e, uint32_t c) { return ((uint64_t)c << 33) | (e & kSafeBit) | kBot; }
  // <E.Cycle, 0, E.Index>
  __device__ __host__ static uint64_t unsafe(uint64_t e) { return e & ~kSafeBit; }
  __device__ __host__ static uint64_t initial() { return kSafeBit | kBot; }          // <0,1,bot> (reading G4)
  // what the slot of a cycle-c ticket holds in steady state: the previous cycle's entry, consumed
  __device__ __host__ static uint64_t predicted(uint32_t c) { return ((uint64_t)((c - 1u) & kCycMask) << 33) | kSafeBit | kBotC; }
  // D9: a vacant slot of an older cycle, made ready for the enqueuer of cycle c by the dequeuer of cycle c that waits on it
  __device__ __host__ static uint64_t repaired(uint64_t, uint32_t c) { return predicted(c); }
};

// ---- direct-payload entry word (G-LFQ-D, DESIGN.md NEXT-3(i)): the uint32 payload sits where G-LFQ keeps the
//      index, and vacancy is a bit of its own so that every 32-bit value can be stored:
//      [63:34] Cycle(30) | [33] Safe | [32] Vacant | [31:0] payload
struct DirFmt {
  static constexpr int kCycBits = 30;
  static constexpr int kCtrShift = 0;
  static constexpr uint32_t kBotC = 0xFFFFFFFFu;
  static constexpr uint32_t kBot = 0xFFFFFFFEu;
  static constexpr uint64_t kIdxMask = 0xFFFFFFFFull;
  static constexpr uint64_t kVacBit = 1ull << 32;
  static constexpr uint64_t kSafeBit = 1ull << 33;
  static constexpr uint64_t kConsumeMask = kVacBit | kIdxMask;       // CONSUME: Vacant <- 1, payload <- all ones
  static constexpr uint32_t kCycMask = 0x3FFFFFFFu;
  __device__ __host__ static uint32_t cycle(uint64_t e) { return (uint32_t)(e >> 34); }
  __device__ __host__ static uint32_t index(uint64_t e) { return (uint32_t)e; }
  __device__ __host__ static bool safe(uint64_t e) { return (e & kSafeBit) != 0; }
  __device__ __host__ static bool enq_visible(uint64_t) { return true; }
  __device__ __host__ static bool vacant(uint64_t e) { return (e & kVacBit) != 0; }
  __device__ __host__ static uint64_t installed(uint64_t, uint32_t c, uint32_t x) { return ((uint64_t)c << 34) | kSafeBit | x; }
  __device__ __host__ static uint64_t advanced(uint64_t e, uint32_t c) { return ((uint64_t)c << 34) | (e & kSafeBit) | kVacBit | kBot; }
  __device__ __host__ static uint64_t unsafe(uint64_t e) { return e & ~kSafeBit; }
  __device__ __host__ static uint64_t initial() { return kSafeBit | kVacBit | kBot; }
  __device__ __host__ static uint64_t predicted(uint32_t c) { return ((uint64_t)((c - 1u) & kCycMask) << 34) | kSafeBit | kVacBit | kBotC; }
  __device__ __host__ static uint64_t repaired(uint64_t, uint32_t c) { return predicted(c); }
};

// ---- G-WFQ entry word (Fig. 2 missing -> reading W1):
//      [63:48] Cycle(16) | [47:32] Note(16) | [31] Safe | [30] Enq | [29:0] Index(30)
struct WfqFmt {
  static constexpr int kCycBits = 16;
  static constexpr int kCtrShift = 20;                   // Head/Tail word: counter(44) | ThrIdx(20)
  static constexpr uint32_t kBotC = 0x3FFFFFFFu;
  static constexpr uint32_t kBot = 0x3FFFFFFEu;
  static constexpr uint64_t kIdxMask = 0x3FFFFFFFull;
  static constexpr uint64_t kEnqBit = 1ull << 30;
  static constexpr uint64_t kSafeBit = 1ull << 31;
  static constexpr uint64_t kNoteMask = 0xFFFFull << 32;
  static constexpr uint64_t kConsumeMask = kIdxMask | kEnqBit;   // sets Enq=1 and Index=botc together
  static constexpr uint32_t kCycMask = 0xFFFFu;
  static constexpr uint64_t kThrIdxMask = (1ull << kCtrShift) - 1;
  static constexpr uint64_t kThrNull = kThrIdxMask;
  __device__ __host__ static uint32_t cycle(uint64_t e) { return (uint32_t)(e >> 48); }
  __device__ __host__ static uint32_t note(uint64_t e) { return (uint32_t)(e >> 32) & 0xFFFFu; }
  __device__ __host__ static uint32_t index(uint64_t e) { return (uint32_t)(e & kIdxMask); }
  __device__ __host__ static bool safe(uint64_t e) { return (e & kSafeBit) != 0; }
  __device__ __host__ static bool enq_visible(uint64_t e) { return (e & kEnqBit) != 0; }
  __device__ __host__ static bool vacant(uint64_t e) { return index(e) >= kBot; }
  // Note (Lemma III.8) is compared modulo 2^16 like Cycle (Lemma III.6), so it must stay inside the same
  // window: every write that sets Cycle to c also raises Note to c unless a slow-path helper has already moved
  // it further ahead (that decision must survive: the helpers of one request have to agree on the slots they
  // skip).  Left at its initial value Note would read as "newer" again after 2^15 laps and rule the slot out
  // for every slow-path enqueue.
  __device__ __host__ static uint64_t note_for(uint64_t e, uint32_t c) {
    const uint32_t d = (note(e) - c) & 0xFFFFu;                           // Note ahead of c by d cycles (mod 2^16)
    return (uint64_t)((d != 0 && d < 0x8000u) ? note(e) : c) << 32;
  }
  // fast path installs <c, Safe 1, Enq 1, x>
  __device__ __host__ static uint64_t installed(uint64_t e, uint32_t c, uint32_t x) {
    return ((uint64_t)c << 48) | note_for(e, c) | kSafeBit | kEnqBit | x;
  }
  __device__ __host__ static uint64_t installed_slow(uint64_t e, uint32_t c, uint32_t x) {   // Enq = 0
    return ((uint64_t)c << 48) | note_for(e, c) | kSafeBit | x;
  }
  __device__ __host__ static uint64_t advanced(uint64_t e, uint32_t c) {
    return ((uint64_t)c << 48) | note_for(e, c) | (e & kSafeBit) | kEnqBit | kBot;
  }
  __device__ __host__ static uint64_t unsafe(uint64_t e) { return e & ~kSafeBit; }
  __device__ __host__ static uint64_t with_note(uint64_t e, uint32_t c) { return (e & ~kNoteMask) | ((uint64_t)c << 32); }
  __device__ __host__ static uint64_t initial() { return kSafeBit | kEnqBit | kBot; }       // Cycle 0, Note 0; tickets start at cycle 1
  // steady state: previous cycle, consumed (CONSUME sets Enq with the index), Note = that cycle
  __device__ __host__ static uint64_t predicted(uint32_t c) {
    const uint64_t p = (c - 1u) & kCycMask;
    return (p << 48) | (p << 32) | kSafeBit | kEnqBit | kBotC;
  }
  __device__ __host__ static uint64_t repaired(uint64_t e, uint32_t c) {
    const uint32_t p = (c - 1u) & kCycMask;
    return ((uint64_t)p << 48) | note_for(e, p) | kSafeBit | kEnqBit | kBotC;
  }
};

// Hook run by a dequeuer between finding its entry and CONSUME.  G-LFQ: nothing.
struct NoFinalize {
  __device__ __forceinline__ void operator()(const RingView&, uint64_t /*h*/, uint32_t /*j*/, uint64_t /*E*/) const {}
};


template <class F, bool kUniform, int kWarpFaa = true>
struct Ring {
  __device__ __forceinline__ static uint64_t* slot(const RingView& r, uint32_t j) {
    return r.entry + ((size_t)j << r.slot_shift);
  }
  __device__ __forceinline__ static uint32_t slot_of(const RingView& r, uint64_t t) { return (uint32_t)t & ((1u << r.order) - 1u); }
  __device__ __forceinline__ static uint32_t cycle_of(const RingView& r, uint64_t t) { return (uint32_t)(t >> r.order) & F::kCycMask; }
  __device__ __forceinline__ static uint64_t counter(uint64_t word) { return word >> F::kCtrShift; }

  // ticket reservation: WAVEFAA on a (possibly packed) counter word, through the block's funnel when it has one
  __device__ __forceinline__ static uint64_t take(const RingView& r, bool head) {
    constexpr uint64_t unit = 1ull << F::kCtrShift;
    uint64_t* ctr = head ? r.head : r.tail;
    // kWarpFaa: 0 = one FAA per thread (ablation), 1 = WAVEFAA, 2 = WAVEFAA through the block's funnels (D11)
    const uint64_t w = kWarpFaa ? warp_faa<kUniform>(ctr, unit, kWarpFaa == 2 ? (head ? r.fhead : r.ftail) : nullptr) : lane_faa(ctr, unit);
    return counter(w);
  }

  // "reset Threshold to 3n-1" (Alg. 1): load first, store only when different (reading G8).
  // On a GPU this is not about cache-line ownership (every .gpu access resolves at L2) but about
  // the L2 itself: same-address loads are served far faster than same-address stores.  Measured on
  // B200: a plain store per enqueue (kPlainThrStore) serialises all
  // enqueuers on the Threshold word and costs 50x in throughput.
  __device__ __forceinline__ static void reset_threshold(const RingView& r, uint32_t flags = 0) {
    if (GQ_MUT(MUT_NO_THR_RESET)) return;
    if (flags & kThrRedMax) {
      // Threshold never exceeds 3N-1, so "Threshold <- 3N-1" == max(Threshold, 3N-1): one fire-and-forget
      // reduction by the leader of the lanes whose CAS just succeeded (all of them have their CAS result);
      // converged lanes of a non-uniform caller may name different rings: one leader per Threshold word
      uint32_t mask = __activemask();
      if (!kUniform) mask = __match_any_sync(mask, reinterpret_cast<unsigned long long>(r.threshold));
      if (lane_id() == (uint32_t)__ffs(mask) - 1) red_max_s64_relaxed(r.threshold, r.thr_reset);
      return;
    }
    GQ_TIC(t0);
    const int64_t thr = (flags & kPlainThrStore) ? -1 : (int64_t)ld_relaxed(reinterpret_cast<const uint64_t*>(r.threshold));
    GQ_TOC(LAT_THR_CHECK + 5 * r.id, t0, thr);
    if (thr != r.thr_reset) st_relaxed(reinterpret_cast<uint64_t*>(r.threshold), (uint64_t)r.thr_reset);
  }

  // "catch up Tail to at least h+1" (Alg. 1; reading G9).  Batched like WAVEFAA: the
  // converged lanes agree on their largest target and only the leader touches the hot word
  // (one atomic per warp instead of 32 on the same address).
  __device__ __forceinline__ static void catchup_tail(const RingView& r, uint64_t target) {
    const uint32_t active = __activemask();
    uint32_t mask = active;
    if (!kUniform) mask = __match_any_sync(active, reinterpret_cast<unsigned long long>(r.tail));
    const uint32_t leader = __ffs(mask) - 1;
    const uint64_t base = __shfl_sync(active, target, leader);         // over the converged set, see warp_faa
    const int d = (int)(int64_t)(target - base);                        // tickets of one warp are close
    int dmax = d;
    if (kUniform) {
      dmax = __reduce_max_sync(active, d);
    } else {                                                            // one converged reduction per address group
      for (uint32_t rest = active; rest;) {
        const uint32_t g = __shfl_sync(active, mask, __ffs(rest) - 1);
        const int m = __reduce_max_sync(active, mask == g ? d : INT_MIN);
        if (mask == g) dmax = m;
        rest &= ~g;
      }
    }
    if (lane_id() != leader) return;
    target = base + (int64_t)dmax;
    if (F::kCtrShift == 0) {
      red_max_relaxed(r.tail, target);
    } else {
      uint64_t w = ld_relaxed(r.tail);
      for (int i = 0; i < 64 && counter(w) < target; ++i) {      // bounded; counter field only grows
        const uint64_t nw = (target << F::kCtrShift) | (w & ((1ull << F::kCtrShift) - 1));
        const uint64_t o = cas_relaxed(r.tail, w, nw);
        if (o == w) break;
        w = o;
      }
    }
  }

  __device__ __forceinline__ static uint64_t install_cas(uint64_t* sp, uint64_t E, uint64_t N, uint32_t flags) {
    return (flags & kRelaxedInstall) ? cas_relaxed(sp, E, N) : cas_release(sp, E, N);
  }

  // Alg. 1 L143-163.  Returns RING_OK or RING_RETRY; *t_out = the ticket used.
  //
  // Optimistic install (sm_100a; kNoOptCas switches it off): in steady state the slot of a
  // cycle-c ticket holds the consumed entry of cycle c-1, <c-1, 1, bot_c>, for which every
  // condition of L150-151 holds by construction.  The installing CAS is therefore issued
  // against that predicted word first; when it fails, the value it returns IS the load of
  // L148 and the listing continues from there.  One L2 round trip (FAA -> CAS) instead of two
  // (FAA -> load -> CAS) on the common path; same linearization point (the successful CAS).
  // have/t_pre: the ticket was already reserved by the caller (D5); else it is drawn here.
  __device__ __forceinline__ static int try_enq(const RingView& r, uint32_t x, uint64_t* t_out, uint32_t flags = 0,
                                                bool have = false, uint64_t t_pre = 0) {
    GQ_TIC(t0);
    const uint64_t t = have ? t_pre : take(r, false);                   // L144
    if (!have) GQ_TOC(LAT_TAIL_FAA + 5 * r.id, t0, t);
    *t_out = t;
    // A first-touch CAS is an L2 miss that the slice's atomic unit waits out, with every atomic queued behind
    // it ("cold lines"): for rings that cannot stay L2-resident, fetch a later slot now.
    if (r.prefetch) asm volatile("prefetch.global.L2 [%0];" :: "l"(slot(r, slot_of(r, t + r.prefetch))));
    const uint32_t j = slot_of(r, GQ_MUT(MUT_LIFO_PAIR) ? (t ^ 1) : t), c = cycle_of(r, t);   // L146
    uint64_t* sp = slot(r, j);
    uint64_t E;
    GQ_TIC(t1);
    if (!(flags & kNoOptCas)) {
      E = F::predicted(c);
      const uint64_t o = install_cas(sp, E, F::installed(E, c, x), flags);   // L153 on the predicted entry
      GQ_TOC(LAT_INSTALL_CAS + 5 * r.id, t1, o);
      if (o == E) { GQ_IDX_EVENT(1, r, x, t, o, 0); reset_threshold(r, flags); return RING_OK; }      // L155
      E = o;                                                          // L148: the failed CAS read the slot
    } else {
      E = ld_relaxed(sp);                                             // L148
    }
    if (cycle_newer<F::kCycBits>(c, F::cycle(E)) && F::vacant(E)) {   // E.Cycle < c, Index in {bot,botc}
      bool ok = F::safe(E);
      if (!ok) {                                                      // (E.Safe or Head <= t), reading G5
        fence_acq_rel();                                              // Head must not be older than E
        ok = counter(ld_relaxed(r.head)) <= t;
      }
      if (ok && install_cas(sp, E, F::installed(E, c, x), flags) == E) {   // L153: linearization point (L111)
        GQ_IDX_EVENT(1, r, x, t, E, 1);
        reset_threshold(r, flags);                                    // L155
        return RING_OK;
      }
      GQ_SITE(ok ? SITE_ENQ_CAS_LOST : SITE_ENQ_UNSAFE);
      GQ_TRACE((ok ? SITE_ENQ_CAS_LOST : SITE_ENQ_UNSAFE) | r.id << 8, r, t, E, 0);
    } else {
      GQ_SITE(F::vacant(E) ? SITE_ENQ_SLOT_AHEAD : SITE_ENQ_SLOT_OCCUPIED);
      GQ_TRACE((F::vacant(E) ? SITE_ENQ_SLOT_AHEAD : SITE_ENQ_SLOT_OCCUPIED) | r.id << 8, r, t, E, 0);
    }
    return RING_RETRY;                                                // L163 (reading G7)
  }

  // Alg. 1 L165-211 with the reconstruction of reading G6 (reload on CAS failure).
  // Returns RING_OK (+ *x), RING_EMPTY or RING_RETRY; *h_out = the ticket used.
  //
  // Two bounded additions for sm_100a, where k >> n threads can poll an empty ring
  // (DESIGN.md "departures" D1, D2; each can be switched off for the ablation):
  //  D1 read-only emptiness probe.  Taken when the caller's previous attempt on this ring came
  //     back EMPTY (`probe`) or Threshold is below its reset value (some dequeuer failed since
  //     the last successful enqueue).  Head is read first (acquire), then Tail:
  //     Tail(t2) <= Head(t1) <= Head(t2) is the very condition of L197 ("Tail <= h+1" seen by
  //     the owner of ticket h), observed without claiming a ticket.  EMPTY is returned only
  //     when Head is already park_limit tickets ahead of Tail, i.e. enough dequeuers are
  //     parked (D2) to absorb the next enqueues; below that the caller claims a ticket.
  //  D2 bounded parking.  A dequeuer whose slot is still vacant (its enqueuer has not
  //     installed yet, or has not even claimed ticket h yet) re-reads its OWN slot with
  //     __nanosleep backoff for at most park_ns before it invalidates the slot as L186-188
  //     prescribe.  The wait is on a private address, so parked threads put no load on the
  //     hot Head/Tail/Threshold lines, Head does not run away from Tail, and the enqueuer
  //     that later draws ticket h hands its item straight to the parked dequeuer.  Pure delay
  //     in front of the paper's steps: every operation still finishes in bounded own steps.
  //  D4 Threshold read overlapped with the ticket.  L166-169 ("Threshold < 0 => EMPTY") is an early
  //     exit, not a condition the rest depends on: a dequeuer that skips it simply takes the general
  //     path.  A caller whose last attempt on this ring succeeded (`probe` false) therefore issues
  //     the Threshold load and the Head FAA back to back and looks at the loaded value only after
  //     the ticket has come back: one L2 round trip instead of two.  A value below the reset value
  //     (some dequeuer failed since the last enqueue) only matters if the slot is vacant: the D1
  //     test is then made with the ticket in the place of Head, and parking (D2) is skipped when it
  //     says "empty" or Threshold was negative, which leaves the listing's own steps.  kThrFirst
  //     restores the listed order.
  //  nb != nullptr: non-blocking parking (DeqWait above).  nb->pending() resumes the attempt that holds nb->ticket.
  template <class Finalize>
  __device__ __forceinline__ static int try_deq(const RingView& r, uint32_t* x, uint64_t* h_out, const Finalize& fin,
                                                bool probe = false, uint32_t flags = 0, DeqWait* nb = nullptr) {
    uint32_t park_ns = (flags & kNoDeqSpin) ? 0u : r.park_ns;
    int64_t thr;
    uint64_t h;
    const bool listed = probe || (flags & kThrFirst);
    const bool resume = nb && nb->pending();
    GQ_TIC(t0);
    if (resume) {
      h = nb->ticket;                                                  // drawn by the call that returned RING_PENDING
      thr = r.thr_reset;
    } else if (listed) {
      thr = (int64_t)ld_relaxed(reinterpret_cast<const uint64_t*>(r.threshold));
      if (thr < 0) { GQ_SITE(SITE_DEQ_EMPTY_EARLY); return RING_EMPTY; }   // L166-169
      if (!(flags & kNoProbe) && (probe || thr != r.thr_reset)) {     // D1
        const uint64_t H = counter(ld_acquire(r.head));
        const uint64_t T = counter(ld_relaxed(r.tail));
        if (GQ_MUT(MUT_UNSOUND_EMPTY) && T <= H + 2) return RING_EMPTY;
        if (T + ((park_ns && !(flags & kEagerEmpty)) ? r.park_limit : 0u) <= H) { GQ_SITE(SITE_DEQ_EMPTY_PROBE); return RING_EMPTY; }
      }
      h = take(r, true);                                               // L172
      thr = r.thr_reset;                                              // parking allowed (as before D4)
    } else {
      thr = (int64_t)ld_relaxed(reinterpret_cast<const uint64_t*>(r.threshold));   // in flight with the FAA / slot load
      h = take(r, true);                                               // L172
    }
    GQ_TOC(LAT_HEAD_FAA + 5 * r.id, t0, h);
    *h_out = h;
    if (r.prefetch) asm volatile("prefetch.global.L2 [%0];" :: "l"(slot(r, slot_of(r, h + r.prefetch))));
    const uint32_t j = slot_of(r, h), c = cycle_of(r, h);             // L175
    uint64_t* sp = slot(r, j);
    // park budget in ns: every look at the slot counts its nap plus kPollNs (an L2 round trip under load)
    constexpr uint32_t kPollNs = 384;
    uint32_t waited = 0, nap = 0;
    if (resume) {                                                      // real time spent in line so far (never 0: 0 = first look)
      const uint64_t dt = globaltimer_ns() - nb->since;
      waited = dt >= 0xFFFFFFFFull ? 0xFFFFFFFFu : (dt ? (uint32_t)dt : 1u);
    }
    GQ_TIC(t1);
    for (;;) {
      // L176.  Acquire in every build: it is the consumer side of the hand-over contract of queue.cuh (reading G15): what a
      // producer wrote before __threadfence(); enqueue(v) is visible to the thread that dequeued v.  (A relaxed poll where the
      // library itself needs no edge, D6 / direct payload, was tried: +0.4 %, and the user-kernel litmus failed at once.)
      uint64_t E = ld_acquire(sp);
    classify:
      if (F::cycle(E) == c && !F::vacant(E)) {                        // L178
        GQ_TOC(LAT_SLOT_WAIT + 5 * r.id, t1, E);
        fin(r, h, j, E);                                              // G-WFQ: finalize an Enq=0 entry (W6)
        GQ_IDX_EVENT(5, r, F::index(E), h, E, 0);
        red_or_relaxed(sp, F::kConsumeMask);                          // L180 CONSUME: linearization point
        *x = F::index(E);
        return RING_OK;                                               // L182
      }
      if (cycle_newer<F::kCycBits>(c, F::cycle(E))) {                 // E.Cycle < c (guard lost in extraction)
        if (waited < park_ns && F::vacant(E)) {                       // D2
          if (waited == 0) {                                          // first look at a vacant slot
            if ((flags & kEagerEmpty) && counter(ld_relaxed(r.tail)) <= h) {
              park_ns = 0;                                            // polling consumers: wait only for an enqueuer that
              goto classify;                                          // already holds ticket h, never for a future one
            }
            if (thr != r.thr_reset) {                                 // D4 path, first use of thr: some dequeuer failed since
              const bool dead = thr < 0;                              // the last enqueue, so apply D1 now, with the ticket as Head
              thr = r.thr_reset;
              if (dead || (!(flags & kNoProbe) && counter(ld_relaxed(r.tail)) + ((flags & kEagerEmpty) ? 0u : r.park_limit) <= h)) {
                GQ_SITE(dead ? SITE_DEQ_THR_DEAD : SITE_DEQ_D1_EMPTY);
                GQ_TRACE((dead ? SITE_DEQ_THR_DEAD : SITE_DEQ_D1_EMPTY) | r.id << 8, r, h, E, 0);
                park_ns = 0;
                goto classify;
              }
              GQ_SITE(SITE_DEQ_THR_LOW);                              // thr below reset seen on the D4 path, parking kept
            }
            // D9 repair.  A slot that a dequeuer once marked unsafe (L193) stays unsafe until an enqueuer arrives with
            // Head <= its ticket (L151), which never happens on a ring whose dequeuers wait in line (Head ahead of Tail for
            // good: FQ whenever k > n): the enqueuer of every later cycle gives the slot up and its parked dequeuer waits
            // out the whole park_ns, lap after lap.  The dequeuer that is about to wait here IS the dequeuer of cycle c, so
            // it may declare the slot ready for the enqueuer of cycle c, <c-1, Safe 1, bot_c>, provided no dequeuer of a
            // later cycle has been here before it, i.e. Head has not reached h + 2N (read after E; Head only grows).
            if (!F::safe(E) && !(flags & kNoRepair) && counter(ld_relaxed(r.head)) <= h + (1ull << r.order)) {
              const uint64_t R = F::repaired(E, c);
              const uint64_t o = cas_relaxed(sp, E, R);
              GQ_SITE(SITE_DEQ_REPAIR);
              if (o != E) { E = o; goto classify; }                   // the slot changed under us: classify what the CAS read
            }
          }
          // (Rejected, measured: sizing the nap by the place in line, h - Tail.  Any load of the hot Tail
          //  word inside the polling loop takes the ring from 37 to 12 Gops/s at k = 227 328: parked
          //  threads must stay off the hot lines, which is the point of D2.)
          // The first spin_ns are pure re-reading (the front of the line: the hand-over is detected one nap
          // earlier), after that the nap ladder 32 ns .. park_nap keeps the many threads further back quiet.
          if (nb) {                                                    // wait handed back to the caller, ticket kept
            if (!resume) { nb->ticket = h; nb->since = globaltimer_ns(); }
            return RING_PENDING;
          }
          if (waited >= r.spin_ns && r.park_nap) { nap = nap ? (nap * 2 < r.park_nap ? nap * 2 : r.park_nap) : 32; __nanosleep(nap); }
          waited += nap + kPollNs;
          continue;
        }
        GQ_SITE(F::vacant(E) ? (park_ns ? SITE_DEQ_PARK_EXPIRED : SITE_DEQ_NO_PARK) : SITE_DEQ_SLOT_OCCUPIED);
        GQ_TRACE((F::vacant(E) ? (park_ns ? SITE_DEQ_PARK_EXPIRED : SITE_DEQ_NO_PARK) : SITE_DEQ_SLOT_OCCUPIED) | r.id << 8, r, h, E, waited);
        const uint64_t New = F::vacant(E) ? F::advanced(E, c)         // L186-188
                                          : F::unsafe(E);             // L193
        if (New != E) {
          const uint64_t o = cas_relaxed(sp, E, New);
          if (o != E && !GQ_MUT(MUT_NO_RELOAD)) { E = o; goto classify; }   // reload: the slot changed under us (G6): the failed CAS read it
        }
      }
      break;
    }
    const uint64_t T = counter(ld_relaxed(r.tail));
    if (T <= h + 1) {                                                 // L197
      GQ_SITE(SITE_DEQ_EMPTY_CATCHUP);
      GQ_TRACE(SITE_DEQ_EMPTY_CATCHUP | r.id << 8, r, h, 0, T);
      catchup_tail(r, h + 1);                                         // L200
      warp_dec<kUniform>(r.threshold);                                // L202
      return RING_EMPTY;
    }
    if (warp_dec<kUniform>(r.threshold) <= 0) { GQ_SITE(SITE_DEQ_EMPTY_THR); return RING_EMPTY; }   // L205-208
    GQ_SITE(SITE_DEQ_RETRY);
    GQ_TRACE(SITE_DEQ_RETRY | r.id << 8, r, h, 0, T);
    return RING_RETRY;                                                // L211
  }
};

}  // namespace detail
}  // namespace gq
