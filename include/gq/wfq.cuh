// gq/wfq.cuh — G-WFQ, the bounded wait-free queue (§III-C, Alg. 2).
//
// Same 2N-slot ring and the same fast path as G-LFQ ("G-WFQ uses the same fast-path as
// G-LFQ"), bounded by patience constants; after that the operation publishes a
// fixed per-thread request record and enters the cooperative slow path, where
// owner and helpers advance the global counter exactly once per round with SLOWFAA (Alg. 2,
// Lemma III.7) and act on the slot with TRYENQSLOW / TRYDEQSLOW (Lemma III.8).
// Every shared word that is concurrently modified — slot entry, global Head/Tail, local
// head/tail — is ONE 64-bit word updated by one 64-bit atomic (Lemma III.5); no
// double-width CAS anywhere.
//
// Word layouts (Figs. 2-3 are missing from PAPER.md -> DESIGN.md reading W1):
//   entry  : [63:48] Cycle | [47:32] Note | [31] Safe | [30] Enq | [29:0] Index      (ring.cuh WfqFmt)
//   global : [63:20] counter | [19:0] ThrIdx (0xFFFFF = NULL)
//   local  : [63:20] counter | [19:4] request tag | [1] INC | [0] FIN
// The request tag (low 16 bits of the owner's request sequence number) is this design's own
// addition: every CAS a helper issues on a local word carries the tag of the request it is
// helping, so a helper that outlives "its" request can never touch a later request of the
// same thread (reading W10).
#pragma once
#include "lfq.cuh"

namespace gq {

// One record per (thread, ring), one 128-byte line (request flags, initial and local
// head/tail, payload index, two sequence fields, a phase-2 record).
struct alignas(128) WfqRecord {
  uint64_t localTail, localHead;       // packed local words (shared, CAS)
  uint64_t initTail, initHead;         // counter values at publication
  uint64_t p2_seq1, p2_target, p2_expect, p2_seq2;   // phase-2 record (L, c) + its sequence pair (Alg. 2)
  uint64_t seq1, seq2;                 // request sequence pair
  uint32_t pending, enqueue, index, _r0;
  uint32_t n_slow_enq, n_slow_deq, n_helps, _r1;     // statistics (owner-private)
  // Lemma III.7 bookkeeping, written only by the thread that owns this record, about rounds it performed for ANY request:
  // global increments <c,NULL> -> <c+1,tid> it won, and INC bits it cleared (the end of a logical round), per counter
  uint32_t n_tail_inc, n_tail_clr, n_head_inc, n_head_clr;
};
static_assert(sizeof(WfqRecord) == 128, "one L2 line per record");

struct WfqView {
  RingView aq, fq;          // RingView::rec -> WfqRecord[nthreads] of that ring, ::owner -> Owner[2N]
  uint64_t* data;           // Data[n]: payload cells <ticket tag | v> (D6; the tag is used for fast-path installs only)
  uint32_t capacity;
  uint32_t nthreads;        // help ring size k (reading W7)
  uint32_t enq_patience, deq_patience, help_delay;
  uint32_t flags;
};

namespace detail {

// D6 in G-WFQ.  A fast-path enqueue knows its AQ ticket before it installs, so it can use G-LFQ's
// ticket-tagged payload cell and a relaxed install; a slow-path install happens at a ticket the owner
// does not know in advance (a helper may do it), so it keeps the release/acquire chain of the request
// record instead.  The dequeuer must know which kind of entry it consumed: fast-path installs set
// bit 29 of the 30-bit Index field (indices are < 2^29 - 2), slow-path installs leave it clear.
constexpr uint32_t kWfqFast = 1u << 29, kWfqIdxMask = kWfqFast - 1u;

struct Wf {
  using F = WfqFmt;
  static constexpr int S = WfqFmt::kCtrShift;          // 20
  static constexpr uint64_t kFIN = 1, kINC = 2;
  static constexpr uint64_t kNull = WfqFmt::kThrNull;
  __device__ __forceinline__ static uint32_t tag_of(uint64_t w) { return (uint32_t)(w >> 4) & 0xFFFFu; }
  __device__ __forceinline__ static uint64_t local_word(uint64_t cnt, uint32_t tag) { return (cnt << S) | ((uint64_t)tag << 4); }
  __device__ __forceinline__ static WfqRecord* rec(const RingView& r, uint32_t tid) { return reinterpret_cast<WfqRecord*>(r.rec) + tid; }
  __device__ __forceinline__ static uint64_t* local_ptr(const RingView& r, uint64_t target) {
    WfqRecord* w = rec(r, (uint32_t)(target >> 1));
    return (target & 1) ? &w->localHead : &w->localTail;
  }

  // Help the phase-2 request named by ThrIdx u (Alg. 2): clear INC on the local word
  // its record names.  Accepted only if the record's sequence pair matches, it is a record of THIS
  // global word (a thread has one phase-2 record per ring, used for its Head rounds and its Tail
  // rounds alike: Head may still name u after a Head round of u whose ThrIdx nobody has cleared yet,
  // while u has since published a Tail round; its counter is a Tail counter, and clearing INC on
  // that local tail would hand the request a ticket nobody drew), and its counter is below the
  // global counter c we saw next to u (a record of a later round has counter >= c).
  template <bool kDeq>
  __device__ static void help_phase2(const RingView& r, uint32_t u, uint64_t c, uint32_t me) {
    WfqRecord* p = rec(r, u);
    const uint64_t s2 = ld_acquire(&p->p2_seq2);
    const uint64_t target = ld_relaxed(&p->p2_target);
    const uint64_t expect = ld_relaxed(&p->p2_expect);
    fence_acq_rel();
    if (ld_relaxed(&p->p2_seq1) != s2) return;
    if (((target & 1) != 0) != kDeq && !GQ_MUT(MUT_P2_ANY_SIDE)) return;
    if ((expect >> S) >= c || !(expect & kINC)) return;
    if (cas_relaxed(local_ptr(r, target), expect, expect & ~kINC) == expect) {
      GQ_L_EVENT(r, target, 'P', me, expect, ((uint64_t)u << 44) | c);
      WfqRecord* mine = rec(r, me);
      ++((target & 1) ? mine->n_head_clr : mine->n_tail_clr);
    }
  }

  // Memory orders of the slow path (sm_100a: an acq_rel atomic is MEMBAR.ALL.GPU + ATOM, about two L2 round trips).  Every
  // word below is only ever accessed with L2 atomics and strong loads, and the protocol decides on VALUES (counters, tags,
  // cycles), so most transitions are relaxed.  Two edges carry data and keep their order: (i) the phase-2 record goes out
  // before the CAS that puts this thread's id into G (release; readers of the ThrIdx acquire G); (ii) the payload cell and
  // the request record go out before the entry is installed (the helper acquires the record's sequence word, its
  // installing CAS is a release, the dequeuer's slot load an acquire).
  // SLOWFAA (Alg. 2; reading W4).  G = global Head or Tail word, L = the request's
  // local word, v = last value of L this helper knows, tag = request tag, me = this thread.
  // Returns true with v = <ticket, tag> (no flags) when the round's ticket is known; false when
  // the request is finished (FIN) or no longer the one being helped.
  template <bool kDeq>
  __device__ static bool slow_faa(const RingView& r, uint64_t* G, uint64_t* L, uint64_t& v, uint32_t tag, uint32_t me,
                                  uint64_t target_id) {
    WfqRecord* mine = rec(r, me);
    uint64_t c = 0;
    Backoff bo;
    uint32_t lost_nap = 512;
    [[maybe_unused]] uint32_t sn1 = 0, sn2 = 0;
    for (;;) {
      if (GQ_STUCK(sn1, (kDeq ? 11 : 10) | r.id << 8, me, G, L, kDeq ? r.tail : r.head, r.threshold)) return false;
      bool have = false;
      for (;;) {                                            // L249-257: FIN check, read G, help phase 2
        if (GQ_STUCK(sn2, (kDeq ? 13 : 12) | r.id << 8, me, G, L, kDeq ? r.tail : r.head, r.threshold)) return false;
        const uint64_t lv = ld_acquire(L);
        if (tag_of(lv) != tag || (lv & kFIN)) break;
        const uint64_t g = ld_acquire(G);
        c = g >> S;
        const uint32_t u = (uint32_t)(g & kNull);
        if (u == kNull) { have = true; break; }
        help_phase2<kDeq>(r, u, c, me);
        if (cas_relaxed(G, g, (c << S) | kNull) == g) { have = true; break; }
      }
      const uint64_t want = local_word(c, tag) | kINC;      // L258: synchronize L to c using INC
      if (!have || cas_relaxed(L, v, want) != v) {
        v = ld_acquire(L);
        if (tag_of(v) != tag || (v & kFIN)) return false;
        if (!(v & kINC)) return true;                       // round already completed by another helper
        c = v >> S;
      } else {
        GQ_L_EVENT(r, target_id, 'S', me, v, want);
        v = want;
      }
      // L260: publish phase-2 record (L, c) under its sequence pair
      const uint64_t s = mine->p2_seq1 + 1;
      st_release(&mine->p2_seq1, s);
      st_relaxed(&mine->p2_target, target_id);
      st_relaxed(&mine->p2_expect, v);
      st_release(&mine->p2_seq2, s);
      const uint64_t g0 = (c << S) | kNull;
      if (cas_acq_rel(G, g0, ((c + 1) << S) | me) == g0) break;        // L262: <c,NULL> -> <c+1,tid>; release: the record is visible to whoever reads this ThrIdx
      bo.pause();                                                      // lost the round: thousands of losers must not keep G busy
      // Backoff's ladder ends at 1 us; k losers that come back every microsecond ask G's L2 line for k atomics per microsecond,
      // it serves 1.5 per ns (C1), and the round's winner, whose two dependent CAS on G ARE the round, waits in that line too.
      // RingView::slow_nap (about 1 ns per launched thread) lets the ladder go on.  Still a bounded delay per lost round.
      if (bo.ns >= 1024 && r.slow_nap > 1024) { lost_nap = lost_nap * 2 < r.slow_nap ? lost_nap * 2 : r.slow_nap; if (lost_nap > 1024) __nanosleep(lost_nap - 1024); }
    }
    ++(kDeq ? mine->n_head_inc : mine->n_tail_inc);
    if (kDeq) faa_relaxed(reinterpret_cast<uint64_t*>(r.threshold), (uint64_t)-1ll);   // L264-266
    GQ_L_EVENT(r, target_id, 'W', me, v, c);
    if (cas_relaxed(L, v, v & ~kINC) == v) ++(kDeq ? mine->n_head_clr : mine->n_tail_clr);   // L270: clear INC on L
    cas_relaxed(G, ((c + 1) << S) | me, ((c + 1) << S) | kNull);         // L273: clear ThrIdx in G
    v &= ~kINC;
    return true;
  }

  // A fast-path dequeuer that meets a current-cycle entry with Enq = 0 finalises the
  // enqueuer's request before it consumes (reading W6): FIN on the owner's localTail whose
  // counter equals h.  Owner[j] = <cycle, tid> written by the installer, full scan as fallback.
  struct Finalize {
    uint32_t nthreads;
    __device__ void operator()(const RingView& r, uint64_t h, uint32_t j, uint64_t E) const {
      if (F::enq_visible(E)) return;
      const uint64_t o = ld_acquire(r.owner + j);
      if ((uint32_t)(o >> 32) == F::cycle(E) && (uint32_t)o < nthreads && try_fin(r, (uint32_t)o, h)) return;
      for (uint32_t t = 0; t < nthreads; ++t)
        if (try_fin(r, t, h)) return;
    }
    __device__ static bool try_fin(const RingView& r, uint32_t tid, uint64_t h) {
      uint64_t* L = &rec(r, tid)->localTail;
      const uint64_t v = ld_acquire(L);
      if ((v >> S) != h) return false;
      if (!(v & 3)) cas_relaxed(L, v, v | kFIN);
      return true;
    }
  };

  // TRYENQSLOW (reading W5) for ticket T of the request <x, L, tag>.
  // true: the request is resolved (entry installed at T); false: try the next ticket.
  __device__ static bool try_enq_slow(const RingView& r, uint64_t T, uint32_t x, uint64_t* L, uint64_t v, uint32_t owner) {
    using R = Ring<F, false, true>;
    const uint32_t j = R::slot_of(r, T), c = R::cycle_of(r, T);
    uint64_t* sp = R::slot(r, j);
    [[maybe_unused]] uint32_t sn = 0;
    for (;;) {
      if (GQ_STUCK(sn, 20, owner, sp, L)) return true;
      const uint64_t E = ld_acquire(sp);
      if (cycle_newer<16>(c, F::cycle(E)) && cycle_newer<16>(c, F::note(E))) {
        const bool usable = F::vacant(E) && (F::safe(E) || R::counter(ld_acquire(r.head)) <= T);
        if (!usable) {                                        // Lemma III.8: advance Note, skip this slot
          if (cas_relaxed(sp, E, F::with_note(E, c)) != E) continue;
          return false;
        }
        st_relaxed(r.owner + j, ((uint64_t)c << 32) | owner);
        const uint64_t N = F::installed_slow(E, c, x);        // <c, Safe 1, Enq 0, x>: linearization point
        if (cas_release(sp, E, N) != E) continue;          // release: Data[x] (ordered by the record's acquire) goes with the entry
        GQ_IDX_EVENT(3, r, x, T, E, v);
        if (GQ_MUT(MUT_SLOW_NO_FIN) && (T & 3) == 0) { cas_relaxed(sp, N, N | F::kEnqBit); return false; }
        if (cas_relaxed(L, v, v | kFIN) == v)                 // finalise the request ...
          cas_relaxed(sp, N, N | F::kEnqBit);                 // ... and make the entry visible to fast dequeuers
        R::reset_threshold(r);
        return true;
      }
      if (F::cycle(E) == c && !F::vacant(E)) {                // installed by another helper of this request
        GQ_IDX_EVENT(4, r, x, T, E, v);
        if (cas_relaxed(L, v, v | kFIN) == v) cas_relaxed(sp, E, E | F::kEnqBit);
        R::reset_threshold(r);
        return true;
      }
      return false;                                           // slot ruled out (Note / newer cycle / consumed)
    }
  }

  // FIN on <H, tag>: true iff the request now is finished AT this ticket.
  __device__ __forceinline__ static bool set_fin(uint64_t* L, uint64_t v) {
    const uint64_t o = cas_relaxed(L, v, v | kFIN);
    return o == v || o == (v | kFIN);
  }

  // TRYDEQSLOW (reading W5) for ticket H.  true: resolved (FIN set: entry ready at H,
  // or EMPTY); false: next ticket.
  __device__ static bool try_deq_slow(const RingView& r, uint64_t H, uint64_t* L, uint64_t v) {
    using R = Ring<F, false, true>;
    const uint32_t j = R::slot_of(r, H), c = R::cycle_of(r, H);
    uint64_t* sp = R::slot(r, j);
    [[maybe_unused]] uint32_t sn = 0;
    for (;;) {
      if (GQ_STUCK(sn, 21, 0, sp, L)) return true;
      uint64_t E = ld_acquire(sp);
      if (F::cycle(E) == c && F::index(E) != F::kBot)         // ready (or already consumed by the owner)
        return set_fin(L, v);
      uint64_t New;
      if (!F::vacant(E)) {                                    // occupied by another cycle's element
        if (cycle_newer<16>(c, F::cycle(E)) && cycle_newer<16>(c, F::note(E))) {
          const uint64_t En = F::with_note(E, c);             // later helpers make the same decision
          if (cas_relaxed(sp, E, En) != E) continue;
          E = En;
        }
        New = F::unsafe(E);
      } else {
        New = F::advanced(E, c);
      }
      if (cycle_newer<16>(c, F::cycle(E)) && New != E && cas_relaxed(sp, E, New) != E) continue;
      const uint64_t T = R::counter(ld_acquire(r.tail));
      if (T <= H + 1) {
        R::catchup_tail(r, H + 1);
        if ((int64_t)ld_acquire(reinterpret_cast<const uint64_t*>(r.threshold)) < 0)   // EMPTY
          return set_fin(L, v);          // false if another helper already moved the request past H
      }
      return false;
    }
  }

  __device__ static void enqueue_slow(const RingView& r, uint64_t v, uint32_t x, uint32_t owner, uint32_t tag, uint32_t me) {
    uint64_t* L = &rec(r, owner)->localTail;
    [[maybe_unused]] uint32_t sn = 0;
    while (slow_faa<false>(r, r.tail, L, v, tag, me, (uint64_t)owner << 1)) {
      if (try_enq_slow(r, v >> S, x, L, v, owner)) break;
      if (GQ_STUCK(sn, 30, me, r.tail, r.head, L)) break;
    }
  }
  __device__ static void dequeue_slow(const RingView& r, uint64_t v, uint32_t owner, uint32_t tag, uint32_t me) {
    uint64_t* L = &rec(r, owner)->localHead;
    [[maybe_unused]] uint32_t sn = 0;
    while (slow_faa<true>(r, r.head, L, v, tag, me, ((uint64_t)owner << 1) | 1)) {
      if (try_deq_slow(r, v >> S, L, v)) break;
      if (GQ_STUCK(sn, 31, me, r.tail, r.head, L, r.threshold)) break;
    }
  }

  // Inspect one peer record ("a thread inspects one peer record every D operations");
  // accept it only if the published sequence values match.
  __device__ static void help_peer(const RingView& r, uint32_t peer, uint32_t me) {
    WfqRecord* p = rec(r, peer);
    if (!ld_acquire32(&p->pending)) return;
    const uint64_t s2 = ld_acquire(&p->seq2);
    const uint32_t is_enq = ld_relaxed32(&p->enqueue), x = ld_relaxed32(&p->index);
    const uint64_t it = ld_relaxed(&p->initTail), ih = ld_relaxed(&p->initHead);
    fence_acq_rel();
    if (ld_relaxed(&p->seq1) != s2) return;
    const uint32_t tag = (uint32_t)s2 & 0xFFFFu;
    ++rec(r, me)->n_helps;
    if (is_enq) enqueue_slow(r, local_word(it, tag), x, peer, tag, me);
    else dequeue_slow(r, local_word(ih, tag), peer, tag, me);
  }

  // ring-level enqueue of index x: bounded fast path, then the published slow path
  // have_pre/t_pre: a tail ticket the caller reserved already (D5), used by the first fast attempt.
  // cell/v (AQ side with D6): every fast attempt stores <its ticket | v> into the payload cell and
  // installs x | kWfqFast with a relaxed CAS; the slow path installs plain x behind the record's fences.
  template <bool kUniform, int kWarpFaa>
  __device__ static void ring_enq(const RingView& r, uint32_t x, uint32_t patience, uint32_t me, uint64_t* retries, uint32_t flags,
                                  bool have_pre = false, uint64_t t_pre = 0, uint64_t* cell = nullptr, uint32_t v = 0) {
    using R = Ring<F, kUniform, kWarpFaa>;
    uint64_t t = 0;
    bool have_t = false;
    if (have_pre) {                                                   // consumes one unit of patience; a ticket drawn must be tried
      if (R::try_enq(r, x, &t, flags, true, t_pre) == RING_OK) return;
      have_t = true;
      ++*retries;
    }
    for (uint32_t p = have_pre ? 1 : 0; p < patience; ++p) {
      if (cell) {
        const uint64_t tk = R::take(r, false);
        st_relaxed(cell, cell_word(tk, v));
        if (R::try_enq(r, x | kWfqFast, &t, flags | kRelaxedInstall, true, tk) == RING_OK) return;
      } else if (R::try_enq(r, x, &t, flags) == RING_OK) return;
      have_t = true;
      ++*retries;
    }
    if (cell) st_relaxed(cell, (uint64_t)v);                          // slow path: untagged word (bit 63 clear), payload before the request is published
    // Seed of the local word: a counter value strictly below every ticket the slow path can
    // obtain (a failed fast ticket, or current - 1), else the local word could return to its
    // seed after round one and a late helper's CAS would re-open that round (ABA).
    if (!have_t) t = Ring<F, kUniform, kWarpFaa>::counter(ld_acquire(r.tail)) - 1;
    WfqRecord* my = rec(r, me);
    const uint64_t s = my->seq1;
    const uint32_t tag = (uint32_t)s & 0xFFFFu;
    const uint64_t v0 = local_word(t, tag);
    // publication order of P:L284: payload fields, then sequence field and pending bit
    st_relaxed(&my->localTail, v0);
    st_relaxed(&my->initTail, t);
    st_relaxed32(&my->index, x);
    st_relaxed32(&my->enqueue, 1u);
    st_release(&my->seq2, s);
    st_release32(&my->pending, 1u);
    ++my->n_slow_enq;
    GQ_IDX_EVENT(2, r, x, t, 0, v0);
    GQ_L_EVENT(r, (uint64_t)me << 1, 'I', me, v0, x);
    enqueue_slow(r, v0, x, me, tag, me);
    // The installer may be a helper that has not reached its Threshold reset yet while this
    // owner leaves through the FIN check: re-assert the reset (idempotent) so that the enqueue
    // never returns with a stale negative Threshold (Alg. 1 L155 is part of the operation).
    Ring<F, kUniform, kWarpFaa>::reset_threshold(r);
    st_release32(&my->pending, 0u);
    st_release(&my->seq1, s + 1);
  }

  template <bool kUniform, int kWarpFaa>
  __device__ static int ring_deq(const RingView& r, uint32_t* x, uint32_t patience, uint32_t me, uint32_t nthreads,
                                 uint64_t* retries, bool probe, uint32_t flags, uint64_t* ticket = nullptr) {
    const Finalize fin{nthreads};
    uint64_t h = 0;
    bool have_h = false;
    for (uint32_t p = 0; p < patience; ++p) {
      const int s = Ring<F, kUniform, kWarpFaa>::try_deq(r, x, &h, fin, probe, flags);
      if (s != RING_RETRY) { if (ticket) *ticket = h; return s; }
      have_h = true; probe = true;
      ++*retries;
    }
    if ((int64_t)ld_relaxed(reinterpret_cast<const uint64_t*>(r.threshold)) < 0) return RING_EMPTY;
    // D1 at the slow-path entry: a slow dequeue on an empty ring burns one cooperative ticket (two
    // CAS generations on the global Head word, contended by every slow-path thread) per Threshold
    // unit before it may report EMPTY (Alg. 2), 3N-1 of them after each successful
    // enqueue.  The read-only observation Tail <= Head (Head read first) is the condition of
    // Alg. 1 L197 and lets the operation linearize as EMPTY at the Tail read instead.
    if (!(flags & kNoProbe)) {
      const uint64_t H0 = Ring<F, kUniform, kWarpFaa>::counter(ld_acquire(r.head));
      const uint64_t T0 = Ring<F, kUniform, kWarpFaa>::counter(ld_relaxed(r.tail));
      if (T0 <= H0) return RING_EMPTY;
    }
    if (!have_h) h = Ring<F, kUniform, kWarpFaa>::counter(ld_acquire(r.head)) - 1;   // seed < first ticket (see ring_enq)
    WfqRecord* my = rec(r, me);
    const uint64_t s = my->seq1;
    const uint32_t tag = (uint32_t)s & 0xFFFFu;
    const uint64_t v0 = local_word(h, tag);
    st_relaxed(&my->localHead, v0);
    st_relaxed(&my->initHead, h);
    st_relaxed32(&my->enqueue, 0u);
    st_release(&my->seq2, s);
    st_release32(&my->pending, 1u);
    ++my->n_slow_deq;
    dequeue_slow(r, v0, me, tag, me);
    st_release32(&my->pending, 0u);
    st_release(&my->seq1, s + 1);
    // result of a slow dequeue (reading W9): the slot named by the final localHead
    using R = Ring<F, kUniform, kWarpFaa>;
    const uint64_t H = ld_acquire(&my->localHead) >> S;
    if (ticket) *ticket = H;
    const uint32_t j = R::slot_of(r, H), c = R::cycle_of(r, H);
    uint64_t* sp = R::slot(r, j);
    const uint64_t E = ld_acquire(sp);
    if (F::cycle(E) == c && !F::vacant(E)) {
      fin(r, H, j, E);
      GQ_IDX_EVENT(6, r, F::index(E), H, E, 0);
      red_or_relaxed(sp, F::kConsumeMask);                   // CONSUME: linearization point
      *x = F::index(E);
      return RING_OK;
    }
    return RING_EMPTY;
  }
};

// help scheduling: every D-th operation of a thread inspects one peer, on both rings
__device__ __forceinline__ void wfq_help_threads(const WfqView& q, thread_ctx& ctx) {
  if (ctx.help_cd > 1) { --ctx.help_cd; return; }
  ctx.help_cd = q.help_delay;
  uint32_t peer = ctx.help_peer;
  if (peer >= q.nthreads) peer = 0;
  ctx.help_peer = peer + 1;
  if (peer == ctx.tid) return;
  Wf::help_peer(q.aq, peer, ctx.tid);
  Wf::help_peer(q.fq, peer, ctx.tid);
}

}  // namespace detail

// ring_enq / ring_deq are real functions shared by the AQ and the FQ side of both operations: lanes of one warp that have
// drifted apart (one still in its enqueue, one already in its dequeue; the two roles of a mixed warp) can meet inside them
// naming DIFFERENT rings, whatever the caller promised about the queue.  Inside G-WFQ the WAVEFAA therefore always groups
// lanes by counter address (kUniform = false costs one match.any per ticket).
constexpr bool kSameRing = false;

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int enqueue(const WfqView& q, thread_ctx& ctx, uint32_t v, uint64_t* retries = nullptr) {
  using namespace detail;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  wfq_help_threads(q, ctx);
  uint32_t idx;
  if (Wf::ring_deq<kSameRing, kWarpFaa>(q.fq, &idx, q.deq_patience, ctx.tid, q.nthreads, retries, (ctx.hungry & 2u) != 0, q.flags) == RING_EMPTY) {
    ctx.hungry |= 2u;
    return FULL;
  }
  ctx.hungry &= ~2u;
  GQ_IDX_EVENT(0, q.aq, idx, 0, 0, v);
  uint64_t* cell = q.data + idx;
  if (q.flags & kFencedPayload) {                                   // the paper's scheme: payload, then release-install
    st_relaxed(cell, (uint64_t)v);
    Wf::ring_enq<kSameRing, kWarpFaa>(q.aq, idx, q.enq_patience, ctx.tid, retries, q.flags);
  } else {
    Wf::ring_enq<kSameRing, kWarpFaa>(q.aq, idx, q.enq_patience, ctx.tid, retries, q.flags, false, 0, cell, v);
  }
  return OK;
}

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int dequeue(const WfqView& q, thread_ctx& ctx, uint32_t* out, uint64_t* retries = nullptr) {
  using namespace detail;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  wfq_help_threads(q, ctx);
  uint32_t idx;
  if (Wf::ring_deq<kSameRing, kWarpFaa>(q.aq, &idx, q.deq_patience, ctx.tid, q.nthreads, retries, (ctx.hungry & 1u) != 0, q.flags, &ctx.last_ticket) == RING_EMPTY) {
    ctx.hungry |= 1u;
    return EMPTY;
  }
  ctx.hungry &= ~1u;
  const bool fast = (idx & kWfqFast) != 0;                          // installed by a fast-path enqueue (D6)
  idx &= kWfqIdxMask;
  const uint64_t* cell = q.data + idx;
  uint64_t w = ld_relaxed(cell);
  // D5 as in G-LFQ: the FQ tail ticket is reserved behind the payload load (only when a fast attempt
  // exists to use it).  D6, FQ side: the index goes back into FQ after the payload load has
  // delivered its value (control dependency), so the fast-path install needs no release fence.
  const bool paired = !(q.flags & kNoPairedFaa) && q.enq_patience != 0 && q.enq_patience != 0xFFFFFFFFu;
  uint64_t t = 0;
  if (paired) t = Ring<WfqFmt, kSameRing, kWarpFaa>::take(q.fq, false);
  if (fast) w = cell_await(cell, w, ctx.last_ticket);               // tagged cell: wait for the store of THIS tenure of idx
  *out = (uint32_t)w;
  GQ_IDX_EVENT(7, q.aq, idx, ctx.last_ticket, w, fast);
  const uint32_t fl = (q.flags & kFencedPayload) ? q.flags : (q.flags | kRelaxedInstall);
  Wf::ring_enq<kSameRing, kWarpFaa>(q.fq, idx, q.enq_patience, ctx.tid, retries, fl, paired, t);
  return OK;
}

}  // namespace gq
