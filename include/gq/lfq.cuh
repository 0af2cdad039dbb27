// gq/lfq.cuh — G-LFQ, the lock-free bounded queue (§III-B, Alg. 1).
//
// Outer indirection ("an outer indirection layer that moves indices rather than
// payloads directly"; reading G12): two inner rings over the indices 0..n-1 plus Data[n].
//   enqueue(v): idx <- FQ.dequeue (EMPTY => FULL); Data[idx] <- v; AQ.enqueue(idx)
//   dequeue() : idx <- AQ.dequeue (EMPTY => EMPTY); v <- Data[idx]; FQ.enqueue(idx)
// Retry loops are unbounded: lock-free, not wait-free (Thm III.4).
// Linearization points (L111): the installing CAS in AQ; CONSUME in AQ; for EMPTY the first
// empty observation of the claimed head ticket.
#pragma once
#include "detail/ring.cuh"

namespace gq {

struct thread_ctx {
  uint32_t tid;          // unique per participating thread, < max_threads (record index for G-WFQ / YMC)
  uint32_t hungry = 0;   // bit 0: last dequeue came back EMPTY, bit 1: last enqueue came back FULL (probe hint, D1)
  uint32_t help_cd = 0;  // G-WFQ / YMC: operations until the next peer inspection (help delay D)
  uint32_t help_peer = 0;// next peer record to inspect
  uint64_t last_ticket = 0;  // ticket (AQ head ticket / YMC cell) of the last successful dequeue: FIFO position
};

enum : int { OK = 0, FULL = 1, EMPTY = 2 };   // == GQ_OK / GQ_FULL / GQ_EMPTY of gq.h

struct LfqView {
  RingView aq;        // allocated indices (the queue proper)
  RingView fq;        // free indices
  uint64_t* data;     // Data[n]: payload cells <ticket tag | v> (D6)
  uint32_t capacity;  // n
  uint32_t flags;     // GQ_F_*
};

namespace detail {

template <class F, bool kUniform, int kWarpFaa, class Fin>
__device__ __forceinline__ int ring_deq_loop(const RingView& r, uint32_t* idx, uint64_t* retries, const Fin& fin,
                                             bool probe, uint32_t flags, uint64_t* ticket = nullptr) {
  Backoff bo;
  [[maybe_unused]] uint32_t sn = 0;
  for (;;) {
    uint64_t h;
    if (GQ_STUCK(sn, 1, 0, r.head, r.tail)) return RING_EMPTY;
    const int s = Ring<F, kUniform, kWarpFaa>::try_deq(r, idx, &h, fin, probe, flags);
    if (s != RING_RETRY) { if (ticket) *ticket = h; return s; }
    ++*retries;
    probe = true;
    bo.pause();
  }
}
template <class F, bool kUniform, int kWarpFaa>
__device__ __forceinline__ void ring_enq_loop(const RingView& r, uint32_t idx, uint64_t* retries, uint32_t flags) {
  Backoff bo;
  [[maybe_unused]] uint32_t sn = 0;
  for (;;) {
    uint64_t t;
    if (GQ_STUCK(sn, 2, 0, r.head, r.tail)) return;
    if (Ring<F, kUniform, kWarpFaa>::try_enq(r, idx, &t, flags) == RING_OK) return;
    ++*retries;
    bo.pause();
  }
}

// Payload cells (DESIGN.md departure D6, sm_100a).  The paper's scheme (Data[idx] <- v, then publish
// idx) needs the payload store to be performed before the installing CAS, i.e. a release fence in
// front of each install: MEMBAR.ALL.GPU, which waits for every outstanding store and reduction of
// the thread and costs about two extra L2 round trips per operation on B200 (measured: 31 -> 43
// Gops/s without them).  Instead each Data cell is one 64-bit word <1 | tag | v>, tag = the low 31
// bits of the AQ tail ticket the index is installed under, and the hand-over is a handshake that
// needs no cross-location ordering:
//   enqueue : t <- AQ tail ticket; st Data[idx] <- <1 | t | v>  and  CAS-install idx at slot(t), both
//             relaxed and in flight together (a RETRY with a new ticket t' stores <1 | t' | v> again)
//   dequeue : h = the AQ head ticket that found idx (h == t); re-read Data[idx] until its tag is h
// The dequeuer may arrive before the payload; the store has already been issued, so the wait is
// bounded by memory latency, not by another thread's steps (lock-freedom is unaffected).  A tag
// can only match the store of THIS tenure of idx: stores of earlier tenures carry tickets that
// differ by less than 2^31 (FQ is FIFO, so an index is reused within about n + k tickets), and all
// of them were observed by their own dequeuers, hence performed, before idx was recycled.  Bit 63
// marks a tagged word: a freshly formatted cell (0) and a cell written by G-WFQ's slow path
// (<0 | 0 | v>) match no ticket.  idx goes back into FQ only after the matching load has returned
// its value (control dependency), so the next owner's store cannot be read by it.
// GQ_F_FENCED_PAYLOAD restores release CAS on both sides.
__device__ __forceinline__ uint64_t cell_word(uint64_t ticket, uint32_t v) {
  return (1ull << 63) | ((ticket & 0x7FFFFFFFull) << 32) | v;
}
__device__ __forceinline__ uint32_t cell_tag(uint64_t ticket) { return 0x80000000u | (uint32_t)(ticket & 0x7FFFFFFFull); }
// dequeue side of the handshake: w = first load of the cell (already issued by the caller)
__device__ __forceinline__ uint64_t cell_await(const uint64_t* cell, uint64_t w, uint64_t ticket) {
  const uint32_t tag = cell_tag(ticket);
  [[maybe_unused]] uint32_t sn = 0;
  for (uint32_t nap = 0; (uint32_t)(w >> 32) != tag; nap = nap ? (nap < 256 ? nap * 2 : 256) : 32) {   // payload still in flight
    if (GQ_MUT(MUT_NO_HANDSHAKE) || GQ_MUT(MUT_WRONG_CELL) || GQ_MUT(MUT_EARLY_RECYCLE) || GQ_STUCK(sn, 5, 0, cell)) break;
    if (nap) __nanosleep(nap);
    w = ld_relaxed(cell);
  }
  return w;
}

}  // namespace detail

// kUniform: all lanes converged at the call name the same queue (see warp_faa).
template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int enqueue(const LfqView& q, thread_ctx& ctx, uint32_t v, uint64_t* retries = nullptr) {
  using namespace detail;
  using R = Ring<LfqFmt, kUniform, kWarpFaa>;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  uint32_t idx;
  GQ_TIC(t_op);
  if (ring_deq_loop<LfqFmt, kUniform, kWarpFaa>(q.fq, &idx, retries, NoFinalize{}, (ctx.hungry & 2u) != 0, q.flags) == RING_EMPTY) {
    ctx.hungry |= 2u;
    return FULL;
  }
  ctx.hungry &= ~2u;
  uint64_t* cell = q.data + idx;
  if (q.flags & kFencedPayload) {
    st_relaxed(cell, v);                                           // ordered before the release CAS below
    ring_enq_loop<LfqFmt, kUniform, kWarpFaa>(q.aq, idx, retries, q.flags);
    return OK;
  }
  Backoff bo;
  [[maybe_unused]] uint32_t sn = 0;
  for (;;) {
    if (GQ_STUCK(sn, 3, ctx.tid, q.aq.head, q.aq.tail)) return OK;
    GQ_TIC(t0);
    const uint64_t t = R::take(q.aq, false);
    GQ_TOC(LAT_TAIL_FAA, t0, t);
    if (!GQ_MUT(MUT_NO_HANDSHAKE)) st_relaxed(cell, cell_word(t, v));   // D6: payload tagged with its ticket
    uint64_t tt;
    const int s = R::try_enq(q.aq, idx, &tt, q.flags | kRelaxedInstall, true, t);
    if (GQ_MUT(MUT_NO_HANDSHAKE)) st_relaxed(cell, cell_word(t, v));
    if (s == RING_OK) { GQ_TOC(LAT_ENQUEUE, t_op, tt); return OK; }
    ++*retries;
    bo.pause();
  }
}

// D5 (sm_100a): once the index is known the dequeuer will certainly enqueue it into FQ, so the
// FQ tail ticket is reserved while the payload load is still in flight: the two L2 round trips
// overlap.  No speculation (the ticket is always used at once) and no waiting on another thread
// while it is held.  GQ_F_NO_PAIRED_FAA restores load-then-reserve.
template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int dequeue(const LfqView& q, thread_ctx& ctx, uint32_t* out, uint64_t* retries = nullptr) {
  using namespace detail;
  using R = Ring<LfqFmt, kUniform, kWarpFaa>;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  uint32_t idx;
  GQ_TIC(t_op);
  if (ring_deq_loop<LfqFmt, kUniform, kWarpFaa>(q.aq, &idx, retries, NoFinalize{}, (ctx.hungry & 1u) != 0, q.flags, &ctx.last_ticket) == RING_EMPTY) {
    ctx.hungry |= 1u;
    return EMPTY;
  }
  ctx.hungry &= ~1u;
  const bool fenced = (q.flags & kFencedPayload) != 0;
  const uint32_t fl = fenced ? q.flags : (q.flags | kRelaxedInstall);
  const uint64_t* cell = q.data + ((GQ_MUT(MUT_WRONG_CELL) && (idx ^ 1u) < q.capacity) ? (idx ^ 1u) : idx);
  if (GQ_MUT(MUT_EARLY_RECYCLE)) ring_enq_loop<LfqFmt, kUniform, kWarpFaa>(q.fq, idx, retries, fl);
  GQ_TIC(t0);
  uint64_t w = ld_relaxed(cell);                                   // after the acquire load of the entry
  const bool paired = !(q.flags & kNoPairedFaa) && !GQ_MUT(MUT_EARLY_RECYCLE);
  uint64_t t = 0;
  if (paired) t = R::take(q.fq, false);                              // D5: issued behind the payload load
  if (!fenced) w = cell_await(cell, w, ctx.last_ticket);
  GQ_TOC(LAT_PAYLOAD, t0, w + t);
  *out = (uint32_t)w;
  if (GQ_MUT(MUT_EARLY_RECYCLE)) return OK;
  uint64_t tt;
  if (paired) {
    if (R::try_enq(q.fq, idx, &tt, fl, true, t) == RING_OK) { GQ_TOC(LAT_DEQUEUE, t_op, tt); return OK; }
    ++*retries;
  }
  ring_enq_loop<LfqFmt, kUniform, kWarpFaa>(q.fq, idx, retries, fl);
  return OK;
}


namespace detail {
// Per-lane choice between the two rings of ONE queue.  Only the fields that differ between AQ and FQ are selected (entries,
// hot words, id, funnels); sizes, the Threshold reset value and the parking constants are the same for both rings (one N, one
// gq_opts) and stay warp-uniform kernel parameters.  (Selecting whole RingViews per lane cost the fused operations a 48-byte
// stack frame: 1.1 sectors of local-memory stores per operation in the ncu capture.)
__device__ __forceinline__ RingView pick_ring(bool first, const RingView& a, const RingView& b) {
  RingView r = a;
  r.entry = first ? a.entry : b.entry;
  r.head = first ? a.head : b.head;
  r.tail = first ? a.tail : b.tail;
  r.threshold = first ? a.threshold : b.threshold;
  r.id = first ? a.id : b.id;
  r.fhead = first ? a.fhead : b.fhead;
  r.ftail = first ? a.ftail : b.ftail;
  return r;
}
}  // namespace detail

// Fused operation for warps whose lanes have different roles (BASELINE.json config 3: the role of every
// thread is drawn from the seed, so every warp is a mix of producers and consumers).  Called as two
// separate operations the two groups of a warp run one after the other (SIMT divergence) and their
// WAVEFAA batches are half-size.  But on the rings the two operations are the same program:
//     enqueue: ring_deq(FQ) -> payload store -> ring_enq(AQ)      dequeue: ring_deq(AQ) -> payload load -> ring_enq(FQ)
// so here every lane selects its (first ring, second ring) pair and the whole warp stays converged;
// the address-matched WAVEFAA (warp_faa<false>, reading G10) elects one leader per counter inside the
// converged warp, both leaders issue their FAA in the same instruction, and the L2 round trips of the
// two roles overlap.  *v is the payload (in) for is_enq lanes and the result (out) for the others.
// Returns OK, FULL (enqueue lanes) or EMPTY (dequeue lanes).  Ticket-tagged cells (D6) only; with
// GQ_F_FENCED_PAYLOAD it falls back to the two separate calls.
template <int kWarpFaa = true>
__device__ __forceinline__ int enqueue_or_dequeue(const LfqView& q, thread_ctx& ctx, bool is_enq, uint32_t* v, uint64_t* retries = nullptr) {
  using namespace detail;
  using R = Ring<LfqFmt, false, kWarpFaa>;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  if (q.flags & kFencedPayload) return is_enq ? enqueue<false, kWarpFaa>(q, ctx, *v, retries) : dequeue<false, kWarpFaa>(q, ctx, v, retries);
  const RingView r1 = pick_ring(is_enq, q.fq, q.aq), r2 = pick_ring(is_enq, q.aq, q.fq);   // per-lane ring pair
  const uint32_t hbit = is_enq ? 2u : 1u;
  uint32_t idx;
  uint64_t h1 = 0;
  if (ring_deq_loop<LfqFmt, false, kWarpFaa>(r1, &idx, retries, NoFinalize{}, (ctx.hungry & hbit) != 0, q.flags, &h1) == RING_EMPTY) {
    ctx.hungry |= hbit;
    return is_enq ? FULL : EMPTY;
  }
  ctx.hungry &= ~hbit;
  if (!is_enq) ctx.last_ticket = h1;
  uint64_t* cell = q.data + idx;
  uint64_t w = is_enq ? 0 : ld_relaxed(cell);
  Backoff bo;
  [[maybe_unused]] uint32_t sn = 0;
  for (bool first = true;; first = false) {
    if (GQ_STUCK(sn, 4, ctx.tid, r2.head, r2.tail)) return OK;
    const uint64_t t = R::take(r2, false);                               // two leaders, one instruction
    if (is_enq) {
      st_relaxed(cell, cell_word(t, *v));                              // D6: payload tagged with its AQ ticket
    } else if (first) {
      w = cell_await(cell, w, h1);
      *v = (uint32_t)w;
    }
    uint64_t tt;
    if (R::try_enq(r2, idx, &tt, q.flags | kRelaxedInstall, true, t) == RING_OK) return OK;
    ++*retries;
    bo.pause();
  }
}

// The same fused operation with the wait handed back to the caller (D12).  enqueue_or_dequeue keeps a converged
// warp together, but a lane that has to wait in line (an enqueuer for a free index when the queue is full, a dequeuer for an
// item when it is empty: D2) then holds up the 31 others, and at p = 0.5 BASELINE.json's split benchmark sits at one of the
// two boundaries for most of its run.  Here a lane whose slot is still vacant returns PENDING at once, keeps its ticket in
// `st`, and looks at the slot again on its next call, while the other lanes of the warp complete whole operations: one
// converged chain of L2 round trips per call whatever the number of lanes that wait.
// Contract: after PENDING the thread must call again with the same `st`, role and *v until it gets another result (it holds
// a ticket; the enqueuer of that ticket will install an entry for it).  The operation's interval in a history runs from
// its first call to the call that completes it.  The parking budget (gq_opts.park_ns) runs in real time from the first call.
using op_state = detail::DeqWait;
enum : int { PENDING = 3 };
template <int kWarpFaa = true>
__device__ __forceinline__ int enqueue_or_dequeue_step(const LfqView& q, thread_ctx& ctx, op_state& st, bool is_enq, uint32_t* v,
                                                       uint64_t* retries = nullptr) {
  using namespace detail;
  using R = Ring<LfqFmt, false, kWarpFaa>;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  if (q.flags & kFencedPayload) return is_enq ? enqueue<false, kWarpFaa>(q, ctx, *v, retries) : dequeue<false, kWarpFaa>(q, ctx, v, retries);
  const RingView r1 = pick_ring(is_enq, q.fq, q.aq), r2 = pick_ring(is_enq, q.aq, q.fq);   // per-lane ring pair
  const uint32_t hbit = is_enq ? 2u : 1u;
  uint32_t idx = 0;
  uint64_t h1 = 0;
  int s;
  GQ_TIC(t_op);
  {
    Backoff bo;
    [[maybe_unused]] uint32_t sn = 0;
    bool probe = (ctx.hungry & hbit) != 0;
    for (;;) {
      if (GQ_STUCK(sn, 6, ctx.tid, r1.head, r1.tail)) { s = RING_EMPTY; break; }
      s = R::try_deq(r1, &idx, &h1, NoFinalize{}, probe, q.flags, &st);
      if (s != RING_RETRY) break;
      st.clear();                                                      // that ticket is spent: next attempt draws a new one
      ++*retries;
      probe = true;
      bo.pause();
    }
  }
  if (s == RING_PENDING) { GQ_TOC(is_enq ? LAT_STEP_PENDING_ENQ : LAT_STEP_PENDING_DEQ, t_op, h1); return PENDING; }
  st.clear();
  if (s == RING_EMPTY) {
    ctx.hungry |= hbit;
    return is_enq ? FULL : EMPTY;
  }
  ctx.hungry &= ~hbit;
  if (!is_enq) ctx.last_ticket = h1;
  uint64_t* cell = q.data + idx;
  uint64_t w = is_enq ? 0 : ld_relaxed(cell);
  Backoff bo;
  [[maybe_unused]] uint32_t sn = 0;
  for (bool first = true;; first = false) {
    if (GQ_STUCK(sn, 4, ctx.tid, r2.head, r2.tail)) return OK;
    const uint64_t t = R::take(r2, false);                               // one leader per counter, one instruction
    if (is_enq) {
      st_relaxed(cell, cell_word(t, *v));                              // D6: payload tagged with its AQ ticket
    } else if (first) {
      w = cell_await(cell, w, h1);
      *v = (uint32_t)w;
    }
    uint64_t tt;
    if (R::try_enq(r2, idx, &tt, q.flags | kRelaxedInstall, true, t) == RING_OK) { GQ_TOC(is_enq ? LAT_ENQUEUE : LAT_DEQUEUE, t_op, tt); return OK; }
    ++*retries;
    bo.pause();
  }
}

}  // namespace gq
