// gq/ymc.cuh — G-WFQ-YMC: the wait-free queue of Yang and Mellor-Crummey [5] on a
// preallocated cell pool (§III-A).
//
// PAPER.md does not restate the algorithm ("The queue logic, helping structure, and
// linearization behavior follow Yang and Mellor-Crummey's algorithm [5]", L83); what follows
// is this library's own restatement of [5] (reading Y1), with the GPU adaptation the
// paper describes: "pre-allocate a segment pool on the device and replace dynamic segment
// growth ... with direct arithmetic lookup into the pre-allocated pool" (L83).  cell(i) =
// pool[i]; segments are logical only, there are no next pointers, no hazard pointers and no
// reclamation (reading Y2).  Cells are never reused, so the pool bounds the number of tickets
// a queue can serve between two resets; when it runs out enqueue returns FULL, dequeue
// returns EMPTY and *exhausted is set (reading Y3, the limitation stated at L84).
//
// Words (reading Y4/Y5) — every concurrently modified word is one native 32/64-bit atomic:
//   cell.val : 0 = bot, ~0 = top, (1<<32)|v = payload v
//   cell.enq : 0 = bot_e, ~0 = top_e, t+1 = enqueue request of thread t
//   cell.deq : 0 = bot_d, ~0 = top_d, t+1 = dequeue request of thread t
//   request state : [63] pending | [62:0] id (enqueue) / idx (dequeue)
// Tickets come from T and H with the warp-batched FAA (reading Y7; GQ_F_PER_LANE_FAA = one
// FAA per thread for the ablation).
//
// Two bounded additions, the same as on the rings and switchable with the same flags
// (DESIGN.md departures D1/D2): a dequeuer whose cell is still bot waits on that cell for at
// most park_ns before it marks it top, and a dequeuer whose last attempt came back EMPTY
// probes H and T read-only and returns EMPTY without burning a cell when H is already
// park_limit tickets ahead of T.
#pragma once
#include "lfq.cuh"

namespace gq {

struct alignas(16) YmcCell { uint64_t val; uint32_t enq, deq; };
static_assert(sizeof(YmcCell) == 16, "two cells per 32-byte L2 sector");

// One 128-byte line per thread: its two request records (shared) and its helping state (private).
struct alignas(128) YmcHandle {
  uint64_t enq_val;       // enqueue request: encoded payload            (shared)
  uint64_t enq_state;     //                  pending | id               (shared, CAS)
  uint64_t deq_id;        // dequeue request: id                         (shared)
  uint64_t deq_state;     //                  pending | idx              (shared, CAS)
  uint64_t enq_help_id;   // id of the peer request this thread failed to place (private)
  uint32_t enq_peer, deq_peer;                       // next peers to help (private)
  uint32_t n_slow_enq, n_slow_deq, n_helps, _r0;     // statistics (private)
  uint64_t _pad[8];
};
static_assert(sizeof(YmcHandle) == 128, "one L2 line per handle");

struct YmcView {
  YmcCell* pool;          // pool_cells cells; the last one is a pre-sealed sentinel
  uint64_t pool_cells;
  uint64_t* tail;         // T, own line
  uint64_t* head;         // H, own line
  YmcHandle* handles;     // nthreads handles
  uint64_t* exhausted;    // set to 1 when a ticket ran past the pool
  uint32_t nthreads;      // handle ring size k (reading Y6)
  uint32_t enq_patience, deq_patience, help_delay;
  uint32_t flags;
  uint32_t park_ns, park_limit, park_nap, _pad;
  detail::BlockFunnel* fhead;   // block-level ticket funnels of the calling block (D11), or nullptr
  detail::BlockFunnel* ftail;
};

namespace detail {

struct Ymc {
  static constexpr uint64_t kBot = 0, kTop = ~0ull, kEmptyRet = ~0ull - 1;   // kEmptyRet: return code only
  static constexpr uint32_t kBot32 = 0, kTop32 = ~0u;
  static constexpr uint64_t kPending = 1ull << 63;
  static constexpr uint64_t kNoId = ~0ull >> 1;          // "no request remembered" / withdrawn request
  __device__ __forceinline__ static uint64_t enc(uint32_t v) { return (1ull << 32) | v; }
  __device__ __forceinline__ static bool is_value(uint64_t w) { return w != kBot && w != kTop; }
  __device__ __forceinline__ static uint64_t id_of(uint64_t s) { return s & ~kPending; }
  __device__ __forceinline__ static uint64_t last(const YmcView& q) { return q.pool_cells - 1; }
  __device__ __forceinline__ static YmcCell* cell(const YmcView& q, uint64_t i) {
    return q.pool + (i < q.pool_cells ? i : q.pool_cells - 1);      // clamp: the sentinel is sealed
  }
  __device__ __forceinline__ static uint32_t next(const YmcView& q, uint32_t p) { return p + 1 < q.nthreads ? p + 1 : 0; }

  template <bool kUniform, int kWarpFaa>
  __device__ __forceinline__ static uint64_t take(uint64_t* ctr, BlockFunnel* f = nullptr) {
    return kWarpFaa ? warp_faa<kUniform>(ctr, 1, kWarpFaa == 2 ? f : nullptr) : lane_faa(ctr);
  }
  // [5] advance_end_for_linearizability: E <- max(E, cid), one native atom.max
  __device__ __forceinline__ static void advance(uint64_t* E, uint64_t cid) {
    if (ld_relaxed(E) < cid) red_max_relaxed(E, cid);
  }
  // [5] enq_commit: make T cover the cell, then deposit the value
  __device__ __forceinline__ static void enq_commit(const YmcView& q, YmcCell* c, uint64_t v, uint64_t cid) {
    advance(q.tail, cid + 1);
    st_release(&c->val, v);
  }
  __device__ __forceinline__ static void pool_exhausted(const YmcView& q) {
    if (!ld_relaxed(q.exhausted)) st_relaxed(q.exhausted, 1);
  }

  // [5] help_enq: what a dequeuer (or a dequeue helper) does on cell i.  Returns the value
  // word, kTop ("no value will be taken here by me: retry") or kEmptyRet.
  __device__ static uint64_t help_enq(const YmcView& q, uint32_t me, uint64_t i, uint32_t park_ns) {
    if (i >= last(q)) { pool_exhausted(q); return kEmptyRet; }
    YmcCell* c = cell(q, i);
    uint64_t w = ld_acquire(&c->val);
    if (w == kBot && park_ns && (q.flags & kEagerEmpty) && ld_relaxed(q.tail) <= i) park_ns = 0;   // no enqueuer holds cell i yet
    const uint32_t nap_cap = q.park_nap < 32 ? 32u : q.park_nap;
    for (uint32_t waited = 0, nap = 32; w == kBot && waited < park_ns; waited += nap, nap = nap * 2 < nap_cap ? nap * 2 : nap_cap) {
      __nanosleep(nap);                                       // D2: bounded wait on the own cell
      w = ld_acquire(&c->val);
    }
    if (w == kBot) w = cas_acq_rel(&c->val, kBot, kTop);      // bot -> top: no fast enqueue will land here
    if (is_value(w)) return w;
    // c->val is top: help slow-path enqueues
    YmcHandle* h = q.handles + me;
    uint32_t e = ld_acquire32(&c->enq);
    if (e == kBot32) {
      uint32_t p; uint64_t s;
      for (;;) {                                              // at most two iterations
        p = h->enq_peer < q.nthreads ? h->enq_peer : 0;
        s = ld_acquire(&q.handles[p].enq_state);
        if (h->enq_help_id == kNoId || h->enq_help_id == id_of(s)) break;
        h->enq_help_id = kNoId;                               // that request completed: move on
        h->enq_peer = next(q, p);
      }
      if ((s & kPending) && id_of(s) <= i && cas_acq_rel32(&c->enq, kBot32, p + 1) != kBot32)
        h->enq_help_id = id_of(s);                            // cell lost to another request: remember, retry later
      else
        h->enq_peer = next(q, p);
      if (ld_acquire32(&c->enq) == kBot32) cas_acq_rel32(&c->enq, kBot32, kTop32);   // seal
      e = ld_acquire32(&c->enq);
    }
    if (e == kTop32)                                          // no enqueue will fill this cell
      return ld_acquire(q.tail) <= i ? kEmptyRet : kTop;
    YmcHandle* r = q.handles + (e - 1);
    const uint64_t s = ld_acquire(&r->enq_state);
    const uint64_t v = ld_acquire(&r->enq_val);
    if (id_of(s) > i) {                                       // request is unsuitable for this cell
      if (ld_acquire(&c->val) == kTop && ld_acquire(q.tail) <= i) return kEmptyRet;
    } else if (cas_acq_rel(&r->enq_state, kPending | id_of(s), i) == (kPending | id_of(s)) ||
               (s == i && ld_acquire(&c->val) == kTop)) {     // claimed for this cell but not committed yet
      enq_commit(q, c, v, i);
    }
    return ld_acquire(&c->val);
  }

  // [5] help_deq: complete the dequeue request of thread `ph`.
  __device__ static void help_deq(const YmcView& q, uint32_t me, uint32_t ph) {
    YmcHandle* r = q.handles + ph;
    uint64_t s = ld_acquire(&r->deq_state);
    const uint64_t id = ld_acquire(&r->deq_id);
    if (!(s & kPending) || id_of(s) < id) return;
    s = ld_acquire(&r->deq_state);
    uint64_t prior = id, i = id, cand = 0;
    [[maybe_unused]] uint32_t sn = 0;
    for (;;) {
      if (GQ_STUCK(sn, 40, me, &r->deq_state, &r->deq_id, q.head, q.tail)) return;
      while (!cand && id_of(s) == prior) {                    // look for a candidate cell
        if (GQ_STUCK(sn, 41, me, &r->deq_state, &r->deq_id, q.head, q.tail)) return;
        ++i;
        const uint64_t w = help_enq(q, me, i, 0);
        if (w == kEmptyRet || (w != kTop && ld_acquire32(&cell(q, i)->deq) == kBot32)) cand = i;
        else s = ld_acquire(&r->deq_state);
      }
      if (cand) {                                             // announce it
        cas_acq_rel(&r->deq_state, kPending | prior, kPending | cand);
        s = ld_acquire(&r->deq_state);
      }
      if (!(s & kPending) || ld_acquire(&r->deq_id) != id) return;   // request complete
      YmcCell* c = cell(q, id_of(s));
      if (id_of(s) >= last(q) || ld_acquire(&c->val) == kTop ||
          cas_acq_rel32(&c->deq, kBot32, ph + 1) == kBot32 || ld_acquire32(&c->deq) == ph + 1) {
        cas_acq_rel(&r->deq_state, s, id_of(s));             // clear pending
        return;
      }
      prior = id_of(s);
      if (id_of(s) >= i) { cand = 0; i = id_of(s); }
    }
  }
};

}  // namespace detail

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int enqueue(const YmcView& q, thread_ctx& ctx, uint32_t v, uint64_t* retries = nullptr) {
  using namespace detail;
  using Y = Ymc;
  const uint64_t val = Y::enc(v);
  uint64_t id = 0;
  // fast path ([5] enq_fast): ticket, then one CAS bot -> value
  for (uint32_t p = 0; p < q.enq_patience; ++p) {
    const uint64_t i = Y::take<kUniform, kWarpFaa>(q.tail, q.ftail);
    if (i >= Y::last(q)) { Y::pool_exhausted(q); return FULL; }
    // Cells are never reused, so every deposit CAS would be the first touch of its line: an L2 miss
    // that the atomic unit of that slice waits out, and with it every other atomic queued there, the FAAs on
    // H and T included (ncu: the wait for the dequeue's FAA was 9x that of the enqueue's).  Tickets are
    // sequential, so the line a later wave of tickets will use is known: pull it into L2 one wave
    // (k tickets) ahead.  A hint only; GQ_F_NO_CELL_PREFETCH switches it off.  Measured on B200:
    // 28.4 -> 43.9 Gops/s at 65 536 threads, 24.8 -> 39.6 at full co-residency.
    if (!(q.flags & kNoCellPrefetch)) {
      const uint64_t j = i + q.nthreads;
      if (j < Y::last(q)) asm volatile("prefetch.global.L2 [%0];" :: "l"(q.pool + j));
    }
    // relaxed: the word carries the payload itself and the fast path has published nothing else
    // (the slow path's request record keeps its release/acquire discipline)
    if (cas_relaxed(&Y::cell(q, i)->val, Y::kBot, val) == Y::kBot) return OK;
    id = i;
    if (retries) ++*retries;
    // The cell was burnt by a dequeuer that found it empty, so Head has passed it: jump Tail over
    // the whole burnt stretch at once (reading Y9) instead of drawing and failing on each cell.
    Y::advance(q.tail, ld_acquire(q.head));
  }
  if (q.enq_patience == 0) {                                  // all-slow build: the id is a fresh, unused ticket
    id = Y::take<kUniform, kWarpFaa>(q.tail);
    if (id >= Y::last(q)) { Y::pool_exhausted(q); return FULL; }
  }
  // slow path ([5] enq_slow): publish the request, keep drawing cells until it is claimed
  YmcHandle* h = q.handles + ctx.tid;
  ++h->n_slow_enq;
  st_release(&h->enq_val, val);                               // payload first, then the state word (P:L284 discipline)
  st_release(&h->enq_state, Y::kPending | id);
  [[maybe_unused]] uint32_t sn = 0;
  do {
    if (GQ_STUCK(sn, 42, ctx.tid, &h->enq_state, q.head, q.tail)) break;
    const uint64_t i = Y::take<false, kWarpFaa>(q.tail);
    if (i >= Y::last(q)) {                                    // pool ran out: withdraw unless a helper already placed it
      Y::pool_exhausted(q);
      if (cas_acq_rel(&h->enq_state, Y::kPending | id, Y::kNoId) == (Y::kPending | id)) return FULL;
      break;
    }
    YmcCell* c = Y::cell(q, i);
    if (cas_acq_rel32(&c->enq, Y::kBot32, ctx.tid + 1) == Y::kBot32 && ld_acquire(&c->val) == Y::kBot) {
      cas_acq_rel(&h->enq_state, Y::kPending | id, i);        // claim the request for cell i
      break;                                                  // claimed, by this CAS or by a helper's
    }
    Y::advance(q.tail, ld_acquire(q.head));                   // reading Y9, as on the fast path
  } while (ld_acquire(&h->enq_state) & Y::kPending);
  const uint64_t cid = Y::id_of(ld_acquire(&h->enq_state));
  Y::enq_commit(q, Y::cell(q, cid), val, cid);
  return OK;
}

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int dequeue(const YmcView& q, thread_ctx& ctx, uint32_t* out, uint64_t* retries = nullptr) {
  using namespace detail;
  using Y = Ymc;
  // deq_patience 0 (all-slow build): the cell a dequeuer draws must still be visited by it, or a
  // value deposited there would be lost, so one attempt remains, without parking (reading Y8).
  const uint32_t park_ns = ((q.flags & kNoDeqSpin) || q.deq_patience == 0) ? 0u : q.park_ns;
  const uint32_t attempts = q.deq_patience ? q.deq_patience : 1u;
  if (!(q.flags & kNoProbe) && (ctx.hungry & 1u)) {           // D1: read-only emptiness probe
    const uint64_t H = ld_acquire(q.head);
    const uint64_t T = ld_relaxed(q.tail);
    if (T + ((park_ns && !(q.flags & kEagerEmpty)) ? q.park_limit : 0u) <= H) return EMPTY;
  }
  uint64_t w = Y::kTop, id = 0;
  // fast path ([5] deq_fast)
  for (uint32_t p = 0; p < attempts; ++p) {
    if (p > 0 && !(q.flags & kNoProbe)) {                     // D1 again before another cell is burnt: the cell just
      const uint64_t H = ld_acquire(q.head);                  // visited was top with T beyond it (T may have been
      const uint64_t T = ld_relaxed(q.tail);                  // caught up over burnt cells, reading Y9), which says
      if (T <= H) { w = Y::kEmptyRet; break; }                // nothing about cells ahead; Tail <= Head does
    }
    const uint64_t i = Y::take<kUniform, kWarpFaa>(q.head, q.fhead);
    w = Y::help_enq(q, ctx.tid, i, park_ns);
    if (w == Y::kEmptyRet) {                                  // T <= i was observed: the queue is empty
      // Catch T up to i + 1 (reading Y9; the ring's L200 "catch up Tail" carried over).  Without it every
      // later enqueuer must draw and fail on each cell the polling dequeuers have burnt, one L2
      // round trip per cell.  No enqueuer holds a ticket in [T, i] that it has not drawn already,
      // and each of those cells still belongs to the dequeuer that drew it.
      Y::advance(q.tail, i + 1);
      break;
    }
    // the claim is decided on this one word against the helpers' CAS (help_deq); the value is already in hand: relaxed
    if (w != Y::kTop && (GQ_MUT(MUT_YMC_NO_CLAIM) || cas_relaxed32(&Y::cell(q, i)->deq, Y::kBot32, Y::kTop32) == Y::kBot32)) { ctx.last_ticket = i; break; }   // value claimed
    w = Y::kTop;
    id = i;
    if (retries) ++*retries;
  }
  YmcHandle* h = q.handles + ctx.tid;
  if (w == Y::kTop) {                                         // slow path ([5] deq_slow)
    ++h->n_slow_deq;
    st_release(&h->deq_id, id);
    st_release(&h->deq_state, Y::kPending | id);
    Y::help_deq(q, ctx.tid, ctx.tid);
    const uint64_t i = Y::id_of(ld_acquire(&h->deq_state));
    w = i >= Y::last(q) ? Y::kTop : ld_acquire(&Y::cell(q, i)->val);
    ctx.last_ticket = i;
    Y::advance(q.head, i + 1);
    if (w == Y::kTop) { w = Y::kEmptyRet; if (i < Y::last(q)) Y::advance(q.tail, i + 1); }   // reading Y9
  }
  if (w == Y::kEmptyRet) { ctx.hungry |= 1u; return EMPTY; }
  ctx.hungry &= ~1u;
  // got a value: help one peer's dequeue request ([5] dequeue epilogue), every help_delay-th time
  if (ctx.help_cd > 1) { --ctx.help_cd; }
  else {
    ctx.help_cd = q.help_delay;
    const uint32_t peer = h->deq_peer < q.nthreads ? h->deq_peer : 0;
    if (peer != ctx.tid && (ld_acquire(&q.handles[peer].deq_state) & Y::kPending)) { ++h->n_helps; Y::help_deq(q, ctx.tid, peer); }
    h->deq_peer = Y::next(q, peer);
  }
  *out = (uint32_t)w;
  return OK;
}

}  // namespace gq
