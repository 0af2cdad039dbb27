// gq/ymc.cuh — G-WFQ-YMC: the wait-free queue of Yang and Mellor-Crummey [5] on a
// preallocated cell pool (§III-A), with the pool used as a RING (Y10).
//
// PAPER.md does not restate the algorithm ("The queue logic, helping structure, and
// linearization behavior follow Yang and Mellor-Crummey's algorithm [5]", L83); what follows
// is this library's own restatement of [5] (reading Y1), with the GPU adaptation the
// paper describes: "pre-allocate a segment pool on the device and replace dynamic segment
// growth ... with direct arithmetic lookup into the pre-allocated pool" (L83).  There are no
// next pointers, no hazard pointers and no reclamation pass.
//
// The paper's version never reuses a cell ("not bounded-memory in the strict sense", L84): a queue
// that runs at 45 Gops/s eats 64 GiB of cells in 0.2 s.  Here cell(i) = pool[i mod P] and every cell
// is reused once per lap of the pool.  What makes that safe:
//   * all three words of [5]'s cell (val, enq, deq) live in ONE 64-bit state word together with the
//     lap number (epoch) of the ticket the cell currently serves:
//         [63:40] epoch (24) | [37:36] V: bot / top / value | [35:18] E: bot_e / top_e / tid+1 | [17:0] D: bot_d / top_d / tid+1
//     Every transition of [5] is one CAS on that word, so an operation (a stalled helper above all) whose ticket
//     belongs to an earlier lap can never change a recycled cell: its CAS fails, it sees a newer epoch and gives up;
//   * a cell of lap e-1 is taken over by lap e (one CAS, folded into the first transition of lap e) only when it is
//     FINAL: value consumed (V = value, D = top_d), or burnt and sealed (V = top, E = top_e).  A value that a helper
//     claimed for a slow dequeue (D = tid+1) stays non-final until its owner has read it and acknowledged (D <- top_d);
//   * the 32-bit payload sits in a second word <1 | ticket tag | v> that is written by exactly one thread, the
//     winner of the CAS that set V = value, AFTER that CAS; a dequeuer reads it (waiting for the tag, as in D6)
//     BEFORE it claims the cell, so the cell cannot be recycled under the writer or the reader.
// An operation that laps onto a cell whose previous use is unfinished cannot use it: an enqueuer whose ticket is
// full_limit = P - 2k or more ahead of Head abandons the ticket and returns FULL (the dequeuer that later draws it
// burns it, as it burns the cell of any enqueuer that was too slow); otherwise it was overtaken by less than a lap
// because one operation stalled, and waits for that operation: wait-freedom holds as long as no operation is
// overtaken by a whole lap of the pool (Thm III.10's residency assumption makes every resident thread take steps).
// The capacity bound is therefore soft: FULL appears between n + 2k and P items, P = pow2ceil(n + 4k) unless
// gq_opts.ymc_pool_cells asks for more.
//
// Tickets come from T and H with the warp-batched FAA (reading Y7; GQ_F_PER_LANE_FAA = one
// FAA per thread for the ablation).  Two bounded additions, the same as on the rings and switchable
// with the same flags (DESIGN.md departures D1/D2): a dequeuer whose cell is still bot waits on that
// cell for at most park_ns before it marks it top, and a dequeuer whose last attempt came back EMPTY
// probes H and T read-only and returns EMPTY without burning a cell when H is already
// park_limit tickets ahead of T.
#pragma once
#include "lfq.cuh"

namespace gq {

struct alignas(16) YmcCell { uint64_t state; uint64_t data; };
static_assert(sizeof(YmcCell) == 16, "two cells per 32-byte L2 sector");

// One 128-byte line per thread: its two request records (shared) and its helping state (private).
struct alignas(128) YmcHandle {
  uint64_t enq_val;       // enqueue request: payload                    (shared)
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
  YmcCell* pool;          // P cells, P a power of two; cell(i) = pool[i mod P]
  uint64_t pool_cells;
  uint64_t* tail;         // T, own line
  uint64_t* head;         // H, own line
  YmcHandle* handles;     // nthreads handles
  uint64_t* exhausted;    // unused since the pool is a ring (kept for the layout)
  uint32_t nthreads;      // handle ring size k (reading Y6)
  uint32_t enq_patience, deq_patience, help_delay;
  uint32_t flags;
  uint32_t park_ns, park_limit, park_nap, pool_shift;   // pool_shift = log2 P
  detail::BlockFunnel* fhead;   // block-level ticket funnels of the calling block (D11), or nullptr
  detail::BlockFunnel* ftail;
  uint64_t full_limit;    // an enqueue ticket this far ahead of Head that meets an unfinished cell gives up: FULL
};

namespace detail {

struct Ymc {
  static constexpr uint64_t kPending = 1ull << 63;
  static constexpr uint64_t kNoId = ~0ull >> 1;          // "no request remembered" / withdrawn request
  // ---- the state word
  static constexpr uint32_t kIdMask = (1u << 18) - 1, kIdTop = kIdMask;     // tid + 1 <= kIdTop - 1
  static constexpr uint32_t kEpochMask = (1u << 24) - 1;
  enum : uint32_t { V_BOT = 0, V_TOP = 1, V_VAL = 2 };
  enum : int { HE_VAL = 0, HE_TOP = 1, HE_EMPTY = 2, HE_STALE = 3 };        // results of help_enq
  __device__ __forceinline__ static uint32_t ep(uint64_t w) { return (uint32_t)(w >> 40); }
  __device__ __forceinline__ static uint32_t V(uint64_t w) { return (uint32_t)(w >> 36) & 3u; }
  __device__ __forceinline__ static uint32_t E(uint64_t w) { return (uint32_t)(w >> 18) & kIdMask; }
  __device__ __forceinline__ static uint32_t D(uint64_t w) { return (uint32_t)w & kIdMask; }
  __device__ __forceinline__ static uint64_t make(uint32_t e, uint32_t v, uint32_t en, uint32_t de) {
    return ((uint64_t)e << 40) | ((uint64_t)v << 36) | ((uint64_t)en << 18) | de;
  }
  __device__ __forceinline__ static uint64_t withV(uint64_t w, uint32_t v) { return (w & ~(3ull << 36)) | ((uint64_t)v << 36); }
  __device__ __forceinline__ static uint64_t withE(uint64_t w, uint32_t en) { return (w & ~((uint64_t)kIdMask << 18)) | ((uint64_t)en << 18); }
  __device__ __forceinline__ static uint64_t withD(uint64_t w, uint32_t de) { return (w & ~(uint64_t)kIdMask) | de; }
  __device__ __forceinline__ static bool final_(uint64_t w) {
    return (V(w) == V_VAL && D(w) == kIdTop) || (V(w) == V_TOP && E(w) == kIdTop);
  }
  __device__ __forceinline__ static bool ep_newer(uint32_t a, uint32_t b) {                 // a is a later lap than b
    const uint32_t d = (a - b) & kEpochMask;
    return d != 0 && d < (1u << 23);
  }
  __device__ __forceinline__ static uint64_t id_of(uint64_t s) { return s & ~kPending; }
  __device__ __forceinline__ static YmcCell* cell(const YmcView& q, uint64_t i) { return q.pool + (i & (q.pool_cells - 1)); }
  __device__ __forceinline__ static uint32_t epoch(const YmcView& q, uint64_t i) { return (uint32_t)(i >> q.pool_shift) & kEpochMask; }
  __device__ __forceinline__ static uint32_t next(const YmcView& q, uint32_t p) { return p + 1 < q.nthreads ? p + 1 : 0; }

  template <bool kUniform, int kWarpFaa>
  __device__ __forceinline__ static uint64_t take(uint64_t* ctr, BlockFunnel* f = nullptr) {
    return kWarpFaa ? warp_faa<kUniform>(ctr, 1, kWarpFaa == 2 ? f : nullptr) : lane_faa(ctr);
  }
  // [5] advance_end_for_linearizability: E <- max(E, cid), one native atom.max
  __device__ __forceinline__ static void advance(uint64_t* E_, uint64_t cid) {
    if (ld_relaxed(E_) < cid) red_max_relaxed(E_, cid);
  }

  // The cell of ticket i as lap e sees it.  phys = the word in memory; returns the LOGICAL word of lap e:
  // phys itself when it already belongs to lap e, a fresh <e, bot, bot_e, bot_d> when phys is a finished cell of an
  // earlier lap (the take-over happens with the caller's first CAS, expected value phys).  *st: CELL_OK, CELL_BUSY
  // (earlier lap unfinished) or CELL_STALE (the cell has moved on to a later lap: the caller's ticket is history).
  enum : int { CELL_OK = 0, CELL_BUSY = 1, CELL_STALE = 2 };
  __device__ __forceinline__ static uint64_t logical(uint64_t phys, uint32_t e, int* st) {
    const uint32_t ew = ep(phys);
    if (ew == e) { *st = CELL_OK; return phys; }
    if (ep_newer(ew, e)) { *st = CELL_STALE; return phys; }
    *st = final_(phys) ? CELL_OK : CELL_BUSY;
    return make(e, V_BOT, 0, 0);
  }
  // Load the cell for lap e; while an earlier lap's use is unfinished, waits on it (naps up to 1 us) for at most
  // budget_ns (~0u = for as long as it takes; 0 = not at all) and returns CELL_BUSY when the budget is spent.
  __device__ __forceinline__ static uint64_t load_cell(YmcCell* c, uint32_t e, uint64_t* phys, int* st, bool wait, uint32_t budget_ns = ~0u) {
    [[maybe_unused]] uint32_t sn = 0;
    for (uint32_t nap = 32, waited = 0;; nap = nap < 1024 ? nap * 2 : 1024) {
      *phys = ld_acquire(&c->state);
      const uint64_t w = logical(*phys, e, st);
      if (*st != CELL_BUSY || !wait || waited >= budget_ns) return w;
      if (GQ_STUCK(sn, 43, 0, &c->state)) return w;
      __nanosleep(nap);                                       // overtaken by less than a lap: wait for the straggler
      if (budget_ns != ~0u) waited += nap + 384;
    }
  }
  // one transition of the state word: CAS(phys -> nw); on failure re-derive the logical word.  true iff this CAS made it
  // relaxed: the fast-path deposit and claim, whose payload travels by the tagged data word and orders nothing else (D6)
  __device__ __forceinline__ static bool step(YmcCell* c, uint32_t e, uint64_t* phys, uint64_t* w, uint64_t nw, int* st, bool relaxed = false) {
    const uint64_t o = relaxed ? cas_relaxed(&c->state, *phys, nw) : cas_acq_rel(&c->state, *phys, nw);
    if (o == *phys) { *phys = nw; *w = nw; *st = CELL_OK; return true; }
    *phys = o;
    *w = logical(o, e, st);
    return false;
  }

  // [5] enq_commit: make T cover the cell, then deposit the value.  Whoever turns V into value writes the payload.
  __device__ static void commit(const YmcView& q, uint64_t cid, uint32_t v) {
    YmcCell* c = cell(q, cid);
    const uint32_t e = epoch(q, cid);
    advance(q.tail, cid + 1);
    uint64_t phys; int st;
    uint64_t w = load_cell(c, e, &phys, &st, false);
    [[maybe_unused]] uint32_t sn = 0;
    while (st == CELL_OK && V(w) != V_VAL) {                  // (BUSY / STALE: not, or no longer, a cell of this request)
      if (GQ_STUCK(sn, 44, 0, &c->state)) return;
      if (step(c, e, &phys, &w, withV(w, V_VAL), &st)) { st_relaxed(&c->data, cell_word(cid, v)); return; }
    }
  }

  // [5] help_enq: what a dequeuer (or a dequeue helper) does on cell i.  *w_out = the state it ended on.
  __device__ static int help_enq(const YmcView& q, uint32_t me, uint64_t i, uint32_t park_ns, uint64_t* w_out, uint64_t* phys_out) {
    YmcCell* c = cell(q, i);
    const uint32_t e = epoch(q, i);
    uint64_t phys; int st;
    uint64_t w = load_cell(c, e, &phys, &st, true);
    if (st == CELL_STALE) return HE_STALE;
    if (V(w) == V_BOT && park_ns) {                           // D2: bounded wait on the own cell
      if ((q.flags & kEagerEmpty) && ld_relaxed(q.tail) <= i) park_ns = 0;   // no enqueuer holds cell i yet
      const uint32_t nap_cap = q.park_nap < 32 ? 32u : q.park_nap;
      for (uint32_t waited = 0, nap = 32; V(w) == V_BOT && waited < park_ns; waited += nap, nap = nap * 2 < nap_cap ? nap * 2 : nap_cap) {
        __nanosleep(nap);
        w = load_cell(c, e, &phys, &st, true);
        if (st == CELL_STALE) return HE_STALE;
      }
    }
    YmcHandle* h = q.handles + me;
    [[maybe_unused]] uint32_t sn = 0;
    for (;;) {
      if (GQ_STUCK(sn, 45, me, &c->state, q.head, q.tail)) return HE_TOP;
      if (st == CELL_STALE) return HE_STALE;
      if (st == CELL_BUSY) { w = load_cell(c, e, &phys, &st, true); continue; }
      if (V(w) == V_VAL) { *w_out = w; *phys_out = phys; return HE_VAL; }
      if (V(w) == V_BOT) { step(c, e, &phys, &w, withV(w, V_TOP), &st); continue; }   // bot -> top: no fast enqueue will land here
      // V == top: help slow-path enqueues
      const uint32_t en = E(w);
      if (en == 0) {
        uint32_t p; uint64_t s;
        for (;;) {                                            // at most two iterations
          p = h->enq_peer < q.nthreads ? h->enq_peer : 0;
          s = ld_acquire(&q.handles[p].enq_state);
          if (h->enq_help_id == kNoId || h->enq_help_id == id_of(s)) break;
          h->enq_help_id = kNoId;                             // that request completed: move on
          h->enq_peer = next(q, p);
        }
        if ((s & kPending) && id_of(s) <= i) {
          if (step(c, e, &phys, &w, withE(w, p + 1), &st)) h->enq_peer = next(q, p);
          else h->enq_help_id = id_of(s);                     // the word changed under us: remember the request, look again
        } else {
          h->enq_peer = next(q, p);
          step(c, e, &phys, &w, withE(w, kIdTop), &st);      // nobody to place: seal
        }
        continue;
      }
      if (en == kIdTop) {                                     // no enqueue will fill this cell
        *w_out = w; *phys_out = phys;
        return ld_acquire(q.tail) <= i ? HE_EMPTY : HE_TOP;
      }
      YmcHandle* r = q.handles + (en - 1);
      uint64_t s = ld_acquire(&r->enq_state);
      const uint32_t v = (uint32_t)ld_acquire(&r->enq_val);
      if ((s & kPending) && id_of(s) <= i) {                  // claim the request for this cell
        const uint64_t o = cas_acq_rel(&r->enq_state, s, i);
        s = o == s ? i : o;
      }
      if (s == i) { commit(q, i, v); w = load_cell(c, e, &phys, &st, true); continue; }   // claimed for this cell: deposit (idempotent)
      step(c, e, &phys, &w, withE(w, kIdTop), &st);          // that request will not deposit here: seal, so that the cell can be recycled
    }
  }

  // Take the value of a cell whose state shows V = value: payload first (it is written right behind the CAS that set V),
  // then the claim D: bot_d -> to.  false: another dequeuer owns the value.
  // d0 = a load of the payload word issued together with the state load.
  __device__ __forceinline__ static bool claim(YmcCell* c, uint32_t e, uint64_t i, uint64_t phys, uint64_t w, uint32_t to, uint64_t d0, uint32_t* v) {
    *v = (uint32_t)cell_await(&c->data, d0, i);
    int st = CELL_OK;
    while (st == CELL_OK && V(w) == V_VAL && D(w) == 0) {
      if (GQ_MUT(MUT_YMC_NO_CLAIM)) return true;
      if (step(c, e, &phys, &w, withD(w, to), &st, true)) return true;
    }
    return false;
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
        uint64_t w, phys;
        const int res = help_enq(q, me, i, 0, &w, &phys);
        if (res == HE_STALE) {                                // the pool has lapped cell i
          if (me != ph) return;                               // a helper that old has nothing left to help
          const uint64_t hd = ld_acquire(q.head);
          if (hd > i) i = hd - 1;
          s = ld_acquire(&r->deq_state);
          continue;
        }
        if (res == HE_EMPTY || (res == HE_VAL && D(w) == 0)) cand = i;
        else s = ld_acquire(&r->deq_state);
      }
      if (cand) {                                             // announce it
        cas_acq_rel(&r->deq_state, kPending | prior, kPending | cand);
        s = ld_acquire(&r->deq_state);
      }
      if (!(s & kPending) || ld_acquire(&r->deq_id) != id) return;   // request complete
      const uint64_t ci = id_of(s);
      YmcCell* c = cell(q, ci);
      const uint32_t e = epoch(q, ci);
      uint64_t phys; int st;
      uint64_t w = load_cell(c, e, &phys, &st, true);
      bool resolved = false;
      if (st == CELL_STALE) {                                 // recycled since it was announced: it was final, empty or taken by
        if (me != ph) return;                                 // someone else; the owner looks on from here (always safe)
      } else {
        while (st == CELL_OK && V(w) == V_BOT) step(c, e, &phys, &w, withV(w, V_TOP), &st);   // (candidates are never bot; be sure)
        while (st == CELL_OK && V(w) == V_VAL && D(w) == 0 && !step(c, e, &phys, &w, withD(w, ph + 1), &st)) {}
        resolved = st == CELL_OK && (V(w) == V_TOP || (V(w) == V_VAL && D(w) == ph + 1));     // empty result, or claimed for ph
      }
      if (resolved) { cas_acq_rel(&r->deq_state, s, ci); return; }          // clear pending
      prior = ci;
      if (ci >= i) { cand = 0; i = ci; }
    }
  }
};

}  // namespace detail

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int enqueue(const YmcView& q, thread_ctx& ctx, uint32_t v, uint64_t* retries = nullptr) {
  using namespace detail;
  using Y = Ymc;
  if (ctx.hungry & 2u) {                                      // D1 on the enqueue side: after a FULL, look before a ticket is drawn
    const uint64_t H = ld_acquire(q.head);
    const uint64_t T = ld_relaxed(q.tail);
    if (T >= H + q.full_limit) return FULL;
    ctx.hungry &= ~2u;
  }
  uint64_t id = 0;
  // fast path ([5] enq_fast): ticket, then one CAS bot -> value (which also takes the cell over from the previous lap)
  for (uint32_t p = 0; p < q.enq_patience; ++p) {
    const uint64_t i = Y::take<kUniform, kWarpFaa>(q.tail, q.ftail);
    YmcCell* c = Y::cell(q, i);
    const uint32_t e = Y::epoch(q, i);
    // steady state: the cell holds the consumed value of the previous lap; try the deposit against that word first (one round trip)
    uint64_t phys = e ? Y::make((e - 1) & Y::kEpochMask, Y::V_VAL, 0, Y::kIdTop) : Y::make(0, Y::V_BOT, 0, 0);
    int st = Y::CELL_OK;
    uint64_t w = Y::make(e, Y::V_BOT, 0, 0);
    for (;;) {
      if (st == Y::CELL_BUSY) {                               // the previous lap's item is still there
        // Wait in line on the own cell, as a dequeuer parks on its cell (D2): no load on the hot words, and the consumer that
        // frees the cell hands it over directly.  When the time is up: a lap ahead of Head means full, and the ticket is
        // abandoned (its dequeuer will burn it); otherwise a straggler holds the cell: keep waiting for it.
        w = Y::load_cell(c, e, &phys, &st, true, (q.flags & kNoDeqSpin) ? 0u : q.park_ns);
        if (st == Y::CELL_BUSY && i >= ld_acquire(q.head) + q.full_limit) { ctx.hungry |= 2u; return FULL; }
        continue;
      }
      if (st != Y::CELL_OK || w != Y::make(e, Y::V_BOT, 0, 0)) break;         // burnt by a dequeuer (or lapped): this attempt failed
      if (Y::step(c, e, &phys, &w, Y::make(e, Y::V_VAL, 0, 0), &st, true)) {
        st_relaxed(&c->data, cell_word(i, v));                // the payload follows the CAS that owns the cell (header)
        return OK;
      }
    }
    id = i;
    if (retries) ++*retries;
    // The cell was burnt by a dequeuer that found it empty, so Head has passed it: jump Tail over
    // the whole burnt stretch at once (reading Y9) instead of drawing and failing on each cell.
    Y::advance(q.tail, ld_acquire(q.head));
  }
  if (q.enq_patience == 0) id = Y::take<kUniform, kWarpFaa>(q.tail, q.ftail);   // all-slow build: the id is a fresh, unused ticket
  // slow path ([5] enq_slow): publish the request, keep drawing cells until it is claimed
  YmcHandle* h = q.handles + ctx.tid;
  ++h->n_slow_enq;
  st_release(&h->enq_val, (uint64_t)v);                       // payload first, then the state word (P:L284 discipline)
  st_release(&h->enq_state, Y::kPending | id);
  [[maybe_unused]] uint32_t sn = 0;
  do {
    if (GQ_STUCK(sn, 42, ctx.tid, &h->enq_state, q.head, q.tail)) break;
    const uint64_t i = Y::take<false, kWarpFaa>(q.tail);
    YmcCell* c = Y::cell(q, i);
    const uint32_t e = Y::epoch(q, i);
    uint64_t phys; int st;
    uint64_t w = Y::load_cell(c, e, &phys, &st, false);
    if (st == Y::CELL_BUSY) {
      if (i >= ld_acquire(q.head) + q.full_limit) {           // full: withdraw unless a helper already placed the request
        if (cas_acq_rel(&h->enq_state, Y::kPending | id, Y::kNoId) == (Y::kPending | id)) { ctx.hungry |= 2u; return FULL; }
        break;
      }
      w = Y::load_cell(c, e, &phys, &st, true);
    }
    // reserve the cell just drawn if nobody has touched it ([5]: CAS(c.enq, bot_e, me) and c.val still bot)
    if (st == Y::CELL_OK && w == Y::make(e, Y::V_BOT, 0, 0) && Y::step(c, e, &phys, &w, Y::withE(w, ctx.tid + 1), &st)) {
      cas_acq_rel(&h->enq_state, Y::kPending | id, i);        // claim the request for cell i
      break;                                                  // claimed, by this CAS or by a helper's
    }
    Y::advance(q.tail, ld_acquire(q.head));                   // reading Y9, as on the fast path
  } while (ld_acquire(&h->enq_state) & Y::kPending);
  Y::commit(q, Y::id_of(ld_acquire(&h->enq_state)), v);
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
  int res = Y::HE_TOP;
  uint64_t id = 0;
  uint32_t v = 0;
  // fast path ([5] deq_fast)
  for (uint32_t p = 0; p < attempts; ++p) {
    if (p > 0 && !(q.flags & kNoProbe)) {                     // D1 again before another cell is burnt: the cell just
      const uint64_t H = ld_acquire(q.head);                  // visited was top with T beyond it (T may have been
      const uint64_t T = ld_relaxed(q.tail);                  // caught up over burnt cells, reading Y9), which says
      if (T <= H) { res = Y::HE_EMPTY; break; }               // nothing about cells ahead; Tail <= Head does
    }
    const uint64_t i = Y::take<kUniform, kWarpFaa>(q.head, q.fhead);
    const uint64_t d0 = ld_relaxed(&Y::cell(q, i)->data);     // in flight together with the state load
    uint64_t w, phys;
    res = Y::help_enq(q, ctx.tid, i, park_ns, &w, &phys);
    if (res == Y::HE_EMPTY) {                                 // T <= i was observed: the queue is empty
      // Catch T up to i + 1 (reading Y9; the ring's L200 "catch up Tail" carried over).  Without it every
      // later enqueuer must draw and fail on each cell the polling dequeuers have burnt, one L2
      // round trip per cell.  No enqueuer holds a ticket in [T, i] that it has not drawn already,
      // and each of those cells still belongs to the dequeuer that drew it.
      Y::advance(q.tail, i + 1);
      break;
    }
    if (res == Y::HE_VAL && Y::claim(Y::cell(q, i), Y::epoch(q, i), i, phys, w, Y::kIdTop, d0, &v)) { ctx.last_ticket = i; break; }   // value claimed
    res = Y::HE_TOP;
    id = i;
    if (retries) ++*retries;
  }
  YmcHandle* h = q.handles + ctx.tid;
  if (res == Y::HE_TOP || res == Y::HE_STALE) {               // slow path ([5] deq_slow)
    ++h->n_slow_deq;
    st_release(&h->deq_id, id);
    st_release(&h->deq_state, Y::kPending | id);
    Y::help_deq(q, ctx.tid, ctx.tid);
    const uint64_t i = Y::id_of(ld_acquire(&h->deq_state));
    YmcCell* c = Y::cell(q, i);
    const uint32_t e = Y::epoch(q, i);
    uint64_t phys; int st;
    uint64_t w = Y::load_cell(c, e, &phys, &st, false);
    ctx.last_ticket = i;
    Y::advance(q.head, i + 1);
    if (st == Y::CELL_OK && Y::V(w) == Y::V_VAL && Y::D(w) == ctx.tid + 1) {   // the value the request was resolved to
      v = (uint32_t)cell_await(&c->data, ld_relaxed(&c->data), i);
      while (st == Y::CELL_OK && Y::D(w) == ctx.tid + 1 && !Y::step(c, e, &phys, &w, Y::withD(w, Y::kIdTop), &st)) {}   // read: the cell may be recycled
      res = Y::HE_VAL;
    } else {                                                  // resolved to an empty cell (top, or recycled since: it was final)
      res = Y::HE_EMPTY;
      Y::advance(q.tail, i + 1);                              // reading Y9
    }
  }
  if (res == Y::HE_EMPTY) { ctx.hungry |= 1u; return EMPTY; }
  ctx.hungry &= ~1u;
  // got a value: help one peer's dequeue request ([5] dequeue epilogue), every help_delay-th time
  if (ctx.help_cd > 1) { --ctx.help_cd; }
  else {
    ctx.help_cd = q.help_delay;
    const uint32_t peer = h->deq_peer < q.nthreads ? h->deq_peer : 0;
    if (peer != ctx.tid && (ld_acquire(&q.handles[peer].deq_state) & Y::kPending)) { ++h->n_helps; Y::help_deq(q, ctx.tid, peer); }
    h->deq_peer = Y::next(q, peer);
  }
  *out = v;
  return OK;
}

}  // namespace gq
