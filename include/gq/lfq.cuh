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
  uint32_t* data;     // Data[n], uint32 payloads
  uint32_t capacity;  // n
  uint32_t flags;     // GQ_F_*
};

namespace detail {

template <class F, bool kUniform, bool kWarpFaa, class Fin>
__device__ __forceinline__ int ring_deq_loop(const RingView& r, uint32_t* idx, uint64_t* retries, const Fin& fin,
                                             bool probe, uint32_t flags, uint64_t* ticket = nullptr) {
  Backoff bo;
  uint32_t sn = 0;
  for (;;) {
    uint64_t h;
    if (stuck(sn, 1, 0, ld_relaxed(r.head), ld_relaxed(r.tail))) return RING_EMPTY;
    const int s = Ring<F, kUniform, kWarpFaa>::try_deq(r, idx, &h, fin, probe, flags);
    if (s != RING_RETRY) { if (ticket) *ticket = h; return s; }
    ++*retries;
    probe = true;
    bo.pause();
  }
}
template <class F, bool kUniform, bool kWarpFaa>
__device__ __forceinline__ void ring_enq_loop(const RingView& r, uint32_t idx, uint64_t* retries, uint32_t flags) {
  Backoff bo;
  uint32_t sn = 0;
  for (;;) {
    uint64_t t;
    if (stuck(sn, 2, 0, ld_relaxed(r.head), ld_relaxed(r.tail))) return;
    if (Ring<F, kUniform, kWarpFaa>::try_enq(r, idx, &t, flags) == RING_OK) return;
    ++*retries;
    bo.pause();
  }
}

}  // namespace detail

// kUniform: all lanes converged at the call name the same queue (see warp_faa).
template <bool kUniform = false, bool kWarpFaa = true>
__device__ __forceinline__ int enqueue(const LfqView& q, thread_ctx& ctx, uint32_t v, uint64_t* retries = nullptr) {
  using namespace detail;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  uint32_t idx;
  if (ring_deq_loop<LfqFmt, kUniform, kWarpFaa>(q.fq, &idx, retries, NoFinalize{}, (ctx.hungry & 2u) != 0, q.flags) == RING_EMPTY) {
    ctx.hungry |= 2u;
    return FULL;
  }
  ctx.hungry &= ~2u;
  st_relaxed32(q.data + idx, v);                                   // ordered before the release CAS below
  ring_enq_loop<LfqFmt, kUniform, kWarpFaa>(q.aq, idx, retries, q.flags);
  return OK;
}

template <bool kUniform = false, bool kWarpFaa = true>
__device__ __forceinline__ int dequeue(const LfqView& q, thread_ctx& ctx, uint32_t* out, uint64_t* retries = nullptr) {
  using namespace detail;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  uint32_t idx;
  if (ring_deq_loop<LfqFmt, kUniform, kWarpFaa>(q.aq, &idx, retries, NoFinalize{}, (ctx.hungry & 1u) != 0, q.flags, &ctx.last_ticket) == RING_EMPTY) {
    ctx.hungry |= 1u;
    return EMPTY;
  }
  ctx.hungry &= ~1u;
  *out = ld_relaxed32(q.data + idx);                               // after the acquire load of the entry
  ring_enq_loop<LfqFmt, kUniform, kWarpFaa>(q.fq, idx, retries, q.flags);   // release CAS: the read above is done
  return OK;
}

}  // namespace gq
