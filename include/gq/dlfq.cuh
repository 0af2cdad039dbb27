// gq/dlfq.cuh — G-LFQ-D: the direct-payload, single-ring variant of G-LFQ.
//
// An ABLATION, not the paper's queue: PAPER.md L88 moves indices through an outer indirection layer
// (FQ + AQ + Data); here the uint32 payload itself is installed in the one ring's entry word.  What
// stays is Algorithm 1 unchanged (TRYENQ / TRYDEQ / WAVEFAA of ring.cuh on the DirFmt entry word);
// what goes is half of the work per operation: one ticket, one slot atomic and no payload cell
// per enqueue or dequeue.  What is lost is the exact capacity bound, which the indirection gives for
// free (n indices circulate): here FULL is decided by a read-only test, Tail - Head >= n, before the
// ticket is drawn, so up to one enqueue per concurrent thread can pass the test together and the
// queue holds at most n + k items for a moment (k = participating threads; the ring has 2N >= n + k
// slots, so nothing is overwritten).  EMPTY is strict, as in G-LFQ.  Checker rule: OK-enqueues are
// legal up to n + k items, FULL is legal when |S| >= n - c_i (reading G12).
#pragma once
#include "lfq.cuh"

namespace gq {

struct DlfqView {
  RingView r;         // the one ring; entries carry the payload (DirFmt)
  uint32_t capacity;  // n
  uint32_t flags;     // GQ_F_*
};

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int enqueue(const DlfqView& q, thread_ctx& ctx, uint32_t v, uint64_t* retries = nullptr) {
  using namespace detail;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  if (!(q.flags & kNoFullTest)) {                                   // GQ_F_NO_FULL_TEST: the caller bounds the fill itself
    const uint64_t H = ld_relaxed(q.r.head);                        // Head first: a later Tail can only overstate the fill,
    const uint64_t T = ld_relaxed(q.r.tail);                        // by dequeues that overlap this operation
    if (T >= H + q.capacity) { ctx.hungry |= 2u; return FULL; }
  }
  ctx.hungry &= ~2u;
  // relaxed install: the entry word is the payload, there is nothing else to publish
  ring_enq_loop<DirFmt, kUniform, kWarpFaa>(q.r, v, retries, q.flags | kRelaxedInstall);
  return OK;
}

template <bool kUniform = false, int kWarpFaa = true>
__device__ __forceinline__ int dequeue(const DlfqView& q, thread_ctx& ctx, uint32_t* out, uint64_t* retries = nullptr) {
  using namespace detail;
  uint64_t dummy = 0; if (!retries) retries = &dummy;
  uint32_t v;
  if (ring_deq_loop<DirFmt, kUniform, kWarpFaa>(q.r, &v, retries, NoFinalize{}, (ctx.hungry & 1u) != 0, q.flags, &ctx.last_ticket) == RING_EMPTY) {
    ctx.hungry |= 1u;
    return EMPTY;
  }
  ctx.hungry &= ~1u;
  *out = v;
  return OK;
}

}  // namespace gq
