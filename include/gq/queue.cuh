// gq/queue.cuh — the __device__ API a user kernel includes.
//
//   gq::thread_ctx ctx{tid};                       // tid unique per thread, < max_threads
//   int s = gq::enqueue(view, ctx, v);             // gq::OK | gq::FULL
//   int s = gq::dequeue(view, ctx, &v);            // gq::OK | gq::EMPTY
//
// `view` is the POD LfqView / WfqView / YmcView (or DlfqView, the direct-payload ablation) obtained on the host with
// queue_device_view() (gq.h) and passed to the kernel by value.  Any subset of lanes may
// call, converged or diverged.  Template flag kUniform = true promises that all lanes
// converged at the call use the same queue (skips the address match in warp_faa).
// Memory ordering (reading G15).  The payload itself always arrives intact.  Memory OTHER than the payload
// that a producer wrote before enqueue(v) is visible to the consumer after it dequeued v if the producer issued
// __threadfence() between those stores and the enqueue (the dequeue's entry load is an acquire), or, without any
// fence in user code, if the queue was created with GQ_F_FENCED_PAYLOAD (installing CAS = release, the paper's
// implicit scheme).  The default build installs with relaxed atomics (departure D6) and does not order the
// caller's other stores by itself.  tests/user_kernel/litmus.cu exercises both contracts from a user kernel.
// A G-WFQ / YMC thread must not exit while one of its own requests is published; the
// wait-freedom claim needs all participating threads resident.
#pragma once
#include "lfq.cuh"
#include "wfq.cuh"
#include "ymc.cuh"
#include "dlfq.cuh"

namespace gq {
// Block-level ticket funnels (D11): a kernel whose blocks hammer the same queue can combine the ticket
// requests of its warps per block.  In the kernel:
//     __shared__ gq::BlockFunnel funnels[gq::kFunnelsPerQueue];
//     gq::funnel_init(funnels, gq::kFunnelsPerQueue, /*window_ns=*/0);     // whole block, ends with __syncthreads()
//     auto q = gq::with_funnels(view, funnels);                             // this thread's copy of the view
// and then gq::enqueue<kUniform, 2>(q, ...) / gq::dequeue<kUniform, 2>(q, ...): the second template argument selects how tickets
// are drawn (0 = one FAA per thread, 1 = WAVEFAA, the default, 2 = WAVEFAA through the funnels).  One set of funnels per (block, queue).
// Measured on B200 (D11): +26 % for G-WFQ-YMC (two hot counters, bound by their atomic rate), a loss for the ring
// queues (four dependent tickets per enqueue + dequeue pair: the handshake lengthens every one of them).
using detail::BlockFunnel;
using detail::funnel_init;
constexpr uint32_t kFunnelsPerQueue = 4;
__device__ __forceinline__ LfqView with_funnels(LfqView q, BlockFunnel* f) {
  q.aq.fhead = f; q.aq.ftail = f + 1; q.fq.fhead = f + 2; q.fq.ftail = f + 3; return q;
}
__device__ __forceinline__ WfqView with_funnels(WfqView q, BlockFunnel* f) {
  q.aq.fhead = f; q.aq.ftail = f + 1; q.fq.fhead = f + 2; q.fq.ftail = f + 3; return q;
}
__device__ __forceinline__ DlfqView with_funnels(DlfqView q, BlockFunnel* f) { q.r.fhead = f; q.r.ftail = f + 1; return q; }
__device__ __forceinline__ YmcView with_funnels(YmcView q, BlockFunnel* f) { q.fhead = f; q.ftail = f + 1; return q; }
}  // namespace gq
