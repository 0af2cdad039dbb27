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
// A G-WFQ / YMC thread must not exit while one of its own requests is published; the
// wait-freedom claim needs all participating threads resident.
#pragma once
#include "lfq.cuh"
#include "wfq.cuh"
#include "ymc.cuh"
#include "dlfq.cuh"
