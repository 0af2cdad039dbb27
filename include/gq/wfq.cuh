#pragma once
#include "lfq.cuh"
namespace gq {
struct alignas(128) WfqRecord { uint64_t w[16]; };
struct WfqView { RingView aq, fq; uint32_t* data; WfqRecord* rec; uint32_t capacity, nthreads, enq_patience, deq_patience, help_delay, flags; };
}
