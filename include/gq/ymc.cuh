#pragma once
#include "lfq.cuh"
namespace gq {
struct alignas(16) YmcCell { uint64_t val; uint32_t enq, deq; };
struct alignas(128) YmcHandle { uint64_t w[16]; };
struct YmcView { YmcCell* pool; uint64_t pool_cells; uint64_t* tail; uint64_t* head; YmcHandle* handles; uint32_t nthreads, patience, flags; uint64_t* exhausted; };
}
