// ORACLE — TEST INFRASTRUCTURE ONLY (see fifo_model.hpp header).  Declarations for mutex_queue.cpp.
#pragma once
#include <cstdint>
namespace orc {
struct BenchOut {
  uint64_t succ_enq, succ_deq, full, empty;        // inside the measurement window
  uint64_t tot_enq, tot_deq;                       // whole run incl. prefill (for conservation)
  uint64_t sum_enq, sum_deq, sum_left, left;       // checksums mod 2^64, items left at the end
  double meas_seconds;
};
// mode 0 = balanced, 1 = split.  prefill: values 0..prefill-1 enqueued in order first.
BenchOut mutex_bench(int mode, unsigned threads, uint64_t capacity, uint64_t prefill,
                     double producer_fraction, uint64_t seed, double warmup_ms, double duration_ms);
}  // namespace orc
