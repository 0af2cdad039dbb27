// ORACLE — TEST INFRASTRUCTURE ONLY (see fifo_model.hpp header).
//
// Part (c): the CPU baseline.  The same bounded FIFO (fifo_model.hpp) made thread-safe
// the plainest way there is — one std::mutex around one std::deque — and driven by host
// threads through the paper's two micro-benchmarks:
//   balanced: "each active thread repeatedly performs one enqueue followed by one dequeue"
//   split   : "threads are assigned producer or consumer roles, and the producer fraction
//              is varied"
// Throughput = (successful enq + successful deq) / t_meas   (eq. 1-2);
// EMPTY/FULL returns are excluded (L392).  A warmup interval precedes the measurement
// interval (L359).  Never tuned: it is a reported baseline, not a target.
#include "fifo_model.hpp"
#include "mutex_queue.hpp"

#include <atomic>
#include <chrono>
#include <cstdint>
#include <mutex>
#include <thread>
#include <vector>

namespace orc {

struct MutexQueue {
  std::mutex mu;
  FifoModel q;
  explicit MutexQueue(uint64_t n) : q(n) {}
  Status enq(uint32_t v) { std::lock_guard<std::mutex> g(mu); return q.enq(v); }
  Status deq(uint32_t* out) { std::lock_guard<std::mutex> g(mu); return q.deq(out); }
};

// role hash: producer iff mix32(seed, tid) < p * 2^32 (DESIGN.md input recipe, BJ config 3)
static inline uint32_t mix32(uint32_t x) {
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}


using clk = std::chrono::steady_clock;

BenchOut mutex_bench(int mode, unsigned threads, uint64_t capacity, uint64_t prefill,
                     double producer_fraction, uint64_t seed, double warmup_ms, double duration_ms) {
  MutexQueue mq(capacity);
  for (uint64_t i = 0; i < prefill; ++i) mq.q.enq((uint32_t)i);
  std::atomic<int> ready{0};
  std::atomic<bool> go{false};
  std::vector<BenchOut> per(threads, BenchOut{});
  clk::time_point t0;
  auto worker = [&](unsigned tid) {
    BenchOut& o = per[tid];
    bool producer = true;
    if (mode == 1) {
      uint32_t h = mix32((uint32_t)seed * 0x9e3779b9u + tid);
      producer = (double)h < producer_fraction * 4294967296.0;
    }
    ready.fetch_add(1);
    while (!go.load(std::memory_order_acquire)) {}
    const auto tw = t0 + std::chrono::duration_cast<clk::duration>(std::chrono::duration<double, std::milli>(warmup_ms));
    const auto te = tw + std::chrono::duration_cast<clk::duration>(std::chrono::duration<double, std::milli>(duration_ms));
    uint64_t iter = 0;
    for (;;) {
      uint32_t v = (uint32_t)(prefill + tid + iter * threads), got = 0;
      ++iter;
      Status se = ST_FULL, sd = ST_EMPTY;
      bool did_e = false, did_d = false;
      if (mode == 0 || producer) { se = mq.enq(v); did_e = true; }
      if (mode == 0 || !producer) { sd = mq.deq(&got); did_d = true; }
      auto now = clk::now();
      bool in = now >= tw && now < te;
      if (did_e) { if (se == ST_OK) { o.tot_enq++; o.sum_enq += v; if (in) o.succ_enq++; } else if (in) o.full++; }
      if (did_d) { if (sd == ST_OK) { o.tot_deq++; o.sum_deq += got; if (in) o.succ_deq++; } else if (in) o.empty++; }
      if (now >= te) break;
    }
  };
  std::vector<std::thread> ts;
  for (unsigned t = 0; t < threads; ++t) ts.emplace_back(worker, t);
  while (ready.load() < (int)threads) {}
  t0 = clk::now();
  go.store(true, std::memory_order_release);
  for (auto& t : ts) t.join();
  BenchOut r{};
  for (auto& o : per) {
    r.succ_enq += o.succ_enq; r.succ_deq += o.succ_deq; r.full += o.full; r.empty += o.empty;
    r.tot_enq += o.tot_enq; r.tot_deq += o.tot_deq; r.sum_enq += o.sum_enq; r.sum_deq += o.sum_deq;
  }
  for (uint64_t i = 0; i < prefill; ++i) r.sum_enq += (uint32_t)i;
  r.tot_enq += prefill;
  uint32_t v;
  while (mq.q.deq(&v) == ST_OK) { r.left++; r.sum_left += v; }
  r.meas_seconds = duration_ms * 1e-3;
  return r;
}

}  // namespace orc
