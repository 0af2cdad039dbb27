// ORACLE — TEST INFRASTRUCTURE ONLY (see fifo_model.hpp header).
// Small C ABI over the oracle so that tests/ can call it through ctypes.  Histories come
// in as separate arrays (no struct shared with the CUDA library).
#include "fifo_model.hpp"
#include "lincheck.hpp"
#include "mutex_queue.hpp"

#include <cstdio>
#include <cstring>
#include <thread>


using namespace orc;

static std::vector<Op> gather(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg,
                              const uint32_t* status, const uint32_t* val, const uint64_t* call, const uint64_t* end) {
  std::vector<Op> h(m);
  for (uint64_t i = 0; i < m; ++i) h[i] = Op{proc[i], op[i], arg[i], status[i], val[i], call[i], end[i]};
  return h;
}
static void put_msg(char* buf, uint64_t cap, const std::string& s) {
  if (!buf || cap == 0) return;
  std::snprintf(buf, cap, "%s", s.c_str());
}

extern "C" {

// Replay a sequential script on the model (fifo_model.hpp): op[i] in {0 ENQ, 1 DEQ}.
void orc_fifo_replay(uint64_t capacity, uint64_t m, const uint32_t* op, const uint32_t* arg,
                     uint32_t* status_out, uint32_t* val_out) {
  FifoModel q(capacity);
  for (uint64_t i = 0; i < m; ++i) {
    uint32_t v = 0;
    status_out[i] = op[i] == OP_ENQ ? q.enq(arg[i]) : q.deq(&v);
    val_out[i] = v;
  }
}

int orc_precheck(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg, const uint32_t* status,
                 const uint32_t* val, const uint64_t* call, const uint64_t* end, char* msg, uint64_t msg_cap) {
  std::string s = precheck(gather(m, proc, op, arg, status, val, call, end));
  put_msg(msg, msg_cap, s);
  return s.empty() ? 1 : 0;
}

int orc_brute(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg, const uint32_t* status,
              const uint32_t* val, const uint64_t* call, const uint64_t* end, uint64_t capacity, int relaxed_full) {
  return brute_check(gather(m, proc, op, arg, status, val, call, end), capacity, relaxed_full);
}

int orc_wgl(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg, const uint32_t* status,
            const uint32_t* val, const uint64_t* call, const uint64_t* end, uint64_t capacity, int relaxed_full,
            uint64_t max_steps, uint64_t* steps_out) {
  return wgl_check(gather(m, proc, op, arg, status, val, call, end), capacity, relaxed_full, max_steps, steps_out);
}

int orc_poly(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg, const uint32_t* status,
             const uint32_t* val, const uint64_t* call, const uint64_t* end, char* msg, uint64_t msg_cap) {
  std::string why;
  int r = poly_check(gather(m, proc, op, arg, status, val, call, end), &why);
  put_msg(msg, msg_cap, why);
  return r;
}

int orc_conservation(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg, const uint32_t* status,
                     const uint32_t* val, const uint64_t* call, const uint64_t* end, const uint32_t* leftover,
                     uint64_t n_left, char* msg, uint64_t msg_cap) {
  std::vector<uint32_t> left(leftover, leftover + n_left);
  std::string s = conservation_check(gather(m, proc, op, arg, status, val, call, end), left);
  put_msg(msg, msg_cap, s);
  return s.empty() ? 1 : 0;
}

int orc_capacity(uint64_t m, const uint32_t* proc, const uint32_t* op, const uint32_t* arg, const uint32_t* status,
                 const uint32_t* val, const uint64_t* call, const uint64_t* end, uint64_t capacity, char* msg, uint64_t msg_cap) {
  std::string s = capacity_check(gather(m, proc, op, arg, status, val, call, end), capacity);
  put_msg(msg, msg_cap, s);
  return s.empty() ? 1 : 0;
}

// out[0..9] = succ_enq, succ_deq, full, empty, tot_enq, tot_deq, sum_enq, sum_deq, sum_left, left
void orc_mutex_bench(int mode, uint32_t threads, uint64_t capacity, uint64_t prefill, double producer_fraction,
                     uint64_t seed, double warmup_ms, double duration_ms, uint64_t* out, double* meas_seconds) {
  BenchOut r = mutex_bench(mode, threads, capacity, prefill, producer_fraction, seed, warmup_ms, duration_ms);
  out[0] = r.succ_enq; out[1] = r.succ_deq; out[2] = r.full; out[3] = r.empty; out[4] = r.tot_enq;
  out[5] = r.tot_deq; out[6] = r.sum_enq; out[7] = r.sum_deq; out[8] = r.sum_left; out[9] = r.left;
  *meas_seconds = r.meas_seconds;
}

uint32_t orc_hw_threads() { return std::thread::hardware_concurrency(); }

}  // extern "C"
