// ORACLE — TEST INFRASTRUCTURE ONLY. Not part of the product path.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may use anything under oracle/. It shares no code with the CUDA path.
//
// Part (a): the sequential bounded-FIFO specification.
//
// PAPER.md L345 (footnote 2, §IV): "the model enqueues append to the state list and
// dequeues must return the head or report empty".  "Bounded" (PAPER.md L17, L88-89:
// "logical capacity n") adds: an enqueue on a queue holding n items reports FULL and
// leaves the state unchanged.
//
// This is the plain definition every queue in the paper implements; the linearizability
// checker (lincheck.cpp) searches for an order of the recorded operations that this
// model accepts.
#pragma once
#include <cstdint>
#include <deque>

namespace orc {

enum Status : uint32_t { ST_OK = 0, ST_FULL = 1, ST_EMPTY = 2 };
enum OpKind : uint32_t { OP_ENQ = 0, OP_DEQ = 1 };   // op=0 ENQ, op=1 DEQ

struct FifoModel {
  std::deque<uint32_t> s;   // front = head of the queue
  uint64_t capacity;        // n; UINT64_MAX = unbounded

  explicit FifoModel(uint64_t n) : capacity(n) {}

  // ENQ(v): |S| < n -> append, OK ; else FULL, no change.
  Status enq(uint32_t v) {
    if (s.size() >= capacity) return ST_FULL;
    s.push_back(v);
    return ST_OK;
  }
  // DEQ(): S non-empty -> pop front, OK ; else EMPTY.
  Status deq(uint32_t* out) {
    if (s.empty()) return ST_EMPTY;
    *out = s.front();
    s.pop_front();
    return ST_OK;
  }
};

}  // namespace orc
