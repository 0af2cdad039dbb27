// ORACLE — TEST INFRASTRUCTURE ONLY (see fifo_model.hpp header).
//
// Part (b): linearizability checking of recorded histories against the sequential
// bounded-FIFO model.  This plays the role Porcupine plays in the paper:
// PAPER.md L335 "We log concurrent operations with fields proc, op, arg, ret, call, end
// ... feed the log to the standard FIFO model in Porcupine and check linearizability".
//
// Three independent deciders, cross-checked against each other by the CPU tests:
//   brute_check : definition of linearizability (Herlihy & Wing, PAPER.md ref [15])
//                 written out: enumerate every total order consistent with real-time
//                 precedence and replay it on FifoModel.  Tiny histories only.
//   wgl_check   : Wing-Gong search with Lowe's memoisation (the algorithm family
//                 PAPER.md ref [16] / Porcupine uses).  Exact; has a step budget.
//   poly_check  : unique-value FIFO "bad pattern" test (fresh / repeat / order / empty-witness),
//                 polynomial.  Exact for complete histories of the UNBOUNDED FIFO (OK and
//                 EMPTY returns); FULL returns and the capacity bound are outside it
//                 (capacity_check gives the necessary condition), so with those it is a
//                 sound refuter.
//
// Precedence (reading H2): A precedes B iff A.end < B.call strictly.
// ret_status: 0 OK, 1 FULL (enqueue only), 2 EMPTY (dequeue only).
//
// FULL rule (reading G12): with `relaxed_full` an ENQ->FULL is accepted as a
// no-op when |S| >= n - c_i, c_i = number of other operations whose interval overlaps
// operation i (they may each hold one index of the indirection layer).
// Without it FULL is strict (|S| == n).  EMPTY is always strict.
// relaxed_full == 2 (the direct-payload ablation queue G-LFQ-D, which is not in the paper): the
// capacity is soft on both sides: ENQ->OK is legal while |S| < n + c_i (an enqueue that passed its
// "Tail - Head < n" test at t0 installs at t1 after at most c_i other enqueues linearized in
// between, all of which overlap it), ENQ->FULL as above.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace orc {

struct Op {
  uint32_t proc, op, arg, status, val;
  uint64_t call, end;
};

enum Verdict : int { LIN_OK = 1, LIN_VIOLATION = 0, LIN_UNKNOWN = -1, LIN_MALFORMED = -2 };

// Structural pre-checks with a precise message (empty string = fine):
// end >= call; per-proc intervals do not overlap; status legal for op kind;
// OK-enqueued values unique (required by poly_check and by the token protocol, L336).
std::string precheck(const std::vector<Op>& h);

int brute_check(const std::vector<Op>& h, uint64_t capacity, int relaxed_full);
int wgl_check(const std::vector<Op>& h, uint64_t capacity, int relaxed_full,
              uint64_t max_steps, uint64_t* steps_out);
// returns LIN_VIOLATION with a reason, or LIN_OK meaning "no bad pattern found".
int poly_check(const std::vector<Op>& h, std::string* why);

// Necessary condition for the capacity bound (lower bound on |S(t)| over all linearizations).
std::string capacity_check(const std::vector<Op>& h, uint64_t capacity);

// Conservation / token protocol of PAPER.md L336: (i) exactly once, (ii) no value that
// was never enqueued, (iii) per-producer order: values enqueued by one proc are dequeued
// by any single consumer in the producer's program order.  `leftover` = values the
// caller drained afterwards (FIFO order).  Empty string = fine.
std::string conservation_check(const std::vector<Op>& h, const std::vector<uint32_t>& leftover);

}  // namespace orc
