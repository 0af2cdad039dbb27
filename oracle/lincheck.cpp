// ORACLE — TEST INFRASTRUCTURE ONLY (see fifo_model.hpp / lincheck.hpp headers).
#include "lincheck.hpp"
#include "fifo_model.hpp"

#include <algorithm>
#include <cstring>
#include <map>
#include <unordered_map>
#include <unordered_set>

namespace orc {

// ---------------------------------------------------------------- helpers
static inline bool precedes(const Op& a, const Op& b) { return a.end < b.call; }  // reading H2

// c_i of the relaxed FULL rule: how many OTHER ops overlap op i (not ordered either way).
static std::vector<uint64_t> overlap_counts(const std::vector<Op>& h) {
  std::vector<uint64_t> c(h.size(), 0);
  for (size_t i = 0; i < h.size(); ++i)
    for (size_t j = 0; j < h.size(); ++j)
      if (i != j && !precedes(h[i], h[j]) && !precedes(h[j], h[i])) ++c[i];
  return c;
}

// One step of the model for a recorded op: is the recorded return value what the
// sequential spec (fifo_model.hpp) would return in state m?  Applies the op if so.
static bool model_step(FifoModel& m, const Op& o, int relaxed_full, uint64_t ci) {
  if (o.op == OP_ENQ) {
    if (o.status == ST_OK) {
      if (relaxed_full == 2) {                       // soft capacity (G-LFQ-D): |S| < n + c_i
        if (m.s.size() >= m.capacity + ci) return false;
        m.s.push_back(o.arg);
        return true;
      }
      return m.enq(o.arg) == ST_OK;
    }
    if (o.status == ST_FULL) {
      if (!relaxed_full) return m.s.size() >= m.capacity;
      uint64_t need = m.capacity > ci ? m.capacity - ci : 0;
      return m.s.size() >= need;
    }
    return false;
  }
  if (o.status == ST_OK) {
    if (m.s.empty() || m.s.front() != o.val) return false;
    m.s.pop_front();
    return true;
  }
  if (o.status == ST_EMPTY) return m.s.empty();
  return false;
}
static void model_undo(FifoModel& m, const Op& o) {
  if (o.op == OP_ENQ) { if (o.status == ST_OK) m.s.pop_back(); }
  else if (o.status == ST_OK) m.s.push_front(o.val);
}

// ---------------------------------------------------------------- precheck
std::string precheck(const std::vector<Op>& h) {
  std::unordered_set<uint32_t> enq_vals;
  std::map<uint32_t, std::vector<const Op*>> by_proc;
  for (size_t i = 0; i < h.size(); ++i) {
    const Op& o = h[i];
    if (o.end < o.call) return "op " + std::to_string(i) + ": end < call";
    if (o.op == OP_ENQ) {
      if (o.status != ST_OK && o.status != ST_FULL) return "op " + std::to_string(i) + ": bad enqueue status";
      if (o.status == ST_OK && !enq_vals.insert(o.arg).second)
        return "value " + std::to_string(o.arg) + " enqueued OK twice (values must be unique)";
    } else if (o.op == OP_DEQ) {
      if (o.status != ST_OK && o.status != ST_EMPTY) return "op " + std::to_string(i) + ": bad dequeue status";
    } else return "op " + std::to_string(i) + ": bad op kind";
    by_proc[o.proc].push_back(&o);
  }
  for (auto& kv : by_proc) {
    auto& v = kv.second;
    std::sort(v.begin(), v.end(), [](const Op* a, const Op* b) { return a->call < b->call; });
    for (size_t i = 1; i < v.size(); ++i)
      if (v[i]->call < v[i - 1]->end)
        return "proc " + std::to_string(kv.first) + ": overlapping operations of one process";
  }
  return "";
}

// ---------------------------------------------------------------- brute force
// Definition of linearizability written out: DFS over all total orders that extend the
// real-time partial order, replaying each prefix on the model.
static bool brute_rec(const std::vector<Op>& h, const std::vector<uint64_t>& ci, std::vector<char>& done,
                      size_t ndone, FifoModel& m, int relaxed) {
  if (ndone == h.size()) return true;
  for (size_t i = 0; i < h.size(); ++i) {
    if (done[i]) continue;
    bool minimal = true;   // every op that precedes i must already be linearized
    for (size_t j = 0; j < h.size() && minimal; ++j)
      if (!done[j] && j != i && precedes(h[j], h[i])) minimal = false;
    if (!minimal) continue;
    if (!model_step(m, h[i], relaxed, ci[i])) continue;
    done[i] = 1;
    if (brute_rec(h, ci, done, ndone + 1, m, relaxed)) return true;
    done[i] = 0;
    model_undo(m, h[i]);
  }
  return false;
}

int brute_check(const std::vector<Op>& h, uint64_t capacity, int relaxed_full) {
  if (h.size() > 12) return LIN_UNKNOWN;
  std::vector<char> done(h.size(), 0);
  FifoModel m(capacity);
  auto ci = overlap_counts(h);
  return brute_rec(h, ci, done, 0, m, relaxed_full) ? LIN_OK : LIN_VIOLATION;
}

// ---------------------------------------------------------------- WGL + memoisation
namespace {
struct Ev {
  bool is_call;
  uint32_t id;       // op index
  uint64_t t;
  Ev *prev, *next, *match;   // match: call -> its return event
};
}  // namespace

int wgl_check(const std::vector<Op>& h, uint64_t capacity, int relaxed_full,
              uint64_t max_steps, uint64_t* steps_out) {
  const size_t m = h.size();
  if (steps_out) *steps_out = 0;
  if (m == 0) return LIN_OK;
  std::vector<uint64_t> ci = relaxed_full ? overlap_counts(h) : std::vector<uint64_t>(m, 0);

  // 2 events per op, sorted by time; at equal time calls come before returns so that
  // "A.end == B.call" leaves A and B concurrent (reading H2).
  std::vector<Ev> evs(2 * m);
  for (size_t i = 0; i < m; ++i) {
    evs[2 * i] = Ev{true, (uint32_t)i, h[i].call, nullptr, nullptr, nullptr};
    evs[2 * i + 1] = Ev{false, (uint32_t)i, h[i].end, nullptr, nullptr, nullptr};
  }
  std::vector<Ev*> order(2 * m);
  for (size_t i = 0; i < 2 * m; ++i) order[i] = &evs[i];
  std::stable_sort(order.begin(), order.end(), [](const Ev* a, const Ev* b) {
    if (a->t != b->t) return a->t < b->t;
    return a->is_call && !b->is_call;
  });
  Ev head{false, 0, 0, nullptr, nullptr, nullptr};
  Ev* p = &head;
  for (Ev* e : order) { p->next = e; e->prev = p; p = e; }
  p->next = nullptr;
  for (size_t i = 0; i < m; ++i) evs[2 * i].match = &evs[2 * i + 1];

  auto lift = [](Ev* c) {          // unlink call and its return
    c->prev->next = c->next; if (c->next) c->next->prev = c->prev;
    Ev* r = c->match;
    r->prev->next = r->next; if (r->next) r->next->prev = r->prev;
  };
  auto unlift = [](Ev* c) {        // exact reverse
    Ev* r = c->match;
    r->prev->next = r; if (r->next) r->next->prev = r;
    c->prev->next = c; if (c->next) c->next->prev = c;
  };

  FifoModel model(capacity);
  const size_t words = (m + 63) / 64;
  std::vector<uint64_t> lin(words, 0);
  std::unordered_set<std::string> cache;   // exact key: linearized bitset + queue contents
  std::string key;
  uint64_t steps = 0;

  // Search order only (never the verdict): among the minimal operations — the call events
  // that come before the first return event still in the list, exactly the set plain WGL
  // would try one after another — try first a dequeue whose value is at the front, then
  // EMPTY/FULL, then enqueues in the order in which their values are dequeued.  A FIFO
  // dequeues in enqueue order, so on a correct history this guess is almost always right
  // and the DFS hardly backtracks; on a wrong guess the search still visits every
  // alternative, so the result is the same as with time order.
  std::vector<uint64_t> deq_call(m, UINT64_MAX);
  {
    std::unordered_map<uint32_t, uint64_t> dc;
    for (const Op& o : h) if (o.op == OP_DEQ && o.status == ST_OK) {
      auto it = dc.find(o.val);
      if (it == dc.end() || o.call < it->second) dc[o.val] = o.call;
    }
    for (size_t i = 0; i < m; ++i) if (h[i].op == OP_ENQ && h[i].status == ST_OK) {
      auto it = dc.find(h[i].arg);
      if (it != dc.end()) deq_call[i] = it->second;
    }
  }
  struct Frame { std::vector<Ev*> cands; size_t next; Ev* taken; };
  std::vector<Frame> stack;
  auto make_frame = [&]() {
    Frame f; f.next = 0; f.taken = nullptr;
    for (Ev* e = head.next; e && e->is_call; e = e->next) f.cands.push_back(e);
    auto prio = [&](const Ev* e) -> std::pair<int, uint64_t> {
      const Op& o = h[e->id];
      if (o.op == OP_DEQ && o.status == ST_OK) return {0, o.call};
      if (o.status != ST_OK) return {1, o.call};
      return {2, deq_call[e->id]};
    };
    std::stable_sort(f.cands.begin(), f.cands.end(), [&](const Ev* a, const Ev* b) { return prio(a) < prio(b); });
    return f;
  };
  stack.push_back(make_frame());
  while (head.next != nullptr) {
    Frame& f = stack.back();
    bool descended = false;
    while (f.next < f.cands.size()) {
      if (++steps > max_steps) { if (steps_out) *steps_out = steps; return LIN_UNKNOWN; }
      Ev* e = f.cands[f.next++];
      const Op& o = h[e->id];
      if (!model_step(model, o, relaxed_full, ci[e->id])) continue;
      lin[e->id >> 6] |= 1ull << (e->id & 63);
      key.assign((const char*)lin.data(), words * 8);
      for (uint32_t v : model.s) key.append((const char*)&v, 4);
      if (cache.insert(key).second) {
        f.taken = e;
        lift(e);
        stack.push_back(make_frame());
        descended = true;
        break;
      }
      lin[e->id >> 6] &= ~(1ull << (e->id & 63));
      model_undo(model, o);
    }
    if (descended) continue;
    // every minimal op tried: the first return event cannot be passed -> backtrack
    stack.pop_back();
    if (stack.empty()) { if (steps_out) *steps_out = steps; return LIN_VIOLATION; }
    Ev* c = stack.back().taken;
    lin[c->id >> 6] &= ~(1ull << (c->id & 63));
    model_undo(model, h[c->id]);
    unlift(c);
  }
  if (steps_out) *steps_out = steps;
  return LIN_OK;
}

// ---------------------------------------------------------------- polynomial check
// Unique-value FIFO bad patterns (complete histories):
//   fresh : a dequeue returns a value never enqueued, or returns before that enqueue began
//   repeat: a value dequeued twice
//   order : enq(a) precedes enq(b) and ( deq(b) precedes deq(a)  or  b dequeued, a never )
//   empty : DEQ->EMPTY d, and some value v has enq(v) finished before d began while
//           deq(v) began after d ended or never happened  (necessary condition only)
int poly_check(const std::vector<Op>& h, std::string* why) {
  auto fail = [&](const std::string& s) { if (why) *why = s; return (int)LIN_VIOLATION; };
  std::unordered_map<uint32_t, const Op*> enq, deq;
  for (const Op& o : h) {
    if (o.op == OP_ENQ && o.status == ST_OK) enq[o.arg] = &o;
  }
  for (const Op& o : h) {
    if (o.op == OP_DEQ && o.status == ST_OK) {
      auto it = enq.find(o.val);
      if (it == enq.end()) return fail("fresh: dequeued value " + std::to_string(o.val) + " never enqueued");
      if (precedes(o, *it->second)) return fail("fresh: value " + std::to_string(o.val) + " dequeued before its enqueue began");
      if (!deq.emplace(o.val, &o).second) return fail("repeat: value " + std::to_string(o.val) + " dequeued twice");
    }
  }
  std::vector<std::pair<const Op*, const Op*>> vals;   // (enq, deq or null)
  vals.reserve(enq.size());
  for (auto& kv : enq) {
    auto it = deq.find(kv.first);
    vals.emplace_back(kv.second, it == deq.end() ? nullptr : it->second);
  }
  for (auto& a : vals)
    for (auto& b : vals) {
      if (a.first == b.first || !precedes(*a.first, *b.first)) continue;
      if (b.second && !a.second)
        return fail("order: " + std::to_string(b.first->arg) + " dequeued but earlier-enqueued " + std::to_string(a.first->arg) + " never");
      if (a.second && b.second && precedes(*b.second, *a.second))
        return fail("order: " + std::to_string(b.first->arg) + " dequeued before earlier-enqueued " + std::to_string(a.first->arg));
    }
  // empty: DEQ->EMPTY d is impossible iff its whole interval is covered by values that are
  // certainly in the queue: a chain x1..xk with enq(x1) finished before d began, enq(x_{i+1})
  // finished before deq(x_i) began (x_{i+1} is in before x_i can leave), and deq(x_k) begun
  // after d ended (or never).  Reachability over "enq(y) precedes deq(x)" edges.
  const size_t nv = vals.size();
  std::vector<std::vector<uint32_t>> succ(nv);
  bool any_empty = false;
  for (const Op& d : h) if (d.op == OP_DEQ && d.status == ST_EMPTY) any_empty = true;
  if (any_empty) {
    for (size_t x = 0; x < nv; ++x)
      for (size_t y = 0; y < nv; ++y)
        if (x != y && (!vals[x].second || precedes(*vals[y].first, *vals[x].second))) succ[x].push_back((uint32_t)y);
    for (const Op& d : h) {
      if (d.op != OP_DEQ || d.status != ST_EMPTY) continue;
      std::vector<char> seen(nv, 0);
      std::vector<uint32_t> stack;
      for (size_t x = 0; x < nv; ++x)
        if (precedes(*vals[x].first, d)) { seen[x] = 1; stack.push_back((uint32_t)x); }
      while (!stack.empty()) {
        const uint32_t x = stack.back(); stack.pop_back();
        if (!vals[x].second || precedes(d, *vals[x].second))
          return fail("empty: EMPTY returned although the queue held a value throughout the dequeue (chain ends at " +
                      std::to_string(vals[x].first->arg) + ")");
        // x leaves during or before d: only values certainly in before x can leave AND still
        // relevant (their enqueue precedes x's dequeue) extend the cover
        for (uint32_t y : succ[x]) if (!seen[y]) { seen[y] = 1; stack.push_back(y); }
      }
    }
  }
  if (why) why->clear();
  return LIN_OK;
}

// ---------------------------------------------------------------- capacity bound
// Necessary condition for the bound |S| <= n: in every linearization, at time t every OK enqueue
// that finished before t is in and no OK dequeue invoked after t is, so
// |S(t)| >= #enqOK(end < t) - #deqOK(call <= t).  That lower bound must never exceed n.
std::string capacity_check(const std::vector<Op>& h, uint64_t capacity) {
  std::vector<std::pair<uint64_t, int>> ev;   // (time, +1 enq finished [counts for t > end] / -1 deq invoked)
  for (const Op& o : h) {
    if (o.status != ST_OK) continue;
    if (o.op == OP_ENQ) ev.emplace_back(o.end + 1, +1);   // strictly after its end
    else ev.emplace_back(o.call, -1);
  }
  std::sort(ev.begin(), ev.end(), [](const std::pair<uint64_t, int>& a, const std::pair<uint64_t, int>& b) {
    return a.first != b.first ? a.first < b.first : a.second < b.second;   // dequeues first at equal time
  });
  int64_t lb = 0;
  for (auto& e : ev) {
    lb += e.second;
    if (lb > (int64_t)capacity)
      return "capacity: at t=" + std::to_string(e.first) + " at least " + std::to_string(lb) + " items must be in a queue of " + std::to_string(capacity);
  }
  return "";
}

// ---------------------------------------------------------------- conservation
std::string conservation_check(const std::vector<Op>& h, const std::vector<uint32_t>& leftover) {
  std::unordered_map<uint32_t, int> count;       // value -> times seen leaving the queue
  std::unordered_map<uint32_t, std::pair<uint32_t, uint64_t>> origin;   // value -> (producer, enq call)
  for (const Op& o : h)
    if (o.op == OP_ENQ && o.status == ST_OK) { origin[o.arg] = {o.proc, o.call}; count[o.arg] = 0; }
  for (const Op& o : h)
    if (o.op == OP_DEQ && o.status == ST_OK) {
      auto it = count.find(o.val);
      if (it == count.end()) return "value " + std::to_string(o.val) + " dequeued but never enqueued";
      if (++it->second > 1) return "value " + std::to_string(o.val) + " dequeued more than once";
    }
  for (uint32_t v : leftover) {
    auto it = count.find(v);
    if (it == count.end()) return "drained value " + std::to_string(v) + " never enqueued";
    if (++it->second > 1) return "value " + std::to_string(v) + " left the queue more than once";
  }
  for (auto& kv : count)
    if (kv.second != 1) return "value " + std::to_string(kv.first) + " enqueued but never dequeued or drained";
  // (iii) per consumer, per producer: dequeued in the producer's program order.
  std::map<uint32_t, std::vector<const Op*>> by_consumer;
  for (const Op& o : h) if (o.op == OP_DEQ && o.status == ST_OK) by_consumer[o.proc].push_back(&o);
  for (auto& kv : by_consumer) {
    auto& v = kv.second;
    std::sort(v.begin(), v.end(), [](const Op* a, const Op* b) { return a->call < b->call; });
    std::unordered_map<uint32_t, uint64_t> last;   // producer -> enq call time of last value seen
    for (const Op* d : v) {
      auto org = origin[d->val];
      auto it = last.find(org.first);
      if (it != last.end() && org.second < it->second)
        return "consumer " + std::to_string(kv.first) + " saw producer " + std::to_string(org.first) + "'s values out of order";
      last[org.first] = org.second;
    }
  }
  return "";
}

}  // namespace orc
