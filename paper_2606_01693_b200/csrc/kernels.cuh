// Harness kernels: the paper's balanced / split micro-benchmarks as one
// persistent, fully co-resident kernel (Thm III.10 residency assumption, L327-331), the
// device-side history recorder (L335), and the small service kernels behind the C ABI.
#pragma once
#include <cooperative_groups.h>
#include <cstdint>

#include "gq.h"
#include "gq/queue.cuh"

namespace gqk {
namespace cg = cooperative_groups;
using namespace gq;
using namespace gq::detail;

enum { MODE_BALANCED = 0, MODE_SPLIT = 1 };
// counter slots in the device result block
enum { C_SUCC_ENQ, C_SUCC_DEQ, C_FULL, C_EMPTY, C_TOT_ENQ, C_TOT_DEQ, C_TOT_FULL, C_TOT_EMPTY,
       C_SUM_ENQ, C_SUM_DEQ, C_RETRIES, C_T0, C_T_END, C_POOL, C_COUNT = 16 };

struct BenchParams {
  uint32_t threads, mode;
  uint64_t warmup_ns, duration_ns;
  uint64_t prod_threshold;     // producer iff mix32(..) < prod_threshold  (p * 2^32)
  uint32_t seed, ops_per_thread;
  uint32_t jitter_ns, fail_backoff_ns;
  uint64_t value_base;
  const uint32_t* perm;        // physical -> logical thread id (role_layout 1), or nullptr
  uint32_t tid_shift;          // > 0: payload = value_base + (thread << tid_shift | iter) (BASELINE.json configs[0]); 0: value_base + thread + iter * threads
  uint32_t _pad;
  uint32_t fused, converged;   // role_layout 2: mixed warps call the fused enqueue_or_dequeue (G-LFQ); converged: see gq_run_cfg
  uint32_t block_faa, funnel_window_ns;   // block-level ticket funnels (gq_run_cfg)
};

// the fused mixed-warp operation exists for G-LFQ (lfq.cuh); other kinds run the two calls
template <class Q> struct HasFused { static constexpr bool value = false; };
template <> struct HasFused<LfqView> { static constexpr bool value = true; };
template <int kWarpFaa, class Q>
__device__ __forceinline__ int fused_op(const Q&, thread_ctx&, bool, uint32_t*, uint64_t*) { return -1; }
template <int kWarpFaa>
__device__ __forceinline__ int fused_op(const LfqView& q, thread_ctx& ctx, bool is_enq, uint32_t* v, uint64_t* retries) {
  return enqueue_or_dequeue<kWarpFaa>(q, ctx, is_enq, v, retries);
}
template <int kWarpFaa, class Q>
__device__ __forceinline__ int fused_step(const Q&, thread_ctx&, op_state&, bool, uint32_t*, uint64_t*) { return -1; }
template <int kWarpFaa>
__device__ __forceinline__ int fused_step(const LfqView& q, thread_ctx& ctx, op_state& st, bool is_enq, uint32_t* v, uint64_t* retries) {
  return enqueue_or_dequeue_step<kWarpFaa>(q, ctx, st, is_enq, v, retries);
}

__device__ __forceinline__ uint64_t warp_sum(uint64_t v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// the unique payload of (logical thread, iteration)
__device__ __forceinline__ uint32_t payload_of(const BenchParams& p, uint32_t ltid, uint32_t iter) {
  return p.tid_shift ? (uint32_t)(p.value_base + ((uint64_t)ltid << p.tid_shift | iter))
                     : (uint32_t)(p.value_base + ltid + (uint64_t)iter * p.threads);
}

// per-thread tallies of the benchmark loop
struct Tally {
  uint32_t succ_enq = 0, succ_deq = 0, full = 0, empty = 0, tot_enq = 0, tot_deq = 0, tot_full = 0, tot_empty = 0, fail_ns = 0;
  uint64_t sum_enq = 0, sum_deq = 0, retries = 0;
};
__device__ __forceinline__ void fail_backoff(const BenchParams& p, Tally& a) {
  if (p.fail_backoff_ns) { a.fail_ns = a.fail_ns ? min(a.fail_ns * 2, p.fail_backoff_ns) : 64; __nanosleep(a.fail_ns); }
}
// one enqueue / one dequeue of the benchmark loop, with its history record (kHist) and its tallies; returns the end stamp
template <class Q, bool kHist, int kWarpFaa>
__device__ __forceinline__ uint64_t enq_step(const Q& q, thread_ctx& ctx, const BenchParams& p, uint32_t ltid, uint32_t iter,
                                             uint64_t tw, uint64_t te, Tally& a, gq_hist_rec*& my) {
  const uint32_t v = payload_of(p, ltid, iter);
  uint64_t t_call = 0;
  if (kHist) {
    if (p.jitter_ns) __nanosleep(mix32(p.seed ^ (ltid * 0x85ebca6bu) ^ (iter * 2u + 0x1234567u)) % (p.jitter_ns + 1));
    t_call = globaltimer_ns();
  }
  const int s = enqueue<true, kWarpFaa>(q, ctx, v, &a.retries);
  if (kHist) { __threadfence(); }               // effects performed before `end` is read (reading H1)
  const uint64_t now = globaltimer_ns();
  if (kHist) *my++ = gq_hist_rec{ltid, GQ_OP_ENQ, v, (uint32_t)s, 0u, 0u, t_call, now};
  const bool in = now >= tw && now < te;
  if (s == OK) { ++a.tot_enq; a.sum_enq += v; a.succ_enq += in; a.fail_ns = 0; }
  else { ++a.tot_full; a.full += in; fail_backoff(p, a); }
  return now;
}
template <class Q, bool kHist, int kWarpFaa>
__device__ __forceinline__ uint64_t deq_step(const Q& q, thread_ctx& ctx, const BenchParams& p, uint32_t ltid, uint32_t iter,
                                             uint64_t tw, uint64_t te, Tally& a, gq_hist_rec*& my) {
  uint32_t v = 0;
  uint64_t t_call = 0;
  if (kHist) {
    if (p.jitter_ns) __nanosleep(mix32(p.seed ^ (ltid * 0xc2b2ae35u) ^ (iter * 2u + 0x7654321u)) % (p.jitter_ns + 1));
    t_call = globaltimer_ns();
  }
  const int s = dequeue<true, kWarpFaa>(q, ctx, &v, &a.retries);
  if (kHist) { __threadfence(); }
  const uint64_t now = globaltimer_ns();
  if (kHist) *my++ = gq_hist_rec{ltid, GQ_OP_DEQ, 0u, (uint32_t)s, s == OK ? v : 0u, 0u, t_call, now};
  const bool in = now >= tw && now < te;
  if (s == OK) { ++a.tot_deq; a.sum_deq += v; a.succ_deq += in; a.fail_ns = 0; }
  else { ++a.tot_empty; a.empty += in; fail_backoff(p, a); }
  return now;
}

// End of one benchmark iteration.  cfg.converged: the lanes of a warp that run this loop start their next iteration
// together (one ballot over the lanes still looping), which is how a lock-step wavefront runs the paper's kernels
// (wave64) and what kUniform callers promise anyway; without it a warp that has split once (lanes leave a wait
// loop at different polls) stays split for the rest of the launch and all its later WAVEFAA batches are partial.
__device__ __forceinline__ bool loop_done(const BenchParams& p, uint32_t& act, bool done) {
  if (p.converged) {
    const uint32_t cont = __ballot_sync(act, !done);
    act = cont;
  }
  return done;
}

// One kernel for both micro-benchmarks.  kHist: record {proc,op,arg,ret,call,end} per op.
// Split mode ("each thread is a pure producer or a pure consumer"): the role is fixed for the whole launch, so
// producers and consumers run two separate loops.  One shared loop with `if (producer) ... if (consumer) ...` inside
// makes the two halves of a mixed warp wait for each other at the reconvergence point of every iteration, i.e. run
// one after the other (measured: 27 Gops/s at p = 0.5 against 56 with homogeneous warps).
template <class Q, bool kHist, int kWarpFaa, bool kFused = false>
__global__ void __launch_bounds__(512, 2) bench_kernel(Q q, BenchParams p, uint64_t* ctr, gq_hist_rec* hist) {
  cg::grid_group grid = cg::this_grid();
  __shared__ BlockFunnel s_funnels[kWarpFaa == 2 ? kFunnelsPerQueue : 1];
  if (kWarpFaa == 2) {                                  // D11: this block's ticket funnels, one per hot counter
    funnel_init(s_funnels, kFunnelsPerQueue, p.funnel_window_ns);
    q = with_funnels(q, s_funnels);
  }
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid == 0) st_relaxed(ctr + C_T0, globaltimer_ns());
  grid.sync();                                        // one time base for every thread
  const uint64_t t0 = ld_relaxed(ctr + C_T0);
  const bool fixed = p.ops_per_thread != 0;
  const uint64_t tw = fixed ? 0 : t0 + p.warmup_ns;
  const uint64_t te = fixed ? ~0ull : tw + p.duration_ns;
  Tally a;

  if (tid < p.threads) {
    const uint32_t ltid = p.perm ? p.perm[tid] : tid;      // logical thread (roles, payloads, records); tid = physical
    thread_ctx ctx{ltid};
    ctx.help_peer = ltid + 1;
    const bool split = p.mode == MODE_SPLIT;
    const bool do_enq = !split || (uint64_t)mix32(p.seed * 0x9e3779b9u + ltid) < p.prod_threshold;
    gq_hist_rec* my = kHist ? hist + (size_t)ltid * p.ops_per_thread * (split ? 1 : 2) : nullptr;
    if (kFused && HasFused<Q>::value) {                     // split mode, mixed warps, one converged call per iteration
      // p.fused == 1: gq::enqueue_or_dequeue_step, lanes that have to wait in line hand the wait back (PENDING) and the warp
      // goes on; the operation of such a lane spans several iterations.  p.fused == 2: the blocking gq::enqueue_or_dequeue.
      uint32_t act = __activemask();
      op_state st;
      uint32_t iter = 0;
      uint64_t t_call = 0;
      // a thread has one role: one set of tallies in the loop (the kernel sits at its register limit), sorted by role afterwards
      uint32_t n_succ = 0, n_fail = 0, n_tot = 0, n_tot_fail = 0;
      uint64_t sum = 0;
      for (;;) {
        uint32_t v = payload_of(p, ltid, iter);
        const uint32_t v_in = v;
        if (kHist && !st.pending()) {
          if (p.jitter_ns) __nanosleep(mix32(p.seed ^ (ltid * 0x85ebca6bu) ^ (iter * 2u + 0x1234567u)) % (p.jitter_ns + 1));
          t_call = globaltimer_ns();
        }
        const int s = p.fused == 2 ? fused_op<kWarpFaa>(q, ctx, do_enq, &v, &a.retries)
                                   : fused_step<kWarpFaa>(q, ctx, st, do_enq, &v, &a.retries);
        if (kHist) { __threadfence(); }
        const uint64_t now = globaltimer_ns();
        bool done = false;
        if (s != PENDING) {
          if (kHist) *my++ = do_enq ? gq_hist_rec{ltid, GQ_OP_ENQ, v_in, (uint32_t)s, 0u, 0u, t_call, now}
                                    : gq_hist_rec{ltid, GQ_OP_DEQ, 0u, (uint32_t)s, s == OK ? v : 0u, 0u, t_call, now};
          const bool in = now >= tw && now < te;
          if (s == OK) { ++n_tot; sum += v; n_succ += in; } else { ++n_tot_fail; n_fail += in; }   // v: the payload put in / taken out
          ++iter;
          done = fixed ? (iter >= p.ops_per_thread) : (now >= te);   // a pending operation is always brought to its end
        }
        if (loop_done(p, act, done)) break;
      }
      if (do_enq) { a.succ_enq = n_succ; a.full = n_fail; a.tot_enq = n_tot; a.tot_full = n_tot_fail; a.sum_enq = sum; }
      else        { a.succ_deq = n_succ; a.empty = n_fail; a.tot_deq = n_tot; a.tot_empty = n_tot_fail; a.sum_deq = sum; }
    } else if (!split) {
      uint32_t act = __activemask();
      for (uint32_t iter = 0;; ++iter) {
        enq_step<Q, kHist, kWarpFaa>(q, ctx, p, ltid, iter, tw, te, a, my);
        const uint64_t now = deq_step<Q, kHist, kWarpFaa>(q, ctx, p, ltid, iter, tw, te, a, my);
        if (loop_done(p, act, fixed ? (iter + 1 >= p.ops_per_thread) : (now >= te))) break;
      }
    } else if (do_enq) {
      uint32_t act = __activemask();
      for (uint32_t iter = 0;; ++iter) {
        const uint64_t now = enq_step<Q, kHist, kWarpFaa>(q, ctx, p, ltid, iter, tw, te, a, my);
        if (loop_done(p, act, fixed ? (iter + 1 >= p.ops_per_thread) : (now >= te))) break;
      }
    } else {
      uint32_t act = __activemask();
      for (uint32_t iter = 0;; ++iter) {
        const uint64_t now = deq_step<Q, kHist, kWarpFaa>(q, ctx, p, ltid, iter, tw, te, a, my);
        if (loop_done(p, act, fixed ? (iter + 1 >= p.ops_per_thread) : (now >= te))) break;
      }
    }
  }
  __syncwarp();
  // warp-reduce, one atomic per warp per counter
  uint64_t vals[11] = {a.succ_enq, a.succ_deq, a.full, a.empty, a.tot_enq, a.tot_deq, a.tot_full, a.tot_empty, a.sum_enq, a.sum_deq, a.retries};
#pragma unroll
  for (int i = 0; i < 11; ++i) {
    const uint64_t s = warp_sum(vals[i]);
    if (lane_id() == 0 && s) red_add_relaxed(ctr + i, s);
  }
  if (tid == 0) red_max_relaxed(ctr + C_T_END, globaltimer_ns());
}

// ---- service kernels --------------------------------------------------------------------
// One warp enqueues vals[0..count) in array order.  On a quiescent queue the fast path succeeds
// at the first ticket, so lane order = ticket order = FIFO order.  Two cases need care:
//  - G-WFQ-YMC after EMPTY dequeues has H > T, and the cells in between are burnt (marked top):
//    T is first advanced to H, which is what the failed tickets would do one by one;
//  - all-slow builds (patience 0) place concurrent requests in any order, which is linearizable
//    but not array order: `serial` makes the lanes take turns.
__device__ __forceinline__ void prefill_prepare(const LfqView&) {}
__device__ __forceinline__ void prefill_prepare(const DlfqView&) {}
__device__ __forceinline__ void prefill_prepare(const WfqView&) {}
__device__ __forceinline__ void prefill_prepare(const YmcView& q) { Ymc::advance(q.tail, ld_acquire(q.head)); }

// `lanes` (<= 32, <= the queue's max_threads) lanes of the warp take part: thread_ctx::tid indexes per-thread records.
template <class Q>
__global__ void prefill_kernel(Q q, const uint32_t* vals, uint64_t count, uint64_t* n_ok, uint32_t serial, uint32_t lanes) {
  thread_ctx ctx{threadIdx.x};
  uint64_t ok = 0;
  if (threadIdx.x == 0) prefill_prepare(q);
  __syncwarp();
  for (uint64_t base = 0; base < count; base += lanes) {
    const uint64_t i = base + threadIdx.x;
    const bool mine = threadIdx.x < lanes && i < count;
    if (serial) {
      for (uint32_t l = 0; l < lanes; ++l) {
        if (threadIdx.x == l && mine && enqueue<false, true>(q, ctx, vals[i]) == OK) ++ok;
        __syncwarp();
      }
    } else {
      if (mine && enqueue<true, true>(q, ctx, vals[i]) == OK) ++ok;
    }
    __syncwarp();
  }
  ok = warp_sum(ok);
  if (threadIdx.x == 0) *n_ok = ok;
}

// One warp dequeues until EMPTY (or max) in FIFO order.  Each round's values are written in the
// order of the tickets they were dequeued at (thread_ctx::last_ticket: AQ head ticket / YMC
// cell), not in lane order: a lane that met a hole left by an abandoned ticket retries at a
// later ticket.  Rounds are sequential, so ticket order across rounds is round order.
template <class Q>
__global__ void drain_kernel(Q q, uint32_t* out, uint64_t max, uint64_t* n_out, uint32_t lanes) {
  thread_ctx ctx{threadIdx.x};
  uint64_t n = 0;
  for (;;) {
    const uint64_t want = max - n < lanes ? max - n : lanes;
    if (want == 0) break;
    uint32_t v = 0;
    int s = EMPTY;
    if (threadIdx.x < want) s = dequeue<true, true>(q, ctx, &v);
    __syncwarp();
    const uint32_t okmask = __ballot_sync(0xffffffffu, s == OK);
    const uint64_t mine = s == OK ? ctx.last_ticket : ~0ull;
    uint32_t rank = 0;
    for (int l = 0; l < 32; ++l) rank += __shfl_sync(0xffffffffu, mine, l) < mine;
    if (s == OK) out[n + rank] = v;
    n += __popc(okmask);
    if (__popc(okmask) < (int)want) break;
  }
  if (threadIdx.x == 0) *n_out = n;
}

// Single thread runs a script of operations (differential test against the sequential model).
template <class Q>
__global__ void script_kernel(Q q, const uint32_t* op, const uint32_t* arg, uint64_t count, uint32_t tid,
                              uint32_t* status, uint32_t* val) {
  thread_ctx ctx{tid};
  for (uint64_t i = 0; i < count; ++i) {
    uint32_t v = 0;
    const int s = op[i] == GQ_OP_ENQ ? enqueue<false, true>(q, ctx, arg[i]) : dequeue<false, true>(q, ctx, &v);
    status[i] = (uint32_t)s;
    val[i] = v;
  }
}

// Lemma III.1 probe: warp_faa inside seeded, nested divergent control flow.
// funnel_mode: 0 = plain WAVEFAA, 1 = through a block-level funnel (D11) with window funnel_window_ns.  tickets == nullptr:
// the tickets are only summed (long soak runs); *checksum then holds the sum of all tickets handed out.
__global__ void warp_faa_probe_kernel(uint64_t* counter, uint32_t threads, uint32_t rounds, uint32_t seed, uint64_t* tickets,
                                      uint32_t funnel_mode, uint32_t funnel_window_ns, unsigned long long* checksum) {
  __shared__ BlockFunnel s_funnel[1];
  if (funnel_mode) funnel_init(s_funnel, 1, funnel_window_ns);
  BlockFunnel* f = funnel_mode ? s_funnel : nullptr;
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= threads) return;
  unsigned long long sum = 0, n = 0;
  for (uint32_t r = 0; r < rounds; ++r) {
    const uint32_t h = mix32(seed ^ (tid * 0x9e3779b9u) ^ (r * 0x85ebca6bu));
    uint64_t t = ~0ull;
    if (h & 1) {                       // participate?
      if (h & 2) {                     // two diverged groups name the same counter
        if (h & 4) __nanosleep(h >> 24);
        t = warp_faa<true>(counter, 1, f);
      } else {
        t = warp_faa<false>(counter, 1, f);  // address-matched variant
      }
      sum += t; ++n;
    }
    if (tickets) tickets[(size_t)tid * rounds + r] = t;
  }
  if (checksum) { atomicAdd(checksum, sum); atomicAdd(checksum + 1, n); }
}

// Ceiling C1: bare WAVEFAA loop (BASELINE.json north_star: "a bare warp-aggregated FAA loop on one
// counter at the same occupancy").  counters are 1 KiB apart.
template <int kWarpFaa>
__global__ void __launch_bounds__(512) faa_ceiling_kernel(uint64_t* counters, uint32_t n_counters, BenchParams p, uint64_t* ctr) {
  cg::grid_group grid = cg::this_grid();
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid == 0) st_relaxed(ctr + C_T0, globaltimer_ns());
  grid.sync();
  const uint64_t t0 = ld_relaxed(ctr + C_T0);
  const bool fixed = p.ops_per_thread != 0;
  const uint64_t tw = fixed ? 0 : t0 + p.warmup_ns, te = fixed ? ~0ull : tw + p.duration_ns;
  uint64_t n_in = 0, n_tot = 0, acc = 0;
  if (tid < p.threads) {
    for (uint32_t iter = 0;; ++iter) {
      uint64_t* c = counters + (size_t)(iter % n_counters) * 128;
      acc ^= kWarpFaa ? warp_faa<true>(c) : lane_faa(c);
      const uint64_t now = globaltimer_ns();
      ++n_tot; n_in += (now >= tw && now < te);
      if (fixed ? (iter + 1 >= p.ops_per_thread) : (now >= te)) break;
    }
  }
  __syncwarp();
  const uint64_t a = warp_sum(n_in), b = warp_sum(n_tot), x = warp_sum(acc);
  if (lane_id() == 0) { if (a) red_add_relaxed(ctr + C_SUCC_ENQ, a); if (b) red_add_relaxed(ctr + C_TOT_ENQ, b); if (x == 1) red_add_relaxed(ctr + C_RETRIES, 1); }
  if (tid == 0) red_max_relaxed(ctr + C_T_END, globaltimer_ns());
}

// Ceiling C2: what one ring operation does to its slot, without tickets: a coalesced
// {8 B load, 64-bit CAS, red.or} stream over `slots` consecutive words.
__global__ void __launch_bounds__(512) slot_ceiling_kernel(uint64_t* buf, uint64_t slots, BenchParams p, uint64_t* ctr) {
  cg::grid_group grid = cg::this_grid();
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid == 0) st_relaxed(ctr + C_T0, globaltimer_ns());
  grid.sync();
  const uint64_t t0 = ld_relaxed(ctr + C_T0);
  const bool fixed = p.ops_per_thread != 0;
  const uint64_t tw = fixed ? 0 : t0 + p.warmup_ns, te = fixed ? ~0ull : tw + p.duration_ns;
  uint64_t n_in = 0, n_tot = 0;
  if (tid < p.threads) {
    for (uint32_t iter = 0;; ++iter) {
      uint64_t* s = buf + ((uint64_t)tid + (uint64_t)iter * p.threads) % slots;
      const uint64_t e = ld_relaxed(s);
      cas_relaxed(s, e, e + 2);
      red_or_relaxed(s, 1);
      const uint64_t now = globaltimer_ns();
      ++n_tot; n_in += (now >= tw && now < te);
      if (fixed ? (iter + 1 >= p.ops_per_thread) : (now >= te)) break;
    }
  }
  __syncwarp();
  const uint64_t a = warp_sum(n_in), b = warp_sum(n_tot);
  if (lane_id() == 0) { if (a) red_add_relaxed(ctr + C_SUCC_ENQ, a); if (b) red_add_relaxed(ctr + C_TOT_ENQ, b); }
  if (tid == 0) red_max_relaxed(ctr + C_T_END, globaltimer_ns());
}

}  // namespace gqk
