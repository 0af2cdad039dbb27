// gq/detail/debug.cuh — instrumentation and fault injection, all compiled out of the product build.
//
// Three independent build switches (passed through GQ_NVCC_EXTRA, see paper_2606_01693_b200/build.py);
// without them every macro below is a constant and the hot-path headers carry no debug code:
//
//   -DGQ_DBG_SITES          per-site event counters (GQ_SITE) and a trace ring holding the first
//                           kTraceCap abnormal events of a launch (GQ_TRACE); read back with the
//                           C-ABI call gq_dbg_sites / gq_dbg_trace (gq.h, same switch).
//   -DGQ_DEBUG_STUCK=<cap>  livelock detector (SURVEY section 5 "failure detection"): a retry loop
//                           that passes <cap> iterations records where it is and ends the kernel.
//   -DGQ_MUTANTS            fault-injection build (SURVEY section 4 "mutation tests"): every GQ_MUT(n)
//                           site is compiled in and gq_set_mutation(n) arms exactly one of them at run
//                           time.  tests/test_mutants_gpu.py shows that the parity suite refuses each.
#pragma once
#include <cstdint>

namespace gq {
namespace detail {

// ---- fault injection ----------------------------------------------------------------------------
// The mutants (each one a plausible mistake in the path; PAPER.md lines of the step it breaks):
enum : uint32_t {
  MUT_NONE = 0,
  MUT_NO_RELOAD = 1,        // TRYDEQ walks away after a failed slot CAS instead of reloading (reading G6): lost item
  MUT_NO_HANDSHAKE = 2,     // payload stored after the index is published, reader does not wait for it (P:L88 order): stale value
  MUT_WRONG_CELL = 3,       // dequeue reads Data[idx ^ 1] (P:L88 indirection): foreign / duplicate value
  MUT_UNSOUND_EMPTY = 4,    // emptiness probe reports EMPTY while Tail <= Head + 2 (P:L197 off by two): EMPTY with items present
  MUT_EARLY_RECYCLE = 5,    // index goes back to FQ before its payload has been read (P:L88 order on the dequeue side)
  MUT_RANK_OFF_BY_ONE = 6,  // WAVEFAA rank counts the own lane (Alg. 1, Lemma III.1): tickets handed out twice
  MUT_NO_THR_RESET = 7,     // enqueue never resets Threshold (Alg. 1): EMPTY with items present once it is negative
  MUT_SLOW_NO_FIN = 8,      // G-WFQ: slow-path install does not finalise the request: item enqueued twice
  MUT_YMC_NO_CLAIM = 9,     // G-WFQ-YMC: fast dequeue takes the value without claiming the cell ([5] deq_fast): item dequeued twice
  MUT_LIFO_PAIR = 10,       // ring enqueue installs at slot t ^ 1 (P:L107 SLOT): neighbouring tickets swap their FIFO places
  MUT_P2_ANY_SIDE = 11,     // G-WFQ: a phase-2 helper accepts a Tail-round record while helping on Head and vice versa (Alg. 2):
                            // INC cleared on a local word whose round nobody won, two requests share one ticket, items lost
  MUT_COUNT
};
// self-contained (prim.cuh includes this file): plain volatile accesses are good enough for diagnostics
__device__ __forceinline__ uint64_t dbg_ld(const void* p) { return p ? *static_cast<const volatile uint64_t*>(p) : 0; }
__device__ __forceinline__ uint64_t dbg_now() { uint64_t t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t) :: "memory"); return t; }
#ifndef GQ_DBG_SITES
#undef GQ_TRACE_BY_INDEX
#endif
#ifdef GQ_MUTANTS
static __device__ uint32_t g_mutation = 0;
#define GQ_MUT(n) (::gq::detail::g_mutation == (uint32_t)(n))
#else
#define GQ_MUT(n) false
#endif

// ---- event counters and trace ring --------------------------------------------------------------
#ifdef GQ_DBG_SITES
constexpr uint32_t kTraceCap = 1u << 16;
struct TraceRec { uint64_t ns, site_tid, ticket, entry, head, tail; int64_t thr; uint64_t aux; };
static __device__ unsigned long long g_dbg[80];      // [0,32) event counters, [32,48) latency sums (clock cycles), [48,64) latency samples
static __device__ unsigned long long g_trace_n;
static __device__ TraceRec g_trace[kTraceCap];
#define GQ_SITE(i) atomicAdd(&::gq::detail::g_dbg[i], 1ull)
#define GQ_COUNT(i, v) atomicAdd(&::gq::detail::g_dbg[i], (unsigned long long)(v))
// first kTraceCap events only; once the ring is full the cost is one load of its own line
#ifndef GQ_TRACE_MIN
#define GQ_TRACE_MIN 0       /* -DGQ_TRACE_MIN=<n>: record only events whose site id (low byte) is >= n */
#endif
#define GQ_TRACE(site, r, ticket, entry, aux)                                                                    \
  do {                                                                                                           \
    if (((site) & 0xffu) >= GQ_TRACE_MIN && ::gq::detail::dbg_ld(&::gq::detail::g_trace_n) < ::gq::detail::kTraceCap) { \
      const unsigned long long i_ = atomicAdd(&::gq::detail::g_trace_n, 1ull);                                   \
      if (i_ < ::gq::detail::kTraceCap)                                                                          \
        ::gq::detail::g_trace[i_] = ::gq::detail::TraceRec{::gq::detail::dbg_now(),                              \
            (uint64_t)(site) | ((uint64_t)(blockIdx.x * blockDim.x + threadIdx.x) << 32), (uint64_t)(ticket), (uint64_t)(entry), \
            ::gq::detail::dbg_ld((r).head), ::gq::detail::dbg_ld((r).tail),                                      \
            (int64_t)::gq::detail::dbg_ld((r).threshold), (uint64_t)(aux)};                                      \
    }                                                                                                            \
  } while (0)
// -DGQ_TRACE_BY_INDEX (with GQ_DBG_SITES): the trace ring is used as tables instead, for chasing the fate of one queue
// index through FQ -> enqueuer -> AQ -> dequeuer -> FQ (this is how the shared phase-2 record of G-WFQ was found, D10):
//   records [0, 65536/2)      the LAST event of each kind (8 kinds) per (ring, index < 4096): GQ_IDX_EVENT
//   records [24576, 24576+2048*16)  the last 16 transitions of each G-WFQ local word of the AQ ring: GQ_L_EVENT
// Both stop recording once event counter 70 is set (a check that wants the state frozen sets it with GQ_COUNT(70, 1)).
#ifdef GQ_TRACE_BY_INDEX
static __device__ unsigned int g_lcnt[2048];
#define GQ_IDX_EVENT(kind, r, idx, ticket, entry, aux)                                                           \
  do {                                                                                                           \
    if (::gq::detail::dbg_ld(&::gq::detail::g_dbg[70]) == 0) {                                                    \
      const uint32_t i_ = (((uint32_t)(idx) & 0xFFFu) + 4096u * (r).id) * 8u + (kind);                            \
      if (i_ < 24576u)                                                                                           \
        ::gq::detail::g_trace[i_] = ::gq::detail::TraceRec{::gq::detail::dbg_now(),                               \
            (uint64_t)(kind) | ((uint64_t)(blockIdx.x * blockDim.x + threadIdx.x) << 32), (uint64_t)(ticket), (uint64_t)(entry), \
            0, 0, 0, (uint64_t)(aux)};                                                                           \
      ::gq::detail::g_trace_n = ::gq::detail::kTraceCap;                                                         \
    }                                                                                                            \
  } while (0)
#define GQ_L_EVENT(r, target, kind, me, a, b)                                                                     \
  do {                                                                                                           \
    if ((r).id == 0 && ::gq::detail::dbg_ld(&::gq::detail::g_dbg[70]) == 0) {                                     \
      const uint32_t t_ = (uint32_t)(target) & 2047u;                                                             \
      const uint32_t n_ = atomicAdd(&::gq::detail::g_lcnt[t_], 1u);                                               \
      ::gq::detail::g_trace[24576 + t_ * 16 + (n_ & 15u)] = ::gq::detail::TraceRec{::gq::detail::dbg_now(),       \
          (uint64_t)(kind) | ((uint64_t)(me) << 32), (uint64_t)(a), (uint64_t)(b), n_, 0, 0, 0};                  \
    }                                                                                                            \
  } while (0)
#else
#define GQ_IDX_EVENT(kind, r, idx, ticket, entry, aux) ((void)0)
#define GQ_L_EVENT(r, target, kind, me, a, b) ((void)0)
#endif
// Sampled latency probes: one thread in 2048 accumulates clock64 deltas per site.  `dep` is the value whose
// arrival ends the interval: the compare makes the (in-order) warp wait for it before the clock is read.
#define GQ_SAMPLED (((blockIdx.x * blockDim.x + threadIdx.x) & 2047u) == 0)
#define GQ_TIC(var) const long long var = GQ_SAMPLED ? clock64() : 0
#define GQ_TOC(site, var, dep)                                                     \
  do {                                                                             \
    if (GQ_SAMPLED) {                                                              \
      if ((uint64_t)(dep) == 0x5DEADBEEF5A5A5A5ull) GQ_SITE(64);                    \
      const long long d_ = clock64() - var;                                        \
      GQ_COUNT(32 + (site), d_); GQ_COUNT(48 + (site), 1);                         \
    }                                                                              \
  } while (0)
#else
#define GQ_SITE(i) ((void)0)
#define GQ_COUNT(i, v) ((void)0)
#define GQ_TRACE(site, r, ticket, entry, aux) ((void)0)
#define GQ_IDX_EVENT(kind, r, idx, ticket, entry, aux) ((void)0)
#define GQ_L_EVENT(r, target, kind, me, a, b) ((void)0)
#define GQ_TIC(var) ((void)0)
#define GQ_TOC(site, var, dep) ((void)0)
#endif

// ---- livelock detector --------------------------------------------------------------------------
// Every retry loop of the slow paths calls GQ_STUCK(counter, location, tid, word pointers...); the first
// thread over the cap records {loc, tid, *a..*d}, raises the abort word, and from then on every
// instrumented loop bails out, so the kernel drains and the host can read the record (capi.cu).
#ifdef GQ_DEBUG_STUCK
static __device__ unsigned long long g_stuck[2 + 16 * 6];
__device__ __forceinline__ bool stuck(uint32_t& n, uint32_t loc, uint32_t tid, const void* a = nullptr, const void* b = nullptr,
                                      const void* c = nullptr, const void* d = nullptr) {
  if ((++n & 1023u) != 0) return false;                       // look at the abort word every 1024th iteration only
  const bool aborted = dbg_ld(&g_stuck[0]) != 0;
  if (!aborted && n < (uint32_t)(GQ_DEBUG_STUCK)) return false;
  const unsigned long long k = atomicAdd(&g_stuck[1], 1ull);
  if (k < 16) {
    unsigned long long* r = g_stuck + 2 + 6 * k;
    r[0] = loc | ((unsigned long long)n << 32); r[1] = tid; r[2] = dbg_ld(a); r[3] = dbg_ld(b); r[4] = dbg_ld(c); r[5] = dbg_ld(d);
  }
  __threadfence();
  *reinterpret_cast<volatile unsigned long long*>(&g_stuck[0]) = 1;
  return true;
}
#define GQ_STUCK(...) ::gq::detail::stuck(__VA_ARGS__)
#else
#define GQ_STUCK(n, ...) ((void)(n), false)
#endif

}  // namespace detail
}  // namespace gq
