// gq/detail/prim.cuh — device primitives for sm_100a.
//
// Memory-model wrappers.  Every shared word of the queues is accessed through these: explicit
// order (.relaxed / .acquire / .release), explicit scope (.gpu) and explicit state space
// (.global).  They are what cuda::atomic_ref<T, thread_scope_device> means, minus its
// generic-address lowering: on sm_100a nvcc 12.9 turns atomic_ref on a generic pointer into
// ATOM.E + an ATOMS.CAST.SPIN shared-memory fallback branch per call and never emits RED for
// a discarded result.  With .global the SASS is one
// ATOMG / REDG / LDG.STRONG.GPU per call.
//
// WAVEFAA (Alg. 1, Lemma III.1) is warp_faa() below, re-derived for
// 32-lane warps with independent thread scheduling (reading G10).
#pragma once
#include <climits>
#include <cstdint>
#include <cstdio>

#include "debug.cuh"

namespace gq {
namespace detail {

__device__ __forceinline__ uint32_t lane_id() { uint32_t l; asm("mov.u32 %0, %%laneid;" : "=r"(l)); return l; }
__device__ __forceinline__ uint32_t lanemask_lt() { uint32_t m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }
// %globaltimer: ns, one clock for the whole GPU.  volatile + memory clobber keep the read
// where it is written relative to the surrounding memory operations (reading H1).
__device__ __forceinline__ uint64_t globaltimer_ns() {
  uint64_t t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t) :: "memory"); return t;
}

// ---- loads / stores -------------------------------------------------------------------
__device__ __forceinline__ uint64_t ld_relaxed(const uint64_t* p) {
  uint64_t v; asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ uint64_t ld_acquire(const uint64_t* p) {
  uint64_t v; asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ uint32_t ld_relaxed32(const uint32_t* p) {
  uint32_t v; asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ uint32_t ld_acquire32(const uint32_t* p) {
  uint32_t v; asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_relaxed(uint64_t* p, uint64_t v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_release(uint64_t* p, uint64_t v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_relaxed32(uint32_t* p, uint32_t v) {
  asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void st_release32(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_acq_rel() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }

// ---- read-modify-write ----------------------------------------------------------------
__device__ __forceinline__ uint64_t faa_relaxed(uint64_t* p, uint64_t v) {
  uint64_t o; asm volatile("atom.relaxed.gpu.global.add.u64 %0, [%1], %2;" : "=l"(o) : "l"(p), "l"(v) : "memory"); return o;
}
__device__ __forceinline__ void red_add_relaxed(uint64_t* p, uint64_t v) {
  asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void red_or_relaxed(uint64_t* p, uint64_t v) {
  asm volatile("red.relaxed.gpu.global.or.b64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint64_t fetch_max_relaxed(uint64_t* p, uint64_t v) {
  uint64_t o; asm volatile("atom.relaxed.gpu.global.max.u64 %0, [%1], %2;" : "=l"(o) : "l"(p), "l"(v) : "memory"); return o;
}
__device__ __forceinline__ void red_max_relaxed(uint64_t* p, uint64_t v) {
  asm volatile("red.relaxed.gpu.global.max.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void red_max_s64_relaxed(int64_t* p, int64_t v) {
  asm volatile("red.relaxed.gpu.global.max.s64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
// CAS returning the value found (success iff result == expected).
__device__ __forceinline__ uint64_t cas_relaxed(uint64_t* p, uint64_t expected, uint64_t desired) {
  uint64_t o; asm volatile("atom.relaxed.gpu.global.cas.b64 %0, [%1], %2, %3;" : "=l"(o) : "l"(p), "l"(expected), "l"(desired) : "memory"); return o;
}
__device__ __forceinline__ uint64_t cas_release(uint64_t* p, uint64_t expected, uint64_t desired) {
  uint64_t o; asm volatile("atom.release.gpu.global.cas.b64 %0, [%1], %2, %3;" : "=l"(o) : "l"(p), "l"(expected), "l"(desired) : "memory"); return o;
}
__device__ __forceinline__ uint64_t cas_acq_rel(uint64_t* p, uint64_t expected, uint64_t desired) {
  uint64_t o; asm volatile("atom.acq_rel.gpu.global.cas.b64 %0, [%1], %2, %3;" : "=l"(o) : "l"(p), "l"(expected), "l"(desired) : "memory"); return o;
}
__device__ __forceinline__ uint32_t cas_relaxed32(uint32_t* p, uint32_t expected, uint32_t desired) {
  uint32_t o; asm volatile("atom.relaxed.gpu.global.cas.b32 %0, [%1], %2, %3;" : "=r"(o) : "l"(p), "r"(expected), "r"(desired) : "memory"); return o;
}
__device__ __forceinline__ uint32_t cas_acq_rel32(uint32_t* p, uint32_t expected, uint32_t desired) {
  uint32_t o; asm volatile("atom.acq_rel.gpu.global.cas.b32 %0, [%1], %2, %3;" : "=r"(o) : "l"(p), "r"(expected), "r"(desired) : "memory"); return o;
}

// ---- block-level ticket funnel (D11; "Aggregating Funnels ... our G-LFQ uses this direction as
//      inspiration", L95) ------------------------------------------------------------------------------------------
// One BlockFunnel per (thread block, hot counter), in shared memory.  The leaders of the warps of a block that ask for
// tickets of the same counter at about the same time are combined into ONE global FAA:
//   join    : old = atomicAdd(gate, <1 warp, cnt tickets>)   ->  batch number, place in the batch, ticket offset
//   combine : the warp that opened the batch (place 0) closes it with atomicExch(gate, <next batch, 0, 0>), issues
//             FAA(counter, total) and publishes the base in the batch's slot;
//   follow  : every other warp of the batch waits for that slot and takes base + its offset.
// Nobody waits for a warp that is not already executing these very steps: a follower waits for its combiner, which is
// inside its FAA; a combiner waits only for the previous tenant of its slot (an older batch, same argument).  A warp
// that finds the gate idle pays two shared-memory atomics more than the plain WAVEFAA.  `window_ns` > 0 keeps a batch
// open that long so that more warps can join (fewer global atomics against a longer wait for the ticket).
// Lemma III.1 carries over batch-wise: one FAA of `total` hands out `total` distinct consecutive tickets, each warp gets
// the contiguous sub-range [off, off + cnt), each lane its rank inside it.
constexpr uint32_t kFunnelSlots = 8;
struct FunnelSlot { unsigned long long base; unsigned int seq; unsigned int readers; };
struct alignas(16) BlockFunnel {
  unsigned long long gate;                  // [63:32] batch | [31:16] warps joined | [15:0] tickets asked
  unsigned int window_ns, _pad;
  FunnelSlot slot[kFunnelSlots];
};
// call with the whole block before first use (ends with __syncthreads)
__device__ __forceinline__ void funnel_init(BlockFunnel* f, uint32_t n, uint32_t window_ns) {
  for (uint32_t i = threadIdx.x; i < n * kFunnelSlots; i += blockDim.x) {
    FunnelSlot* s = &f[i / kFunnelSlots].slot[i % kFunnelSlots];
    s->base = 0; s->readers = 0; s->seq = (i % kFunnelSlots) - kFunnelSlots;      // "batch seq - slots was published and read"
  }
  for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) { f[i].gate = 0; f[i].window_ns = window_ns; }
  __syncthreads();
}

// ---- WAVEFAA --------------------------------------------------------------------------
// PAPER.md Alg. 1: mask <- Ballot(active); count <- Popcount(mask); leader <-
// FirstSetBit(mask)-1; leader: base <- FAA(C, count); base <- Shuffle(base, leader);
// rank <- Popcount(mask & lower_lanes(lane)); return base + rank.
//
// sm_100a: the "active" set is whatever group of lanes is converged here.  kUniform = true
// takes __activemask() as is (all converged callers name the same counter: benchmark
// kernels, where divergence by role already splits the groups).  kUniform = false groups
// lanes by counter address with match.any first, so converged lanes may target different
// queues.  The one mask is used for leader, rank and shuffle; lanes outside it take no part,
// and no lane waits for a lane outside its own mask (reading G10).  `unit` scales the add
// for packed counters (G-WFQ: unit = 1 << THRIDX_BITS); the returned value is the raw word
// base + rank*unit.
// The funnel steps of one WAVEFAA group (mask, leader), executed by ALL lanes of the group together: only single atomics sit
// inside `if (lead)`, every wait is a loop the whole group runs converged, and results travel by __shfl_sync(mask).
// (Measured on sm_100a: when only the leader waited, inside a divergent region, with its group parked at the compiler's
//  reconvergence barrier, other diverged groups of the same warp passing through the same code released that barrier
//  early and the group read the leader's base before it was there.  No lane may wait for another one at a BSYNC.)
__device__ __forceinline__ uint64_t funnel_faa(BlockFunnel* f, uint64_t* counter, uint64_t unit, uint32_t mask, uint32_t leader) {
  const bool lead = lane_id() == leader;
  unsigned long long old = 0;
  if (lead) old = atomicAdd(&f->gate, (1ull << 16) | (unsigned long long)__popc(mask));          // join
  old = __shfl_sync(mask, old, leader);
  const uint32_t seq = (uint32_t)(old >> 32), place = (uint32_t)(old >> 16) & 0xFFFFu, off = (uint32_t)old & 0xFFFFu;
  FunnelSlot* s = &f->slot[seq & (kFunnelSlots - 1)];
  volatile unsigned int* vseq = &s->seq;
  volatile unsigned int* vreaders = &s->readers;
  if (place != 0) {                                                   // follow (the whole group)
    [[maybe_unused]] uint32_t sn = 0;
    while (*vseq != seq) {                                            // the nap lets diverged lanes of this very warp run: the combiner may be one
      if (GQ_STUCK(sn, 50, seq, &f->gate, &s->base, &s->seq)) break;
      __nanosleep(20);
    }
    const uint64_t base = *reinterpret_cast<volatile unsigned long long*>(&s->base);
    if (lead) atomicSub(&s->readers, 1u);
    return base + (uint64_t)off * unit;
  }
  if (f->window_ns) __nanosleep(f->window_ns);                        // combine
  unsigned long long closed = 0;
  if (lead) closed = atomicExch(&f->gate, (unsigned long long)(seq + 1u) << 32);
  closed = __shfl_sync(mask, closed, leader);
  const uint32_t total = (uint32_t)closed & 0xFFFFu, warps = (uint32_t)(closed >> 16) & 0xFFFFu;
  uint64_t base = 0;
  if (lead) base = faa_relaxed(counter, (uint64_t)total * unit);
  base = __shfl_sync(mask, base, leader);                             // the group waits for the FAA here, converged
#ifdef GQ_DBG_SITES
  if (lead && (blockIdx.x & 63u) == 0) { GQ_COUNT(22, 1); GQ_COUNT(23, warps); }   // funnel batches, groups per batch (sampled blocks)
#endif
  {
    [[maybe_unused]] uint32_t sn = 0;
    while (*vseq != seq - kFunnelSlots || *vreaders != 0) {           // previous tenant of the slot published and read
      if (GQ_STUCK(sn, 51, seq, &f->gate, &s->base, &s->seq)) break;
      __nanosleep(20);
    }
    if (lead) {
      *reinterpret_cast<volatile unsigned long long*>(&s->base) = base;
      *vreaders = warps - 1u;
      __threadfence_block();
      *vseq = seq;
    }
  }
  return base;
}

template <bool kUniform>
__device__ __forceinline__ uint64_t warp_faa(uint64_t* counter, uint64_t unit = 1, BlockFunnel* funnel = nullptr) {
  const uint32_t active = __activemask();
  uint32_t mask = active;
  if (!kUniform) mask = __match_any_sync(active, reinterpret_cast<unsigned long long>(counter));
#ifdef GQ_DBG_SITES
  if (kUniform && __match_any_sync(mask, reinterpret_cast<unsigned long long>(counter)) != mask) GQ_COUNT(71, 1);   // kUniform promise broken
#endif
  const uint32_t leader = __ffs(mask) - 1;
  const uint32_t rank = __popc(mask & lanemask_lt()) + (GQ_MUT(MUT_RANK_OFF_BY_ONE) ? 1u : 0u);
  // Only a whole warp goes through the funnel: then no warp ever has two groups inside one (a follower and its combiner,
  // or a combiner and a reader it waits for, in the same warp would depend on how the hardware interleaves diverged lanes);
  // the stragglers of a diverged warp draw their tickets directly.
  if (funnel && mask == 0xFFFFFFFFu) return funnel_faa(funnel, counter, unit, mask, leader) + (uint64_t)rank * unit;
  uint64_t base = 0;
  if (lane_id() == leader) {
    base = faa_relaxed(counter, (uint64_t)__popc(mask) * unit);
#ifdef GQ_DBG_SITES
    if ((blockIdx.x & 63u) == 0) { GQ_COUNT(20, 1); GQ_COUNT(21, __popc(mask)); }   // WAVEFAA batch size (sampled blocks)
    if ((blockIdx.x & 63u) == 0 && lane_id() == (uint32_t)__ffs(active) - 1) { GQ_COUNT(24, 1); GQ_COUNT(25, __popc(active)); }   // converged set
#endif
  }
  // One shuffle over the converged set, every lane reading from the leader of its own group.  (A shuffle per group,
  // __shfl_sync(mask, ..), is a WARPSYNC on lane-dependent masks: measured on sm_100a, it splits the converged warp
  // into its address groups for good, and the groups then run one after the other, each waiting out the other's L2
  // round trips: the fused mixed-role operation of lfq.cuh was no faster than two diverged calls because of it.)
  base = __shfl_sync(active, base, leader);
  return base + (uint64_t)rank * unit;
}
// Two WAVEFAAs issued back to back by the same leader before either result is consumed: the two
// L2 round trips overlap (DESIGN.md departure D5, "paired reservation").  Lemma III.1 holds for
// each counter separately: one group, one leader, one FAA per counter, ranks from the same mask.
template <bool kUniform>
__device__ __forceinline__ void warp_faa2(uint64_t* ca, uint64_t* cb, uint64_t unit_a, uint64_t unit_b, uint64_t* a, uint64_t* b) {
  const uint32_t active = __activemask();
  uint32_t mask = active;
  if (!kUniform) {
    const uint32_t ma = __match_any_sync(active, reinterpret_cast<unsigned long long>(ca));
    mask = ma & __match_any_sync(active, reinterpret_cast<unsigned long long>(cb));
  }
  const uint32_t leader = __ffs(mask) - 1;
  const uint32_t rank = __popc(mask & lanemask_lt());
  uint64_t ba = 0, bb = 0;
  if (lane_id() == leader) {
    ba = faa_relaxed(ca, (uint64_t)__popc(mask) * unit_a);
    bb = faa_relaxed(cb, (uint64_t)__popc(mask) * unit_b);
  }
  ba = __shfl_sync(active, ba, leader);
  bb = __shfl_sync(active, bb, leader);
  *a = ba + (uint64_t)rank * unit_a;
  *b = bb + (uint64_t)rank * unit_b;
}
// The "naive" per-thread FAA of PAPER.md L95, kept for the ablation (GQ_F_PER_LANE_FAA).
// ptxas (12.9, sm_100a) warp-aggregates an atom.add by itself when it can prove the address and the
// operand warp-uniform (queue views are kernel parameters, so it can): SASS shows an elected lane and
// one ATOMG.  The term below is always 0 but depends on the thread index, which keeps the address
// from being provably uniform, so that this really is one FAA per thread.
__device__ __forceinline__ uint64_t lane_faa(uint64_t* counter, uint64_t unit = 1) {
  counter += (blockIdx.x * blockDim.x + threadIdx.x) >> 31;
  return faa_relaxed(counter, unit);
}

// Same batching for FAA(Threshold, -1) (Alg. 1): lanes of one group get the values
// a lane-ordered sequence of single decrements would have returned.
template <bool kUniform>
__device__ __forceinline__ int64_t warp_dec(int64_t* counter) {
  const uint32_t active = __activemask();
  uint32_t mask = active;
  if (!kUniform) mask = __match_any_sync(active, reinterpret_cast<unsigned long long>(counter));
  const uint32_t leader = __ffs(mask) - 1;
  const uint32_t rank = __popc(mask & lanemask_lt());
  uint64_t base = 0;
  if (lane_id() == leader) base = faa_relaxed(reinterpret_cast<uint64_t*>(counter), (uint64_t)(-(int64_t)__popc(mask)));
  base = __shfl_sync(active, base, leader);
  return (int64_t)base - (int64_t)rank;
}

// ---- modular cycle compare (PAPER.md Lemma III.6) -----------------------------
// a is newer than b iff 0 < (a - b) mod R < R/2, R = 2^bits.
template <int kBits>
__device__ __host__ __forceinline__ bool cycle_newer(uint32_t a, uint32_t b) {
  constexpr uint32_t R_MASK = kBits == 32 ? 0xFFFFFFFFu : ((1u << (kBits & 31)) - 1u);
  const uint32_t d = (a - b) & R_MASK;
  return d != 0 && d < (1u << (kBits - 1));
}

// bounded exponential backoff for retry loops (north_star: "bounded spin with __nanosleep backoff")
struct Backoff {
  uint32_t ns = 0;
  __device__ __forceinline__ void pause() {
    if (ns) __nanosleep(ns);
    ns = ns ? (ns < 1024 ? ns * 2 : 1024) : 32;
  }
};

// counter-based 32-bit mixer (roles, jitter): not part of any queue algorithm
__device__ __host__ __forceinline__ uint32_t mix32(uint32_t x) {
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}

}  // namespace detail
}  // namespace gq
