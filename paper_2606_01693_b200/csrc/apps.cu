// apps.cu — the application drivers of PAPER.md §V-B (L365-366) behind the C ABI:
//   bfs_run / bfs_run_ex : level-synchronous BFS with two alternating frontier queues
//   rt_render            : tile-based persistent wavefront path tracer on one work queue
// Both use the queues only through the public __device__ API (include/gq/queue.cuh) and the host
// C ABI (queue_create_ex / queue_device_view / queue_destroy): they are clients of the library.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "gq.h"
#include "gq/queue.cuh"
#include "host_util.h"

namespace cg = cooperative_groups;
using namespace gq;
using namespace gq::detail;

namespace {

__device__ __forceinline__ uint64_t warp_sum64(uint64_t v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// G-WFQ-YMC after EMPTY dequeues has H > T with the cells in between burnt: move T up to H before
// the queue is filled again (what the failed tickets would do one by one).
__device__ __forceinline__ void requeue_prepare(const LfqView&) {}
__device__ __forceinline__ void requeue_prepare(const DlfqView&) {}
__device__ __forceinline__ void requeue_prepare(const WfqView&) {}
__device__ __forceinline__ void requeue_prepare(const YmcView& q) { Ymc::advance(q.tail, ld_acquire(q.head)); }
__device__ __forceinline__ bool pool_exhausted(const LfqView&) { return false; }
__device__ __forceinline__ bool pool_exhausted(const DlfqView&) { return false; }
__device__ __forceinline__ bool pool_exhausted(const WfqView&) { return false; }
__device__ __forceinline__ bool pool_exhausted(const YmcView& q) { return ld_relaxed(q.exhausted) != 0; }

template <class Q> struct ViewOf;
template <> struct ViewOf<LfqView> { static constexpr int kind = GQ_LFQ; };
template <> struct ViewOf<DlfqView> { static constexpr int kind = GQ_LFQ_DIRECT; };
template <> struct ViewOf<WfqView> { static constexpr int kind = GQ_WFQ; };
template <> struct ViewOf<YmcView> { static constexpr int kind = GQ_WFQ_YMC; };

// RAII over queue_create_ex / queue_destroy, plus the device view
template <class Q>
struct OwnedQueue {
  gq_queue* h = nullptr;
  Q view{};
  int create(uint64_t capacity, const gq_opts& o) {
    int rc = queue_create_ex(ViewOf<Q>::kind, capacity, &o, &h);
    if (rc) return rc;
    return queue_device_view(h, &view, sizeof view);
  }
  ~OwnedQueue() { if (h) queue_destroy(h); }
};

uint64_t pow2ceil64(uint64_t x) { uint64_t p = 1; while (p < x) p <<= 1; return p; }

}  // namespace

// =====================================================================================  BFS
namespace {

enum { B_NEXT0 = 0, B_NEXT1, B_NEXT2, B_EDGES, B_DEQ, B_ENQ, B_LEVELS, B_ERROR, B_HUGE0, B_HUGE1, B_COUNT = 16 };
#ifndef GQ_BFS_CHUNK
#define GQ_BFS_CHUNK 64
#endif
constexpr uint32_t kChunk = GQ_BFS_CHUNK;      // edges per grid-phase work item (measured at scale 20: 256 -> 0.97 ms, 128 -> 0.90, 64 -> 0.79, 32 -> 0.79)
struct Chunk { uint64_t begin; uint32_t count, _pad; };

struct BfsArgs {
  const uint64_t* rowptr; const uint32_t* col; int32_t* dist;
  uint32_t nv, src, huge_degree, max_chunks;
  uint64_t* ctr; Chunk* chunks;
};

// "newly visited vertices are marked and are enqueued into the next frontier"
template <class Q>
__device__ __forceinline__ void bfs_visit(const Q& nxt, thread_ctx& ctx, const BfsArgs& a, uint32_t w, int32_t d, uint32_t& n_next) {
  int32_t* p = a.dist + w;
  if (ld_relaxed32(reinterpret_cast<const uint32_t*>(p)) != 0xFFFFFFFFu) return;     // already marked (filter)
  if (atomicCAS(p, -1, d) != -1) return;                                             // the mark: exactly one winner
  if (enqueue<true, true>(nxt, ctx, w) != OK) st_relaxed(a.ctr + B_ERROR, 1);
  else ++n_next;
}

template <class Q>
__global__ void __launch_bounds__(512) bfs_kernel(Q qa, Q qb, BfsArgs a) {
  cg::grid_group grid = cg::this_grid();
  __shared__ uint32_t s_end[16][32];
  __shared__ uint64_t s_start[16][32];
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const uint32_t gwarp = tid >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  thread_ctx ctx{tid};
  ctx.help_peer = tid + 1;
  uint64_t edges = 0, n_deq = 0, n_enq = 0;
  if (tid == 0) {
    a.dist[a.src] = 0;
    if (enqueue<false, true>(qa, ctx, a.src) != OK) st_relaxed(a.ctr + B_ERROR, 1);
    n_enq = 1;
  }
  __threadfence();
  grid.sync();
  uint32_t level = 0;
  for (;; ++level) {
    const Q& cur = (level & 1) ? qb : qa;
    const Q& nxt = (level & 1) ? qa : qb;
    uint64_t* next_cnt = a.ctr + B_NEXT0 + (level + 1) % 3;
    uint64_t* huge_cnt = a.ctr + B_HUGE0 + (level & 1);
    if (tid == 0) {                                  // counters nobody touches during this level
      st_relaxed(a.ctr + B_NEXT0 + (level + 2) % 3, 0);
      st_relaxed(a.ctr + B_HUGE0 + ((level + 1) & 1), 0);
    }
    const int32_t d = (int32_t)level + 1;
    uint32_t n_next = 0;
    // ---- phase 1: "the current frontier is dequeued, outgoing neighbors are examined"
    for (;;) {
      uint32_t v = 0;
      const bool have = dequeue<true, true>(cur, ctx, &v) == OK;     // EMPTY is final: nobody enqueues into cur now
      __syncwarp();
      if (!__any_sync(0xffffffffu, have)) break;
      uint64_t start = 0;
      uint32_t deg = 0;
      if (have) {
        ++n_deq;
        start = a.rowptr[v];
        deg = (uint32_t)(a.rowptr[v + 1] - start);
        edges += deg;
        if (deg >= a.huge_degree) {                  // hubs: hand the list to the whole grid (phase 2)
          const uint32_t nch = (deg + kChunk - 1) / kChunk;
          const uint64_t base = faa_relaxed(huge_cnt, nch);
          for (uint32_t c = 0; c < nch; ++c)
            if (base + c < a.max_chunks)
              a.chunks[base + c] = Chunk{start + (uint64_t)c * kChunk, min(kChunk, deg - c * kChunk), 0u};
          deg = 0;
        }
      }
      // the warp's remaining lists, flattened: lane i takes edges i, i+32, ... of the concatenation
      uint32_t incl = deg;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
      const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
      s_end[wib][lane] = incl;
      s_start[wib][lane] = start - (incl - deg);     // edge index = s_start[owner] + flat index
      __syncwarp();
      for (uint32_t i = lane; i < total; i += 32) {
        uint32_t lo = 0, hi = 31;                    // smallest owner with s_end[owner] > i
        while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (s_end[wib][mid] > i) hi = mid; else lo = mid + 1; }
        bfs_visit(nxt, ctx, a, a.col[s_start[wib][lo] + i], d, n_next);
      }
      __syncwarp();
    }
    __threadfence();
    grid.sync();
    // ---- phase 2: adjacency lists of hubs, one 256-edge chunk per warp at a time
    {
      const uint64_t nch = min((uint64_t)a.max_chunks, ld_relaxed(huge_cnt));
      for (uint64_t c = gwarp; c < nch; c += nwarps) {
        const Chunk ch = a.chunks[c];
        for (uint32_t i = lane; i < ch.count; i += 32) bfs_visit(nxt, ctx, a, a.col[ch.begin + i], d, n_next);
      }
    }
    __syncwarp();
    {
      const uint64_t s = warp_sum64(n_next);
      if (lane == 0 && s) red_add_relaxed(next_cnt, s);
      n_enq += n_next;
    }
    if (tid == 0) requeue_prepare(cur);              // cur is drained and idle: it is the next level's `nxt`
    __threadfence();
    grid.sync();
    if (ld_relaxed(next_cnt) == 0) break;            // "until the next frontier is empty"
  }
  edges = warp_sum64(edges); n_deq = warp_sum64(n_deq); n_enq = warp_sum64(n_enq);
  if (lane == 0) {
    if (edges) red_add_relaxed(a.ctr + B_EDGES, edges);
    if (n_deq) red_add_relaxed(a.ctr + B_DEQ, n_deq);
    if (n_enq) red_add_relaxed(a.ctr + B_ENQ, n_enq);
  }
  if (tid == 0) {
    st_relaxed(a.ctr + B_LEVELS, level + 1);
    if (pool_exhausted(qa) || pool_exhausted(qb)) st_relaxed(a.ctr + B_ERROR, 2);
  }
}

template <class Q>
int bfs_run_t(const uint64_t* d_rowptr, const uint32_t* d_col, uint32_t nv, uint32_t src, int32_t* d_dist,
              const gq_bfs_opts& o, gq_bfs_stats* st_out, cudaStream_t stream) {
  const auto t_begin = std::chrono::steady_clock::now();
  const int sms = gq_device_sms();
  if (sms <= 0) { gq_set_error("no CUDA device"); return GQ_E_CUDA; }
  const uint32_t block = o.block_threads ? o.block_threads : 256;
  if (block % 32 || block > 512) return GQ_E_INVAL;
  int nb = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, bfs_kernel<Q>, (int)block, 0));
  if (nb <= 0) return GQ_E_CUDA;
  const uint32_t full = (uint32_t)nb * block * sms;
  uint32_t threads = o.threads ? o.threads : full;
  const uint32_t blocks = (threads + block - 1) / block;
  threads = blocks * block;                               // whole blocks: every launched thread takes part
  if (threads > full) return GQ_E_RESIDENCY;              // Thm III.10 assumption

  uint64_t ne = 0;
  CU(cudaMemcpyAsync(&ne, d_rowptr + nv, 8, cudaMemcpyDeviceToHost, stream));
  CU(cudaStreamSynchronize(stream));

  gq_opts qo{};
  qo.max_threads = threads;
  qo.flags = o.flags | GQ_F_NO_DEQ_SPIN | GQ_F_EAGER_EMPTY | GQ_F_NO_FULL_TEST;   // each vertex is enqueued at most once: never nv items;   // nothing arrives in `cur` during a level: never park
  qo.ymc_pool_cells = 0;                                  // G-WFQ-YMC: the default ring pool, pow2ceil(capacity + 4k) cells (Y10)
  OwnedQueue<Q> qa, qb;
  const uint64_t cap = pow2ceil64(std::max<uint32_t>(nv, 2));
  int rc = qa.create(cap, qo);
  if (rc == 0) rc = qb.create(cap, qo);
  if (rc) return rc;

  BfsArgs a{};
  a.rowptr = d_rowptr; a.col = d_col; a.dist = d_dist; a.nv = nv; a.src = src;
  a.huge_degree = std::max<uint32_t>(o.huge_degree ? o.huge_degree : 64u, kChunk);   // measured at scale 22: 1024 -> 3.3 ms, 256 -> 2.4 ms
  a.max_chunks = (uint32_t)std::min<uint64_t>(2 * ne / kChunk + 2, 0x7FFFFFFFu);
  char* scratch = nullptr;
  const size_t ctr_bytes = B_COUNT * 8, chunk_bytes = (size_t)a.max_chunks * sizeof(Chunk);
  CU(cudaMalloc(&scratch, ctr_bytes + chunk_bytes));
  a.ctr = reinterpret_cast<uint64_t*>(scratch);
  a.chunks = reinterpret_cast<Chunk*>(scratch + ctr_bytes);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  auto cleanup = [&]() { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); cudaFree(scratch); };
  cudaError_t e = cudaMemsetAsync(scratch, 0, ctr_bytes, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_dist, 0xFF, (size_t)nv * 4, stream);
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) e = cudaEventRecord(e0, stream);
  if (e != cudaSuccess) { cleanup(); return gq_cuda_fail(e, "bfs setup"); }
  void* args[] = {&qa.view, &qb.view, &a};
  e = cudaLaunchCooperativeKernel((void*)bfs_kernel<Q>, dim3(blocks), dim3(block), args, 0, stream);
  if (e != cudaSuccess) { cleanup(); return e == cudaErrorCooperativeLaunchTooLarge ? GQ_E_RESIDENCY : gq_cuda_fail(e, "bfs launch"); }
  cudaEventRecord(e1, stream);
  rc = gq_wait_event(e1, gq_watchdog_slack_s());
  if (rc == GQ_E_TIMEOUT) { qa.h = qb.h = nullptr; return rc; }   // kernel still running: freeing would block on it
  uint64_t c[B_COUNT] = {};
  float ms = 0;
  if (rc == 0) {
    e = cudaMemcpy(c, a.ctr, sizeof c, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e != cudaSuccess) rc = gq_cuda_fail(e, "bfs results");
  }
  cleanup();
  if (rc) return rc;
  if (c[B_ERROR] == 2) return GQ_E_POOL;
  if (c[B_ERROR]) return GQ_E_STATE;
  if (st_out) {
    gq_bfs_stats s{};
    s.levels = (uint32_t)c[B_LEVELS]; s.threads = threads; s.edges_scanned = c[B_EDGES];
    s.vertices_visited = c[B_DEQ]; s.queue_ops = c[B_DEQ] + c[B_ENQ]; s.ms = ms;
    s.total_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    *st_out = s;
  }
  return 0;
}

}  // namespace

extern "C" int bfs_run_ex(int kind, const uint64_t* d_rowptr, const uint32_t* d_col, uint32_t nv, uint32_t src,
                          int32_t* d_dist, const gq_bfs_opts* opts, gq_bfs_stats* stats_out, void* stream) {
  if (!d_rowptr || !d_col || !d_dist || nv == 0 || src >= nv) return GQ_E_INVAL;
  gq_bfs_opts o{};
  if (opts) o = *opts;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  switch (kind) {
    case GQ_LFQ: return bfs_run_t<LfqView>(d_rowptr, d_col, nv, src, d_dist, o, stats_out, st);
    case GQ_LFQ_DIRECT: return bfs_run_t<DlfqView>(d_rowptr, d_col, nv, src, d_dist, o, stats_out, st);
    case GQ_WFQ: return bfs_run_t<WfqView>(d_rowptr, d_col, nv, src, d_dist, o, stats_out, st);
    case GQ_WFQ_YMC: return bfs_run_t<YmcView>(d_rowptr, d_col, nv, src, d_dist, o, stats_out, st);
    default: return GQ_E_INVAL;
  }
}
extern "C" int bfs_run(int kind, const uint64_t* d_rowptr, const uint32_t* d_col, uint32_t nv, uint32_t src,
                       int32_t* d_dist, gq_bfs_stats* stats_out, void* stream) {
  return bfs_run_ex(kind, d_rowptr, d_col, nv, src, d_dist, nullptr, stats_out, stream);
}

// =====================================================================================  tracer
// DESIGN.md §6 states every constant and the order of every floating-point operation; this file
// is compiled with -fmad=false, so each * and + below is individually rounded (IEEE fp32), and
// sqrtf / division are the correctly rounded forms (no fast-math).
namespace {

struct V3 { float x, y, z; };
__device__ __forceinline__ V3 vadd(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V3 vsub(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V3 vmul(V3 a, V3 b) { return {a.x * b.x, a.y * b.y, a.z * b.z}; }
__device__ __forceinline__ V3 vscale(V3 a, float s) { return {a.x * s, a.y * s, a.z * s}; }
__device__ __forceinline__ V3 vdiv(V3 a, float s) { return {a.x / s, a.y / s, a.z / s}; }
__device__ __forceinline__ float vdot(V3 a, V3 b) { return (a.x * b.x + a.y * b.y) + a.z * b.z; }

__device__ __forceinline__ uint32_t fmix32(uint32_t x) {
  x ^= x >> 16; x *= 0x85ebca6bu; x ^= x >> 13; x *= 0xc2b2ae35u; x ^= x >> 16;
  return x;
}
// u(seed, pixel, sample, bounce, dim) in [0,1): 24 high bits of a three-round integer hash
__device__ __forceinline__ float rt_rnd(uint64_t seed, uint32_t pixel, uint32_t sample, uint32_t bounce, uint32_t dim) {
  uint32_t x = fmix32((uint32_t)seed ^ (pixel * 0x9E3779B1u));
  x = fmix32(x ^ (sample * 0x85EBCA77u + bounce * 0xC2B2AE3Du + dim * 0x27D4EB2Fu));
  x = fmix32(x ^ (uint32_t)(seed >> 32));
  return (float)(x >> 8) * (1.0f / 16777216.0f);
}

constexpr uint32_t kTile = 16, kTilePixels = kTile * kTile, kPerLane = kTilePixels / 32;
constexpr uint32_t kItemTileBits = 20, kItemSampleBits = 6;      // item = tile | sample << 20 | bounce << 26
constexpr uint32_t kMaxSpheres = 1024;
enum { R_PENDING = 0, R_RAYS, R_ENQ, R_DEQ, R_ERROR, R_COUNT = 8 };

struct RtArgs {
  uint32_t width, height, spp, max_bounce, ns, tiles_x, tiles_y, n_items;
  uint64_t seed;
  const float* spheres;
  float* state;          // SoA, 9 planes of n_paths floats: o.xyz, d.xyz, T.xyz
  float* radiance;       // SoA, 3 planes of n_paths floats (written once, when the path ends)
  uint8_t* alive;        // n_paths
  uint64_t n_paths;      // tiles * spp * 256
  uint64_t* ctr;
  float* rgb;
};

// One path, one bounce: camera ray (bounce 0) or the stored ray, nearest hit, shading, scatter.  Returns true iff the path
// lives on (its next ray is in a.state); a path that ends writes its radiance.  Arithmetic and its order: DESIGN.md section 6.
__device__ __forceinline__ bool rt_path_step(const RtArgs& a, const float4* s_sph0, const float4* s_sph1, uint64_t path, uint32_t px,
                                             uint32_t py, uint32_t sample, uint32_t bounce) {
  const float aspect = (float)a.width / (float)a.height;
  const uint32_t pixel = py * a.width + px;
  V3 o, d, T;
  if (bounce == 0) {                                            // primary ray: pinhole camera, DESIGN.md section 6
    const float u0 = rt_rnd(a.seed, pixel, sample, 0, 0), u1 = rt_rnd(a.seed, pixel, sample, 0, 1);
    const float sx = (((float)px + u0) / (float)a.width) * 2.0f - 1.0f;
    const float sy = 1.0f - (((float)py + u1) / (float)a.height) * 2.0f;
    d = V3{sx * (0.36397023f * aspect), sy * 0.36397023f, -1.0f};
    d = vdiv(d, sqrtf(vdot(d, d)));
    o = V3{0.0f, 0.0f, 35.0f};
    T = V3{1.0f, 1.0f, 1.0f};
  } else {
    const float* S = a.state + path;
    o = V3{S[0], S[a.n_paths], S[2 * a.n_paths]};
    d = V3{S[3 * a.n_paths], S[4 * a.n_paths], S[5 * a.n_paths]};
    T = V3{S[6 * a.n_paths], S[7 * a.n_paths], S[8 * a.n_paths]};
  }
  float best_t = __int_as_float(0x7f800000);
  int best = -1;
  for (uint32_t i = 0; i < a.ns; ++i) {                         // brute force, ties -> lowest index
    const float4 c = s_sph0[i];                                 // cx, cy, cz, r
    const V3 oc = vsub(o, V3{c.x, c.y, c.z});
    const float bq = vdot(oc, d);
    const float cq = vdot(oc, oc) - c.w * c.w;
    const float disc = bq * bq - cq;
    if (disc < 0.0f) continue;
    const float sq = sqrtf(disc);
    float t = -bq - sq;
    if (!(t > 1e-3f)) { t = -bq + sq; if (!(t > 1e-3f)) continue; }
    if (t < best_t) { best_t = t; best = (int)i; }
  }
  V3 L = {0.0f, 0.0f, 0.0f};
  bool ended = true;
  if (best < 0) {
    L = vmul(T, V3{0.7f, 0.8f, 1.0f});                           // background
  } else {
    const float4 c = s_sph0[best], m = s_sph1[best];            // m = ar, ag, ab, emissive
    const V3 albedo = {m.x, m.y, m.z};
    if (m.w != 0.0f) {
      L = vmul(T, vscale(albedo, 4.0f));                        // emissive: 4 x albedo, path ends
    } else {
      T = vmul(T, albedo);
      if (bounce != a.max_bounce) {                             // else absorbed at the depth limit
        const V3 hp = vadd(o, vscale(d, best_t));
        const V3 n = vdiv(vsub(hp, V3{c.x, c.y, c.z}), c.w);
        V3 unit = n;
        for (uint32_t k = 0; k < 16; ++k) {                     // rejection sampling in the unit ball
          const V3 v = {2.0f * rt_rnd(a.seed, pixel, sample, bounce, 2 + 3 * k) - 1.0f,
                        2.0f * rt_rnd(a.seed, pixel, sample, bounce, 3 + 3 * k) - 1.0f,
                        2.0f * rt_rnd(a.seed, pixel, sample, bounce, 4 + 3 * k) - 1.0f};
          const float l2 = vdot(v, v);
          if (l2 <= 1.0f && l2 > 1e-12f) { unit = vdiv(v, sqrtf(l2)); break; }
        }
        V3 sdir = vadd(n, unit);
        float l2 = vdot(sdir, sdir);
        if (!(l2 > 1e-12f)) { sdir = n; l2 = vdot(n, n); }
        d = vdiv(sdir, sqrtf(l2));
        o = hp;
        ended = false;
      }
    }
  }
  if (ended) {
    float* R = a.radiance + path;
    R[0] = L.x; R[a.n_paths] = L.y; R[2 * a.n_paths] = L.z;
    a.alive[path] = 0;
    return false;
  }
  float* S = a.state + path;
  S[0] = o.x; S[a.n_paths] = o.y; S[2 * a.n_paths] = o.z;
  S[3 * a.n_paths] = d.x; S[4 * a.n_paths] = d.y; S[5 * a.n_paths] = d.z;
  S[6 * a.n_paths] = T.x; S[7 * a.n_paths] = T.y; S[8 * a.n_paths] = T.z;
  a.alive[path] = 1;
  return true;
}

// Advance the (pixel, sample) paths of one item by one bounce.  Returns true iff any path lives on.
__device__ __forceinline__ bool rt_advance(const RtArgs& a, const float4* s_sph0, const float4* s_sph1, uint32_t item, uint32_t lane,
                                           uint32_t& rays) {
  const uint32_t tile = item & ((1u << kItemTileBits) - 1);
  const uint32_t sample = (item >> kItemTileBits) & ((1u << kItemSampleBits) - 1);
  const uint32_t bounce = item >> (kItemTileBits + kItemSampleBits);
  const uint32_t tx = tile % a.tiles_x, ty = tile / a.tiles_x;
  const uint64_t path0 = ((uint64_t)tile * a.spp + sample) * kTilePixels;
  bool any_alive = false;
  for (uint32_t j = 0; j < kPerLane; ++j) {
    const uint32_t p = lane + 32 * j;
    const uint32_t px = tx * kTile + (p % kTile), py = ty * kTile + (p / kTile);
    if (px >= a.width || py >= a.height) continue;
    const uint64_t path = path0 + p;
    if (bounce != 0 && !a.alive[path]) continue;
    ++rays;
    any_alive |= rt_path_step(a, s_sph0, s_sph1, path, px, py, sample, bounce);
  }
  return __any_sync(0xffffffffu, any_alive);
}

// Persistent tracing kernel: every warp repeatedly dequeues an item, advances its 256 paths by
// one bounce, and re-enqueues the item with bounce+1 while any of them lives.  `pending` counts
// the items that are queued or being processed; a warp leaves when it reads EMPTY and pending == 0.
template <class Q>
__global__ void __launch_bounds__(256) rt_kernel(Q q, RtArgs a) {
  cg::grid_group grid = cg::this_grid();
  __shared__ float4 s_sph0[kMaxSpheres];
  __shared__ float4 s_sph1[kMaxSpheres];
  for (uint32_t i = threadIdx.x; i < a.ns; i += blockDim.x) {
    const float* S = a.spheres + 8 * i;
    s_sph0[i] = make_float4(S[0], S[1], S[2], S[3]);
    s_sph1[i] = make_float4(S[4], S[5], S[6], S[7]);
  }
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
  const uint32_t nthreads = gridDim.x * blockDim.x;
  thread_ctx ctx{tid};
  ctx.help_peer = tid + 1;
  uint32_t n_enq = 0, n_deq = 0, rays = 0;
  // "Primary rays are generated and enqueued": item (tile, sample, bounce 0) for every tile and sample
  for (uint32_t i = tid; i < a.n_items; i += nthreads) {
    const uint32_t item = (i / a.spp) | ((i % a.spp) << kItemTileBits);
    if (enqueue<true, true>(q, ctx, item) != OK) st_relaxed(a.ctr + R_ERROR, 1); else ++n_enq;
  }
  __syncthreads();
  __threadfence();
  grid.sync();
  uint32_t idle_ns = 0;
  for (;;) {
    uint32_t item = 0;
    int s = EMPTY;
    if (lane == 0) s = dequeue<false, true>(q, ctx, &item);
    s = __shfl_sync(0xffffffffu, s, 0);
    if (s != OK) {
      uint32_t stop = 0;                                          // decided by lane 0 for the whole warp
      if (lane == 0) stop = ld_acquire(a.ctr + R_PENDING) == 0 || ld_relaxed(a.ctr + R_ERROR) || pool_exhausted(q);
      if (__shfl_sync(0xffffffffu, stop, 0)) break;               // "until no work remains"
      idle_ns = idle_ns ? min(idle_ns * 2, 2000u) : 100u;
      __nanosleep(idle_ns);
      continue;
    }
    idle_ns = 0;
    item = __shfl_sync(0xffffffffu, item, 0);
    if (lane == 0) ++n_deq;
    const bool more = rt_advance(a, s_sph0, s_sph1, item, lane, rays);
    __threadfence();                                              // path state visible before the item is
    __syncwarp();
    if (lane == 0) {
      if (more) {                                                 // "re-enqueues reflective bounces"
        if (enqueue<false, true>(q, ctx, item + (1u << (kItemTileBits + kItemSampleBits))) != OK) {
          st_relaxed(a.ctr + R_ERROR, 1);
          red_add_relaxed(a.ctr + R_PENDING, (uint64_t)-1ll);
        } else ++n_enq;
      } else {
        red_add_relaxed(a.ctr + R_PENDING, (uint64_t)-1ll);
      }
    }
  }
  const uint64_t r = warp_sum64(rays), e = warp_sum64(n_enq), dq = warp_sum64(n_deq);
  if (lane == 0) {
    if (r) red_add_relaxed(a.ctr + R_RAYS, r);
    if (e) red_add_relaxed(a.ctr + R_ENQ, e);
    if (dq) red_add_relaxed(a.ctr + R_DEQ, dq);
  }
  if (tid == 0 && pool_exhausted(q)) st_relaxed(a.ctr + R_ERROR, 2);
}

// pixel = (sum over samples, in sample order) / spp
__global__ void rt_resolve_kernel(RtArgs a) {
  const uint32_t pixel = blockIdx.x * blockDim.x + threadIdx.x;
  if (pixel >= a.width * a.height) return;
  const uint32_t px = pixel % a.width, py = pixel / a.width;
  const uint32_t tile = (py / kTile) * a.tiles_x + px / kTile, p = (py % kTile) * kTile + px % kTile;
  V3 acc = {0.0f, 0.0f, 0.0f};
  for (uint32_t s = 0; s < a.spp; ++s) {
    const float* R = a.radiance + ((uint64_t)tile * a.spp + s) * kTilePixels + p;
    acc = vadd(acc, V3{R[0], R[a.n_paths], R[2 * a.n_paths]});
  }
  const V3 c = vdiv(acc, (float)a.spp);
  a.rgb[3 * (size_t)pixel + 0] = c.x; a.rgb[3 * (size_t)pixel + 1] = c.y; a.rgb[3 * (size_t)pixel + 2] = c.z;
}

template <class Q>
int rt_render_t(const gq_rt_scene& sc, float* d_rgb, gq_rt_stats* st_out, cudaStream_t stream) {
  const auto t_begin = std::chrono::steady_clock::now();
  const int sms = gq_device_sms();
  if (sms <= 0) { gq_set_error("no CUDA device"); return GQ_E_CUDA; }
  RtArgs a{};
  a.width = sc.width; a.height = sc.height; a.spp = sc.spp; a.max_bounce = sc.max_bounce; a.ns = sc.n_spheres;
  a.seed = sc.seed; a.spheres = sc.d_spheres; a.rgb = d_rgb;
  a.tiles_x = (sc.width + kTile - 1) / kTile; a.tiles_y = (sc.height + kTile - 1) / kTile;
  const uint64_t tiles = (uint64_t)a.tiles_x * a.tiles_y;
  if (tiles >= (1u << kItemTileBits) || sc.spp == 0 || sc.spp >= (1u << kItemSampleBits) || sc.max_bounce >= 60 ||
      sc.n_spheres > kMaxSpheres || (sc.n_spheres && !sc.d_spheres) || (uint64_t)sc.width * sc.height >= (1ull << 31))
    return GQ_E_INVAL;
  a.n_items = (uint32_t)(tiles * sc.spp);
  a.n_paths = (uint64_t)a.n_items * kTilePixels;
  const uint32_t block = 256;
  int nb = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, rt_kernel<Q>, (int)block, 0));
  if (nb <= 0) return GQ_E_CUDA;
  const uint32_t full = (uint32_t)nb * block * sms;
  uint32_t threads = sc.threads ? sc.threads : full;
  const uint32_t blocks = (threads + block - 1) / block;
  threads = blocks * block;
  if (threads > full) return GQ_E_RESIDENCY;

  gq_opts qo{};
  qo.max_threads = threads;
  qo.park_ns = 20000;                                     // a warp waits on its slot only for an item whose enqueuer is in flight
  qo.flags = GQ_F_EAGER_EMPTY | GQ_F_NO_FULL_TEST;        // idle warps poll: EMPTY at once when Tail <= Head; never more than n_items items
  qo.ymc_pool_cells = 0;                                  // G-WFQ-YMC: the default ring pool, pow2ceil(capacity + 4k) cells, stays L2-resident (Y10)
  OwnedQueue<Q> q;
  int rc = q.create(pow2ceil64(std::max<uint32_t>(a.n_items, 2)), qo);
  if (rc) return rc;

  char* scratch = nullptr;
  const size_t ctr_bytes = 256, state_bytes = (size_t)a.n_paths * 9 * 4, rad_bytes = (size_t)a.n_paths * 3 * 4;
  CU(cudaMalloc(&scratch, ctr_bytes + state_bytes + rad_bytes + a.n_paths));
  a.ctr = reinterpret_cast<uint64_t*>(scratch);
  a.state = reinterpret_cast<float*>(scratch + ctr_bytes);
  a.radiance = reinterpret_cast<float*>(scratch + ctr_bytes + state_bytes);
  a.alive = reinterpret_cast<uint8_t*>(scratch + ctr_bytes + state_bytes + rad_bytes);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  auto cleanup = [&]() { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); cudaFree(scratch); };
  uint64_t init[R_COUNT] = {};
  init[R_PENDING] = a.n_items;
  cudaError_t e = cudaMemcpyAsync(a.ctr, init, sizeof init, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(a.radiance, 0, rad_bytes, stream);
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) e = cudaEventRecord(e0, stream);
  if (e != cudaSuccess) { cleanup(); return gq_cuda_fail(e, "rt setup"); }
  void* args[] = {&q.view, &a};
  e = cudaLaunchCooperativeKernel((void*)rt_kernel<Q>, dim3(blocks), dim3(block), args, 0, stream);
  if (e != cudaSuccess) { cleanup(); return e == cudaErrorCooperativeLaunchTooLarge ? GQ_E_RESIDENCY : gq_cuda_fail(e, "rt launch"); }
  const uint32_t npix = sc.width * sc.height;
  rt_resolve_kernel<<<(npix + 255) / 256, 256, 0, stream>>>(a);
  cudaEventRecord(e1, stream);
  rc = gq_wait_event(e1, gq_watchdog_slack_s());
  if (rc == GQ_E_TIMEOUT) { q.h = nullptr; return rc; }           // kernel still running: freeing would block on it
  uint64_t c[R_COUNT] = {};
  float ms = 0;
  if (rc == 0) {
    e = cudaMemcpy(c, a.ctr, sizeof c, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e != cudaSuccess) rc = gq_cuda_fail(e, "rt results");
  }
  cleanup();
  if (rc) return rc;
  if (c[R_ERROR] == 2) return GQ_E_POOL;
  if (c[R_ERROR]) return GQ_E_STATE;
  if (st_out) {
    gq_rt_stats s{};
    s.rays = c[R_RAYS]; s.queue_ops = c[R_ENQ] + c[R_DEQ]; s.ms = ms; s.threads = threads; s.items = a.n_items;
    s.total_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    *st_out = s;
  }
  return 0;
}

// ---- mode 1: one queue per tile, items are rays ("each tile owns its own queue") ---------------------------------
// Block b owns the tiles b, b + gridDim.x, ...  All of its warps serve those queues: in every round a warp looks at four
// consecutive tiles of the block's list, 8 lanes per tile, so that the lanes converged at one enqueue / dequeue name up to four
// different queues (kUniform = false: WAVEFAA elects one leader per queue inside the converged warp).  A lane that receives
// a ray advances that path by one bounce and puts the next ray into the queue of the same tile.  s_pending counts the rays
// of the block that are queued or in flight; the block is done when it reaches 0.  No grid-wide synchronisation.
constexpr uint32_t kRayPixelBits = 8, kRaySampleBits = 6;
template <class Q>
__global__ void __launch_bounds__(256) rt_tiles_kernel(const Q* __restrict__ views, RtArgs a) {
  __shared__ float4 s_sph0[kMaxSpheres];
  __shared__ float4 s_sph1[kMaxSpheres];
  __shared__ unsigned long long s_pending;
  __shared__ uint32_t s_error;
  for (uint32_t i = threadIdx.x; i < a.ns; i += blockDim.x) {
    const float* S = a.spheres + 8 * i;
    s_sph0[i] = make_float4(S[0], S[1], S[2], S[3]);
    s_sph1[i] = make_float4(S[4], S[5], S[6], S[7]);
  }
  if (threadIdx.x == 0) { s_pending = 0; s_error = 0; }
  __syncthreads();
  const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  const uint32_t n_tiles = a.tiles_x * a.tiles_y;
  const uint32_t my_tiles = blockIdx.x < n_tiles ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;   // tiles b, b + grid, ...
  thread_ctx ctx{threadIdx.x};                                       // every tile queue is created for blockDim.x threads
  uint32_t rays = 0, n_enq = 0, n_deq = 0;
  // "Primary rays are generated and enqueued": (pixel, sample, bounce 0) of every tile the block owns
  for (uint32_t i = threadIdx.x; i < my_tiles * a.spp * kTilePixels; i += blockDim.x) {
    const uint32_t k = i / (a.spp * kTilePixels), r = i % (a.spp * kTilePixels), sample = r / kTilePixels, p = r % kTilePixels;
    const uint32_t tile = blockIdx.x + k * gridDim.x;
    const uint32_t px = (tile % a.tiles_x) * kTile + p % kTile, py = (tile / a.tiles_x) * kTile + p / kTile;
    if (px >= a.width || py >= a.height) continue;
    atomicAdd(&s_pending, 1ull);
    if (enqueue<false, 1>(views[tile], ctx, p | sample << kRayPixelBits) != OK) { s_error = 1; atomicAdd(&s_pending, ~0ull); } else ++n_enq;
  }
  __threadfence();
  __syncthreads();
  for (uint32_t round = wib; my_tiles != 0; round += nwarps) {
    if (*reinterpret_cast<volatile unsigned long long*>(&s_pending) == 0 || *reinterpret_cast<volatile uint32_t*>(&s_error)) break;
    const uint32_t k = (round * 4 + (lane >> 3)) % my_tiles;         // four tiles per warp and round, 8 lanes each
    const uint32_t tile = blockIdx.x + k * gridDim.x;
    const Q& q = views[tile];
    uint32_t item = 0;
    if (dequeue<false, 1>(q, ctx, &item) != OK) continue;
    ++n_deq;
    const uint32_t p = item & ((1u << kRayPixelBits) - 1), sample = (item >> kRayPixelBits) & ((1u << kRaySampleBits) - 1);
    const uint32_t bounce = item >> (kRayPixelBits + kRaySampleBits);
    const uint32_t px = (tile % a.tiles_x) * kTile + p % kTile, py = (tile / a.tiles_x) * kTile + p / kTile;
    const uint64_t path = ((uint64_t)tile * a.spp + sample) * kTilePixels + p;
    ++rays;
    if (rt_path_step(a, s_sph0, s_sph1, path, px, py, sample, bounce)) {
      __threadfence();                                               // the path's next ray is visible before its item (queue.cuh, G15)
      if (enqueue<false, 1>(q, ctx, item + (1u << (kRayPixelBits + kRaySampleBits))) != OK) { s_error = 1; atomicAdd(&s_pending, ~0ull); } else ++n_enq;
    } else {
      atomicAdd(&s_pending, ~0ull);
    }
  }
  __syncwarp();
  const uint64_t r = warp_sum64(rays), e = warp_sum64(n_enq), dq = warp_sum64(n_deq);
  if (lane == 0) {
    if (r) red_add_relaxed(a.ctr + R_RAYS, r);
    if (e) red_add_relaxed(a.ctr + R_ENQ, e);
    if (dq) red_add_relaxed(a.ctr + R_DEQ, dq);
  }
  if (threadIdx.x == 0 && s_error) st_relaxed(a.ctr + R_ERROR, 1);
}

template <class Q>
int rt_render_tiles_t(const gq_rt_scene& sc, float* d_rgb, gq_rt_stats* st_out, cudaStream_t stream) {
  const auto t_begin = std::chrono::steady_clock::now();
  const int sms = gq_device_sms();
  if (sms <= 0) { gq_set_error("no CUDA device"); return GQ_E_CUDA; }
  RtArgs a{};
  a.width = sc.width; a.height = sc.height; a.spp = sc.spp; a.max_bounce = sc.max_bounce; a.ns = sc.n_spheres;
  a.seed = sc.seed; a.spheres = sc.d_spheres; a.rgb = d_rgb;
  a.tiles_x = (sc.width + kTile - 1) / kTile; a.tiles_y = (sc.height + kTile - 1) / kTile;
  const uint64_t tiles = (uint64_t)a.tiles_x * a.tiles_y;
  if (tiles >= (1u << kItemTileBits) || sc.spp == 0 || sc.spp >= (1u << kRaySampleBits) || sc.max_bounce >= 60 ||
      sc.n_spheres > kMaxSpheres || (sc.n_spheres && !sc.d_spheres) || (uint64_t)sc.width * sc.height >= (1ull << 31))
    return GQ_E_INVAL;
  a.n_items = (uint32_t)(tiles * sc.spp);
  a.n_paths = (uint64_t)a.n_items * kTilePixels;
  const uint32_t block = 256;
  int nb = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, rt_tiles_kernel<Q>, (int)block, 0));
  if (nb <= 0) return GQ_E_CUDA;
  uint32_t blocks = (uint32_t)nb * sms;
  if (sc.threads) blocks = std::min(blocks, std::max(1u, sc.threads / block));
  blocks = (uint32_t)std::min<uint64_t>(blocks, tiles);

  gq_opts qo{};
  qo.max_threads = block;                                 // a tile queue is served by the threads of one block
  qo.park_ns = 20000;
  qo.flags = GQ_F_EAGER_EMPTY | GQ_F_NO_FULL_TEST;        // polling consumers; a tile never holds more than 256 x spp rays
  std::vector<gq_queue*> qs(tiles);
  void* qblock = nullptr;
  int rc = gq_create_many(ViewOf<Q>::kind, pow2ceil64((uint64_t)kTilePixels * sc.spp), &qo, (uint32_t)tiles, qs.data(), &qblock, stream);
  if (rc) return rc;
  std::vector<Q> h_views(tiles);
  for (uint64_t i = 0; i < tiles && rc == 0; ++i) rc = queue_device_view(qs[i], &h_views[i], sizeof(Q));

  char* scratch = nullptr;
  const size_t ctr_bytes = 256, state_bytes = (size_t)a.n_paths * 9 * 4, rad_bytes = (size_t)a.n_paths * 3 * 4;
  const size_t alive_bytes = (a.n_paths + 255) / 256 * 256, view_bytes = tiles * sizeof(Q);
  cudaError_t e = rc ? cudaSuccess : cudaMalloc(&scratch, ctr_bytes + state_bytes + rad_bytes + alive_bytes + view_bytes);
  if (rc || e != cudaSuccess) { gq_destroy_many(qs.data(), (uint32_t)tiles, qblock); return rc ? rc : gq_cuda_fail(e, "cudaMalloc(rt)"); }
  a.ctr = reinterpret_cast<uint64_t*>(scratch);
  a.state = reinterpret_cast<float*>(scratch + ctr_bytes);
  a.radiance = reinterpret_cast<float*>(scratch + ctr_bytes + state_bytes);
  a.alive = reinterpret_cast<uint8_t*>(scratch + ctr_bytes + state_bytes + rad_bytes);
  Q* d_views = reinterpret_cast<Q*>(scratch + ctr_bytes + state_bytes + rad_bytes + alive_bytes);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  auto cleanup = [&]() { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); cudaFree(scratch); gq_destroy_many(qs.data(), (uint32_t)tiles, qblock); };
  e = cudaMemsetAsync(a.ctr, 0, ctr_bytes, stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_views, h_views.data(), view_bytes, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(a.radiance, 0, rad_bytes, stream);
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) e = cudaEventRecord(e0, stream);
  if (e != cudaSuccess) { cleanup(); return gq_cuda_fail(e, "rt setup"); }
  rt_tiles_kernel<Q><<<blocks, block, 0, stream>>>(d_views, a);
  e = cudaGetLastError();
  if (e != cudaSuccess) { cleanup(); return gq_cuda_fail(e, "rt launch"); }
  const uint32_t npix = sc.width * sc.height;
  rt_resolve_kernel<<<(npix + 255) / 256, 256, 0, stream>>>(a);
  cudaEventRecord(e1, stream);
  rc = gq_wait_event(e1, gq_watchdog_slack_s());
  if (rc == GQ_E_TIMEOUT) return rc;                      // kernel still running: freeing would block on it
  uint64_t c[R_COUNT] = {};
  float ms = 0;
  if (rc == 0) {
    e = cudaMemcpy(c, a.ctr, sizeof c, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e != cudaSuccess) rc = gq_cuda_fail(e, "rt results");
  }
  cleanup();
  if (rc) return rc;
  if (c[R_ERROR]) return GQ_E_STATE;
  if (st_out) {
    gq_rt_stats s{};
    s.rays = c[R_RAYS]; s.queue_ops = c[R_ENQ] + c[R_DEQ]; s.ms = ms; s.threads = blocks * block; s.items = (uint32_t)tiles;
    s.total_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    *st_out = s;
  }
  return 0;
}

}  // namespace

extern "C" int rt_render_ex(int kind, const gq_rt_scene* scene, float* d_rgb, const gq_rt_opts* opts, gq_rt_stats* stats_out, void* stream) {
  if (!opts || opts->mode == 0) return rt_render(kind, scene, d_rgb, stats_out, stream);
  if (!scene || !d_rgb || scene->width == 0 || scene->height == 0 || opts->mode != 1 || opts->reserved) return GQ_E_INVAL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  switch (kind) {
    case GQ_LFQ: return rt_render_tiles_t<LfqView>(*scene, d_rgb, stats_out, st);
    case GQ_LFQ_DIRECT: return rt_render_tiles_t<DlfqView>(*scene, d_rgb, stats_out, st);
    default: return GQ_E_INVAL;                            // per-thread records x thousands of queues: see gq.h
  }
}

extern "C" int rt_render(int kind, const gq_rt_scene* scene, float* d_rgb, gq_rt_stats* stats_out, void* stream) {
  if (!scene || !d_rgb || scene->width == 0 || scene->height == 0) return GQ_E_INVAL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  switch (kind) {
    case GQ_LFQ: return rt_render_t<LfqView>(*scene, d_rgb, stats_out, st);
    case GQ_LFQ_DIRECT: return rt_render_t<DlfqView>(*scene, d_rgb, stats_out, st);
    case GQ_WFQ: return rt_render_t<WfqView>(*scene, d_rgb, stats_out, st);
    case GQ_WFQ_YMC: return rt_render_t<YmcView>(*scene, d_rgb, stats_out, st);
    default: return GQ_E_INVAL;
  }
}
