// capi.cu — host side of libgq.so: handle management, memory layout in HBM, kernel launches.
// Every entry point is declared and documented in include/gq.h.
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <thread>
#include <vector>

#include "gq.h"
#include "host_util.h"
#include "kernels.cuh"

using namespace gq;
using namespace gq::detail;
using namespace gqk;

// ------------------------------------------------------------------------------- errors
static thread_local char g_err[256] = "";
int gq_cuda_fail(cudaError_t e, const char* what) {
  std::snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
  return e == cudaErrorMemoryAllocation ? GQ_E_NOMEM : GQ_E_CUDA;
}
void gq_set_error(const char* text) { std::snprintf(g_err, sizeof g_err, "%s", text); }
static int cuda_fail(cudaError_t e, const char* what) { return gq_cuda_fail(e, what); }

extern "C" const char* gq_last_cuda_error(void) { return g_err; }
extern "C" const char* gq_version(void) { return "gq 0.1 (sm_100a)"; }

static_assert(sizeof(gq_opts) == 64 && sizeof(gq_run_cfg) == 80 && sizeof(gq_run_result) == 144 && sizeof(gq_hist_rec) == 40,
              "ABI structs: the Python binding mirrors these layouts");

// ------------------------------------------------------------------------------- handle
struct gq_queue {
  int kind = 0;
  uint64_t capacity = 0;   // n
  uint64_t N = 0;          // ring parameter (reading G1)
  gq_opts opts{};
  uint32_t max_threads = 0;
  char* base = nullptr;    // device block
  size_t bytes = 0;
  bool owns = false;
  LfqView lfq{};
  DlfqView dlfq{};
  WfqView wfq{};
  YmcView ymc{};
  uint64_t* d_ctr = nullptr;        // C_COUNT result counters
  gq_hist_rec* d_hist = nullptr;
  uint64_t hist_cap = 0, hist_n = 0;
  bool formatted = false;
  bool fresh = false;      // formatted and not operated on since: the fast path cannot fail (queue_prefill)
};

static int g_sms = 0;
static int device_sms();
int gq_device_sms() { return device_sms(); }
static int device_sms() {
  if (!g_sms) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  return g_sms;
}
static uint64_t pow2ceil(uint64_t x) { uint64_t p = 1; while (p < x) p <<= 1; return p; }
static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ------------------------------------------------------------------------------- layout
// One device block per queue:
//   [ hot words, one per 1 KiB ][ AQ entries ][ FQ entries ][ Data ][ kind-specific ... ]
// hot words (Head, Tail, Threshold of each ring) are kHotStride bytes apart; GQ_HOT_STRIDE overrides it for the
// layout ablation (multiple of 128)
static size_t hot_stride_init() {
  const char* e = std::getenv("GQ_HOT_STRIDE");
  const long v = e ? std::atol(e) : 0;
  return (v >= 128 && v % 128 == 0 && v <= (1 << 20)) ? (size_t)v : 1024;
}
static const size_t kHotStride = hot_stride_init();
struct Layout {
  uint64_t N = 0;
  uint32_t order = 0, slot_shift = 0;
  size_t off_hot = 0, off_aq = 0, off_fq = 0, off_data = 0, off_owner_aq = 0, off_owner_fq = 0, off_rec = 0, off_rec_fq = 0, off_pool = 0;
  size_t total = 0;
  uint64_t pool_cells = 0;
  uint32_t park_ns = 0, park_nap = 0, prefetch_dist = 0, spin_ns = 0;
};

template <class Q> static int max_blocks_per_sm(int block_threads);

static uint32_t default_max_threads(int kind);

static int compute_layout(int kind, uint64_t capacity, const gq_opts* o, Layout* L, uint32_t* max_threads_out) {
  if (kind < GQ_LFQ || kind > GQ_LFQ_DIRECT || capacity < 1) return GQ_E_INVAL;
  gq_opts z{}; if (!o) o = &z;
  if (o->layout > 2) return GQ_E_INVAL;
  uint32_t k = o->max_threads ? o->max_threads : default_max_threads(kind);
  if (k == 0) k = 148 * 2048;                         // no device visible: size for a full B200
  *max_threads_out = k;
  L->park_ns = o->park_ns ? o->park_ns : 250000u;
  L->park_nap = o->park_nap_ns ? (o->park_nap_ns < 32u ? 0u : o->park_nap_ns) : 128u;
  L->spin_ns = o->park_spin_ns == GQ_PARK_SPIN_NONE ? 0u : (o->park_spin_ns ? o->park_spin_ns : 2000u);
  L->prefetch_dist = (o->flags & GQ_F_NO_CELL_PREFETCH) ? 0u : k;
  size_t off = 0;
  L->off_hot = off; off += 16 * kHotStride;
  if (kind == GQ_LFQ_DIRECT) {                        // one ring, payload in the entry word: no FQ, no Data
    if (capacity >= (1ull << 31)) return GQ_E_INVAL;
    L->N = pow2ceil(std::max<uint64_t>(capacity, k));
    L->order = 0; while ((1ull << L->order) < 2 * L->N) ++L->order;
    L->slot_shift = o->layout == 0 ? 0 : (o->layout == 1 ? 2 : 4);
    L->off_aq = off; off += (size_t)(2 * L->N) * (8u << L->slot_shift);
  } else if (kind == GQ_LFQ || kind == GQ_WFQ) {
    const uint64_t idx_limit = kind == GQ_LFQ ? 0xFFFFFFFEull : 0x1FFFFFFEull;   // G-WFQ: bit 29 of the Index field marks fast-path installs
    if (capacity >= idx_limit) return GQ_E_INVAL;
    if (kind == GQ_WFQ && k >= WfqFmt::kThrNull) return GQ_E_INVAL;
    L->N = pow2ceil(std::max<uint64_t>(capacity, k));
    L->order = 0; while ((1ull << L->order) < 2 * L->N) ++L->order;
    L->slot_shift = o->layout == 0 ? 0 : (o->layout == 1 ? 2 : 4);
    const size_t ring_bytes = (size_t)(2 * L->N) * (8u << L->slot_shift);
    L->off_aq = off; off += ring_bytes;
    L->off_fq = off; off += ring_bytes;
    // 8 B payload cells (ticket tag + value; D6)
    L->off_data = off; off += align_up((size_t)capacity * 8, 256);
    if (kind == GQ_WFQ) {
      L->off_owner_aq = off; off += (size_t)(2 * L->N) * 8;
      L->off_owner_fq = off; off += (size_t)(2 * L->N) * 8;
      L->off_rec = off; off += (size_t)k * sizeof(WfqRecord);
      L->off_rec_fq = off; off += (size_t)k * sizeof(WfqRecord);
    }
  } else {
    // the pool is a ring of P cells (Y10): P = pow2ceil(max(capacity + 4k, ymc_pool_cells)); FULL from P - 2k tickets on
    if (k + 2 > Ymc::kIdTop || o->ymc_pool_cells >= (1ull << 40)) return GQ_E_INVAL;
    L->pool_cells = pow2ceil(std::max<uint64_t>(std::max<uint64_t>(capacity + 4ull * k, o->ymc_pool_cells), 64));
    L->N = pow2ceil(k);
    L->off_rec = off; off += (size_t)k * sizeof(YmcHandle);
    L->off_pool = off; off += (size_t)L->pool_cells * sizeof(YmcCell);
  }
  L->total = align_up(off, 256);
  return 0;
}

extern "C" size_t queue_storage_bytes(int kind, uint64_t capacity, const gq_opts* opts) {
  Layout L; uint32_t k;
  if (compute_layout(kind, capacity, opts, &L, &k) != 0) return 0;
  return L.total;
}

// ------------------------------------------------------------------------------- format
// Initial states (reading G4).  empty ring: Head = Tail = 2N, entries <0,1,bot>, Threshold = -1.
// ring pre-loaded with indices 0..count-1: Tail = 2N+count, slot i<count = <1,1,i>, Threshold = 3N-1.
template <class F>
__global__ void format_ring_kernel(RingView r, uint64_t slots, uint64_t count) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < slots) {
    uint64_t* sp = r.entry + ((size_t)i << r.slot_shift);
    *sp = i < count ? F::installed(F::initial(), 1u, (uint32_t)i) : F::initial();
    if (r.owner) r.owner[i] = 0;
  }
  if (i == 0) {
    const uint64_t low = F::kCtrShift ? ((1ull << F::kCtrShift) - 1) : 0;   // ThrIdx = NULL
    *r.head = (slots << F::kCtrShift) | low;
    *r.tail = ((slots + count) << F::kCtrShift) | low;
    *r.threshold = count ? r.thr_reset : -1;
  }
}

static RingView make_ring(char* base, const Layout& L, size_t off_entries, size_t off_owner, int hot_slot, size_t off_rec = 0) {
  RingView r{};
  r.entry = reinterpret_cast<uint64_t*>(base + off_entries);
  r.head = reinterpret_cast<uint64_t*>(base + L.off_hot + (hot_slot + 0) * kHotStride);
  r.tail = reinterpret_cast<uint64_t*>(base + L.off_hot + (hot_slot + 1) * kHotStride);
  r.threshold = reinterpret_cast<int64_t*>(base + L.off_hot + (hot_slot + 2) * kHotStride);
  r.owner = off_owner ? reinterpret_cast<uint64_t*>(base + off_owner) : nullptr;
  r.rec = off_rec ? base + off_rec : nullptr;
  r.thr_reset = (int64_t)(3 * L.N - 1);
  r.order = L.order;
  r.slot_shift = L.slot_shift;
  r.park_ns = L.park_ns;
  r.park_nap = L.park_nap;
  r.park_limit = (uint32_t)std::min<uint64_t>(L.N / 2, 0x7FFFFFFFu);
  // rings of 32 MiB and more (BFS frontier queues) do not stay in L2 next to the graph: prefetch k tickets ahead
  const size_t ring_bytes = (size_t)(2 * L.N) * (8u << L.slot_shift);
  r.prefetch = ring_bytes >= (32u << 20) ? L.prefetch_dist : 0;
  r.id = hot_slot ? 1u : 0u;
  r.spin_ns = L.spin_ns;
  return r;
}

// G-WFQ per-thread records: everything zero, sequence pairs apart (seq1 = 1, seq2 = 0) so that no
// helper accepts an unpublished record.
__global__ void format_wfq_records_kernel(WfqRecord* rec, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  WfqRecord z{};
  z.seq1 = 1; z.p2_seq1 = 1;
  rec[i] = z;
}

// G-WFQ-YMC: handles with no request published, helping pointers at the next thread (reading Y6).
__global__ void format_ymc_handles_kernel(YmcHandle* h, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  YmcHandle z{};
  z.enq_help_id = Ymc::kNoId;
  z.enq_peer = z.deq_peer = i + 1 < n ? i + 1 : 0;
  h[i] = z;
}
// T = H = 0 (all cells zero = <epoch 0, bot, bot_e, bot_d>, no payload tag)
__global__ void format_ymc_words_kernel(YmcView q) { *q.tail = 0; *q.head = 0; *q.exhausted = 0; }

static int format_queue(gq_queue* q, cudaStream_t st) {
  if (q->kind == GQ_WFQ_YMC) {
    const uint64_t dirty = q->ymc.pool_cells;
    CU(cudaMemsetAsync(q->ymc.pool, 0, (size_t)dirty * sizeof(YmcCell), st));
    format_ymc_handles_kernel<<<(q->max_threads + 255) / 256, 256, 0, st>>>(q->ymc.handles, q->max_threads);
    format_ymc_words_kernel<<<1, 1, 0, st>>>(q->ymc);
    CU(cudaGetLastError());
    q->formatted = true;
    return 0;
  }
  const uint64_t slots = 2 * q->N;
  const unsigned blk = 256, grd = (unsigned)((slots + blk - 1) / blk);
  if (q->kind == GQ_LFQ_DIRECT) {
    format_ring_kernel<DirFmt><<<grd, blk, 0, st>>>(q->dlfq.r, slots, 0);
  } else if (q->kind == GQ_LFQ) {
    format_ring_kernel<LfqFmt><<<grd, blk, 0, st>>>(q->lfq.aq, slots, 0);
    format_ring_kernel<LfqFmt><<<grd, blk, 0, st>>>(q->lfq.fq, slots, q->capacity);
    CU(cudaMemsetAsync(q->lfq.data, 0, (size_t)q->capacity * 8, st));      // no payload cell carries a live ticket tag (D6)
  } else if (q->kind == GQ_WFQ) {
    format_ring_kernel<WfqFmt><<<grd, blk, 0, st>>>(q->wfq.aq, slots, 0);
    format_ring_kernel<WfqFmt><<<grd, blk, 0, st>>>(q->wfq.fq, slots, q->capacity);
    CU(cudaMemsetAsync(q->wfq.data, 0, (size_t)q->capacity * 8, st));
    const unsigned g2 = (q->max_threads + blk - 1) / blk;
    format_wfq_records_kernel<<<g2, blk, 0, st>>>(static_cast<WfqRecord*>(q->wfq.aq.rec), q->max_threads);
    format_wfq_records_kernel<<<g2, blk, 0, st>>>(static_cast<WfqRecord*>(q->wfq.fq.rec), q->max_threads);
  } else {
    return GQ_E_INVAL;
  }
  CU(cudaGetLastError());
  return 0;
}

// ------------------------------------------------------------------------------- occupancy
template <class Q>
static int max_blocks_per_sm(int block_threads) {
  int nb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, bench_kernel<Q, false, 1>, block_threads, 0) != cudaSuccess) return 0;
  return nb;
}
static int kind_blocks_per_sm(int kind, int block_threads) {
  switch (kind) {
    case GQ_LFQ: return max_blocks_per_sm<LfqView>(block_threads);
    case GQ_WFQ: return max_blocks_per_sm<WfqView>(block_threads);
    case GQ_WFQ_YMC: return max_blocks_per_sm<YmcView>(block_threads);
    case GQ_LFQ_DIRECT: return max_blocks_per_sm<DlfqView>(block_threads);
    default: return 0;
  }
}
static uint32_t default_max_threads(int kind) {
  const int sms = device_sms();
  if (sms <= 0) return 0;
  return (uint32_t)(kind_blocks_per_sm(kind, 256) * 256 * sms);
}

extern "C" int queue_max_coresident_threads(int kind, int block_threads, uint32_t* out) {
  if (!out || kind < GQ_LFQ || kind > GQ_LFQ_DIRECT) return GQ_E_INVAL;
  if (block_threads <= 0) block_threads = 256;
  if (block_threads % 32 || block_threads > 512) return GQ_E_INVAL;
  const int sms = device_sms();
  if (sms <= 0) { std::snprintf(g_err, sizeof g_err, "no CUDA device"); return GQ_E_CUDA; }
  const int nb = kind_blocks_per_sm(kind, block_threads);
  if (nb <= 0) return GQ_E_CUDA;
  *out = (uint32_t)(nb * block_threads * sms);
  return 0;
}

// ------------------------------------------------------------------------------- create / destroy
extern "C" int queue_create_ex(int kind, uint64_t capacity, const gq_opts* opts, gq_queue** out) {
  if (!out) return GQ_E_INVAL;
  if (device_sms() <= 0) { std::snprintf(g_err, sizeof g_err, "no CUDA device"); return GQ_E_CUDA; }
  Layout L; uint32_t k = 0;
  int rc = compute_layout(kind, capacity, opts, &L, &k);
  if (rc) return rc;
  gq_queue* q = new (std::nothrow) gq_queue();
  if (!q) return GQ_E_NOMEM;
  q->kind = kind; q->capacity = capacity; q->N = L.N; q->max_threads = k;
  if (opts) q->opts = *opts;
  q->opts.flags &= kPublicFlags;        // internal flag bits (ring.cuh) cannot be set from outside
  q->bytes = L.total;
  if (opts && opts->storage) {
    if (opts->storage_bytes < L.total || (reinterpret_cast<uintptr_t>(opts->storage) & 255)) { delete q; return GQ_E_INVAL; }
    q->base = static_cast<char*>(opts->storage);
  } else {
    cudaError_t e = cudaMalloc(&q->base, L.total);
    if (e != cudaSuccess) { delete q; return cuda_fail(e, "cudaMalloc(queue)"); }
    q->owns = true;
  }
  cudaError_t e = cudaMalloc(&q->d_ctr, 2 * C_COUNT * sizeof(uint64_t));   // run counters + scratch of collect_stats
  if (e != cudaSuccess) { if (q->owns) cudaFree(q->base); delete q; return cuda_fail(e, "cudaMalloc(counters)"); }
  if (kind == GQ_LFQ_DIRECT) {
    q->dlfq.r = make_ring(q->base, L, L.off_aq, 0, 0);
    q->dlfq.capacity = (uint32_t)capacity;
    q->dlfq.flags = q->opts.flags;
  } else if (kind == GQ_LFQ) {
    q->lfq.aq = make_ring(q->base, L, L.off_aq, 0, 0);
    q->lfq.fq = make_ring(q->base, L, L.off_fq, 0, 3);
    q->lfq.data = reinterpret_cast<uint64_t*>(q->base + L.off_data);
    q->lfq.capacity = (uint32_t)capacity;
    q->lfq.flags = q->opts.flags;
  } else if (kind == GQ_WFQ) {
    q->wfq.aq = make_ring(q->base, L, L.off_aq, L.off_owner_aq, 0, L.off_rec);
    q->wfq.fq = make_ring(q->base, L, L.off_fq, L.off_owner_fq, 3, L.off_rec_fq);
    q->wfq.data = reinterpret_cast<uint64_t*>(q->base + L.off_data);
    q->wfq.capacity = (uint32_t)capacity;
    q->wfq.nthreads = k;
    auto pat = [](uint32_t v, uint32_t dflt) { return v == GQ_PATIENCE_ZERO ? 0u : (v ? v : dflt); };
    q->wfq.enq_patience = pat(q->opts.enq_patience, 64);      // reading W2
    q->wfq.deq_patience = pat(q->opts.deq_patience, 64);
    q->wfq.help_delay = q->opts.help_delay ? q->opts.help_delay : 64;   // D = 64
    q->wfq.flags = q->opts.flags;
  } else {
    auto pat = [](uint32_t v, uint32_t dflt) { return v == GQ_PATIENCE_ZERO ? 0u : (v ? v : dflt); };
    q->ymc.pool = reinterpret_cast<YmcCell*>(q->base + L.off_pool);
    q->ymc.pool_cells = L.pool_cells;
    q->ymc.head = reinterpret_cast<uint64_t*>(q->base + L.off_hot + 0 * kHotStride);
    q->ymc.tail = reinterpret_cast<uint64_t*>(q->base + L.off_hot + 1 * kHotStride);
    q->ymc.exhausted = reinterpret_cast<uint64_t*>(q->base + L.off_hot + 2 * kHotStride);
    q->ymc.handles = reinterpret_cast<YmcHandle*>(q->base + L.off_rec);
    q->ymc.nthreads = k;
    q->ymc.enq_patience = pat(q->opts.enq_patience, 10);      // reading Y8
    q->ymc.deq_patience = pat(q->opts.deq_patience, 10);
    q->ymc.help_delay = q->opts.help_delay ? q->opts.help_delay : 1;   // [5]: after every successful dequeue
    q->ymc.flags = q->opts.flags;
    q->ymc.park_ns = L.park_ns;
    q->ymc.park_nap = L.park_nap;
    q->ymc.park_limit = (uint32_t)std::min<uint64_t>(L.N / 2, 0x7FFFFFFFu);
    q->ymc.pool_shift = 0; while ((1ull << q->ymc.pool_shift) < L.pool_cells) ++q->ymc.pool_shift;
    q->ymc.full_limit = L.pool_cells - 2ull * k;
  }
  rc = format_queue(q, nullptr);
  q->fresh = rc == 0;
  if (rc == 0) { cudaError_t e2 = cudaDeviceSynchronize(); if (e2 != cudaSuccess) rc = cuda_fail(e2, "format"); }
  if (rc) { queue_destroy(q); return rc; }
  *out = q;
  return 0;
}
extern "C" int queue_create(int kind, uint64_t capacity, gq_queue** out) { return queue_create_ex(kind, capacity, nullptr, out); }

// `count` queues of the same shape in ONE device block, formatted on `stream` with one synchronisation at the end (the
// per-tile queues of the multi-queue tracer: thousands of small queues).  G-LFQ / G-LFQ-D only: the kinds with
// per-thread records would need count x max_threads of them.  Handles carry no run counters (no run_* on them).
int gq_create_many(int kind, uint64_t capacity, const gq_opts* opts, uint32_t count, gq_queue** out, void** block_out, cudaStream_t st) {
  if (!out || !block_out || count == 0 || (kind != GQ_LFQ && kind != GQ_LFQ_DIRECT) || (opts && opts->storage)) return GQ_E_INVAL;
  Layout L; uint32_t k = 0;
  int rc = compute_layout(kind, capacity, opts, &L, &k);
  if (rc) return rc;
  char* block = nullptr;
  CU(cudaMalloc(&block, L.total * count));
  for (uint32_t i = 0; i < count; ++i) out[i] = nullptr;
  for (uint32_t i = 0; i < count && rc == 0; ++i) {
    gq_queue* q = new (std::nothrow) gq_queue();
    if (!q) { rc = GQ_E_NOMEM; break; }
    out[i] = q;
    q->kind = kind; q->capacity = capacity; q->N = L.N; q->max_threads = k; q->bytes = L.total;
    if (opts) q->opts = *opts;
    q->opts.flags &= kPublicFlags;
    q->base = block + (size_t)i * L.total;
    if (kind == GQ_LFQ_DIRECT) {
      q->dlfq.r = make_ring(q->base, L, L.off_aq, 0, 0);
      q->dlfq.capacity = (uint32_t)capacity; q->dlfq.flags = q->opts.flags;
    } else {
      q->lfq.aq = make_ring(q->base, L, L.off_aq, 0, 0);
      q->lfq.fq = make_ring(q->base, L, L.off_fq, 0, 3);
      q->lfq.data = reinterpret_cast<uint64_t*>(q->base + L.off_data);
      q->lfq.capacity = (uint32_t)capacity; q->lfq.flags = q->opts.flags;
    }
    rc = format_queue(q, st);
  }
  if (rc == 0) { cudaError_t e = cudaStreamSynchronize(st); if (e != cudaSuccess) rc = cuda_fail(e, "format"); }
  if (rc) { for (uint32_t i = 0; i < count; ++i) delete out[i]; cudaFree(block); return rc; }
  *block_out = block;
  return 0;
}
void gq_destroy_many(gq_queue** qs, uint32_t count, void* block) {
  for (uint32_t i = 0; i < count; ++i) delete qs[i];
  if (block) cudaFree(block);
}

extern "C" int queue_destroy(gq_queue* q) {
  if (!q) return GQ_E_INVAL;
  if (q->owns && q->base) cudaFree(q->base);
  if (q->d_ctr) cudaFree(q->d_ctr);
  if (q->d_hist) cudaFree(q->d_hist);
  delete q;
  return 0;
}

extern "C" int queue_reset(gq_queue* q, void* stream) {
  if (!q) return GQ_E_INVAL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int rc = format_queue(q, st);
  if (rc) return rc;
  CU(cudaStreamSynchronize(st));
  q->fresh = true;
  return 0;
}

extern "C" int queue_kind(const gq_queue* q) { return q ? q->kind : GQ_E_INVAL; }

__global__ void wfq_rounds_kernel(const WfqRecord* a, uint32_t n, uint64_t* out4) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  uint64_t v[4] = {0, 0, 0, 0};
  if (i < n) { v[0] = a[i].n_tail_inc; v[1] = a[i].n_tail_clr; v[2] = a[i].n_head_inc; v[3] = a[i].n_head_clr; }
  for (int k = 0; k < 4; ++k) { const uint64_t s = warp_sum(v[k]); if ((threadIdx.x & 31) == 0 && s) red_add_relaxed(out4 + k, s); }
}
// Quiescent read-back of the hot words (Lemma III.7 tests, diagnostics): ticket counters decoded from their packed form.
extern "C" int queue_debug_counters(gq_queue* q, uint64_t* out8 /* 16 words */) {
  if (!q || !out8) return GQ_E_INVAL;
  CU(cudaDeviceSynchronize());
  std::memset(out8, 0, 16 * sizeof(uint64_t));
  auto rd = [](const void* p, uint64_t* v) { return cudaMemcpy(v, p, 8, cudaMemcpyDeviceToHost); };
  auto ring = [&](const RingView& r, int shift, uint64_t* o) -> cudaError_t {
    cudaError_t e = rd(r.head, o); if (e == cudaSuccess) e = rd(r.tail, o + 1); if (e == cudaSuccess) e = rd(r.threshold, o + 2);
    o[0] >>= shift; o[1] >>= shift;
    return e;
  };
  cudaError_t e = cudaSuccess;
  if (q->kind == GQ_LFQ) { e = ring(q->lfq.aq, 0, out8); if (e == cudaSuccess) e = ring(q->lfq.fq, 0, out8 + 3); }
  else if (q->kind == GQ_WFQ) { e = ring(q->wfq.aq, WfqFmt::kCtrShift, out8); if (e == cudaSuccess) e = ring(q->wfq.fq, WfqFmt::kCtrShift, out8 + 3); }
  else if (q->kind == GQ_LFQ_DIRECT) e = ring(q->dlfq.r, 0, out8);
  else { e = rd(q->ymc.head, out8); if (e == cudaSuccess) e = rd(q->ymc.tail, out8 + 1); }
  out8[6] = q->N; out8[7] = q->max_threads;
  if (e == cudaSuccess && q->kind == GQ_WFQ) {          // slow-path rounds since the last reset (Lemma III.7)
    uint64_t* d = nullptr;
    CU(cudaMalloc(&d, 64));
    cudaMemset(d, 0, 64);
    const unsigned g = (q->max_threads + 255) / 256;
    wfq_rounds_kernel<<<g, 256>>>(static_cast<const WfqRecord*>(q->wfq.aq.rec), q->max_threads, d);
    wfq_rounds_kernel<<<g, 256>>>(static_cast<const WfqRecord*>(q->wfq.fq.rec), q->max_threads, d + 4);
    e = cudaMemcpy(out8 + 8, d, 64, cudaMemcpyDeviceToHost);
    cudaFree(d);
  }
  return e == cudaSuccess ? 0 : cuda_fail(e, "queue_debug_counters");
}

extern "C" int queue_device_view(const gq_queue* q, void* view_out, size_t view_bytes) {
  if (!q || !view_out) return GQ_E_INVAL;
  const void* src = nullptr; size_t n = 0;
  switch (q->kind) {
    case GQ_LFQ: src = &q->lfq; n = sizeof(LfqView); break;
    case GQ_LFQ_DIRECT: src = &q->dlfq; n = sizeof(DlfqView); break;
    case GQ_WFQ: src = &q->wfq; n = sizeof(WfqView); break;
    default: src = &q->ymc; n = sizeof(YmcView); break;
  }
  if (view_bytes < n) return GQ_E_INVAL;
  std::memcpy(view_out, src, n);
  return 0;
}

// ------------------------------------------------------------------------------- kind dispatch
template <class Fn>
static int dispatch(gq_queue* q, Fn&& fn) {
  switch (q->kind) {
    case GQ_LFQ: return fn(q->lfq);
    case GQ_WFQ: return fn(q->wfq);
    case GQ_WFQ_YMC: return fn(q->ymc);
    case GQ_LFQ_DIRECT: return fn(q->dlfq);
    default: return GQ_E_INVAL;
  }
}
static void set_nthreads(LfqView&, uint32_t) {}
static void set_nthreads(DlfqView&, uint32_t) {}
static void set_nthreads(WfqView& v, uint32_t n) {
  v.nthreads = n;
  v.aq.slow_nap = v.fq.slow_nap = std::min(std::max(n, 1024u), 65536u);   // about 1 ns per thread that can lose a SLOWFAA round
}
static void set_nthreads(YmcView& v, uint32_t n) { v.nthreads = n; }

// slow-path statistics live in the per-thread records; sum and clear them after a run
__global__ void wfq_stats_kernel(WfqRecord* a, WfqRecord* b, uint32_t n, uint64_t* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  uint64_t se = 0, sd = 0, hp = 0;
  if (i < n) {
    se = a[i].n_slow_enq + b[i].n_slow_enq; sd = a[i].n_slow_deq + b[i].n_slow_deq; hp = a[i].n_helps + b[i].n_helps;
    a[i].n_slow_enq = a[i].n_slow_deq = a[i].n_helps = 0;
    b[i].n_slow_enq = b[i].n_slow_deq = b[i].n_helps = 0;
  }
  se = warp_sum(se); sd = warp_sum(sd); hp = warp_sum(hp);
  if ((threadIdx.x & 31) == 0) { if (se) red_add_relaxed(out, se); if (sd) red_add_relaxed(out + 1, sd); if (hp) red_add_relaxed(out + 2, hp); }
}
__global__ void ymc_stats_kernel(YmcHandle* a, uint32_t n, uint64_t* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  uint64_t se = 0, sd = 0, hp = 0;
  if (i < n) {
    se = a[i].n_slow_enq; sd = a[i].n_slow_deq; hp = a[i].n_helps;
    a[i].n_slow_enq = a[i].n_slow_deq = a[i].n_helps = 0;
  }
  se = warp_sum(se); sd = warp_sum(sd); hp = warp_sum(hp);
  if ((threadIdx.x & 31) == 0) { if (se) red_add_relaxed(out, se); if (sd) red_add_relaxed(out + 1, sd); if (hp) red_add_relaxed(out + 2, hp); }
}
static int collect_stats(gq_queue* q, gq_run_result* res) {
  if (q->kind == GQ_LFQ || q->kind == GQ_LFQ_DIRECT) return 0;
  uint64_t* d = q->d_ctr + C_COUNT; uint64_t h[4] = {0, 0, 0, 0};
  CU(cudaMemset(d, 0, 32));
  if (q->kind == GQ_WFQ)
    wfq_stats_kernel<<<(q->max_threads + 255) / 256, 256>>>(static_cast<WfqRecord*>(q->wfq.aq.rec), static_cast<WfqRecord*>(q->wfq.fq.rec), q->max_threads, d);
  else {
    ymc_stats_kernel<<<(q->max_threads + 255) / 256, 256>>>(q->ymc.handles, q->max_threads, d);
    cudaMemcpyAsync(d + 3, q->ymc.exhausted, 8, cudaMemcpyDeviceToDevice);
  }
  cudaError_t e = cudaMemcpy(h, d, 32, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess && h[3]) res->pool_exhausted = 1;
  if (e != cudaSuccess) return cuda_fail(e, "stats");
  res->slow_enq = h[0]; res->slow_deq = h[1]; res->helps = h[2];
  return 0;
}

// ------------------------------------------------------------------------------- launches
// Wait for `ev` with a host-side watchdog so that a livelocked kernel fails a call instead of
// hanging it (SURVEY §5 "failure detection").
static double watchdog_slack_s();
static int wait_event(cudaEvent_t ev, double budget_s);
double gq_watchdog_slack_s() { return watchdog_slack_s(); }
int gq_wait_event(cudaEvent_t ev, double budget_s) { return wait_event(ev, budget_s); }
static double watchdog_slack_s() {
  const char* e = std::getenv("GQ_WATCHDOG_S");     // seconds granted on top of warmup + duration (default 60)
  const double v = e ? std::atof(e) : 0.0;
  return v > 0 ? v : 60.0;
}
static int wait_event(cudaEvent_t ev, double budget_s) {
  const auto t0 = std::chrono::steady_clock::now();
  for (;;) {
    cudaError_t e = cudaEventQuery(ev);
    if (e == cudaSuccess) return 0;
    if (e != cudaErrorNotReady) return cuda_fail(e, "kernel");
    if (std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count() > budget_s) {
      std::snprintf(g_err, sizeof g_err, "watchdog: kernel still running after %.0f s", budget_s);
      return GQ_E_TIMEOUT;
    }
    std::this_thread::sleep_for(std::chrono::microseconds(200));
  }
}

// Events and scratch of one launch, released on every path out of the caller.  After a watchdog time-out the kernel is
// still running and cudaFree / cudaEventDestroy would block on it: `abandon()` leaves them to the (stuck) context.
struct LaunchRes {
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  void* scratch = nullptr;
  bool abandoned = false;
  int create() { CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1)); return 0; }
  void abandon() { abandoned = true; }
  ~LaunchRes() {
    if (abandoned) return;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (scratch) cudaFree(scratch);
  }
};

struct Resolved { uint32_t threads, block, blocks, blocks_per_sm; };
static int resolve_launch(int blocks_per_sm, const gq_run_cfg* cfg, uint32_t thread_cap, Resolved* r) {
  const int sms = device_sms();
  if (sms <= 0) { std::snprintf(g_err, sizeof g_err, "no CUDA device"); return GQ_E_CUDA; }
  r->block = cfg->block_threads ? cfg->block_threads : 256;
  if (r->block % 32 || r->block > 512) return GQ_E_INVAL;
  if (blocks_per_sm <= 0) return GQ_E_CUDA;
  const uint32_t full = (uint32_t)blocks_per_sm * r->block * sms;
  r->threads = cfg->threads ? cfg->threads : std::min(full, thread_cap);
  if (r->threads > thread_cap) return GQ_E_INVAL;
  r->blocks = (r->threads + r->block - 1) / r->block;
  r->blocks_per_sm = (uint32_t)blocks_per_sm;
  if (r->blocks > (uint32_t)blocks_per_sm * sms) return GQ_E_RESIDENCY;   // Thm III.10 assumption
  return 0;
}

static BenchParams make_params(const gq_run_cfg* cfg, const Resolved& r, int mode) {
  BenchParams p{};
  p.threads = r.threads; p.mode = (uint32_t)mode;
  p.warmup_ns = (uint64_t)(cfg->warmup_ms * 1e6); p.duration_ns = (uint64_t)(cfg->duration_ms * 1e6);
  double pf = cfg->producer_fraction; if (pf < 0) pf = 0; if (pf > 1) pf = 1;
  p.prod_threshold = (uint64_t)(pf * 4294967296.0);
  p.seed = (uint32_t)cfg->seed; p.ops_per_thread = cfg->ops_per_thread;
  p.jitter_ns = cfg->jitter_ns; p.fail_backoff_ns = cfg->fail_backoff_ns; p.value_base = cfg->value_base;
  p.converged = cfg->converged;
  p.block_faa = cfg->block_faa; p.funnel_window_ns = cfg->funnel_window_ns;
  // history runs small enough for it use the payload encoding of BASELINE.json configs[0]: thread << 16 | iteration
  p.tid_shift = (cfg->record_history && r.threads <= 65536 && cfg->ops_per_thread <= 65536) ? 16u : 0u;
  return p;
}

static int finish_run(uint64_t* d_ctr, cudaEvent_t e0, cudaEvent_t e1, const gq_run_cfg* cfg, const Resolved& r, gq_run_result* res) {
  uint64_t c[C_COUNT];
  CU(cudaMemcpy(c, d_ctr, sizeof c, cudaMemcpyDeviceToHost));
  float ms = 0; CU(cudaEventElapsedTime(&ms, e0, e1));
  std::memset(res, 0, sizeof *res);
  res->succ_enq = c[C_SUCC_ENQ]; res->succ_deq = c[C_SUCC_DEQ]; res->full = c[C_FULL]; res->empty = c[C_EMPTY];
  res->tot_enq = c[C_TOT_ENQ]; res->tot_deq = c[C_TOT_DEQ]; res->tot_full = c[C_TOT_FULL]; res->tot_empty = c[C_TOT_EMPTY];
  res->sum_enq = c[C_SUM_ENQ]; res->sum_deq = c[C_SUM_DEQ]; res->retries = c[C_RETRIES];
  res->kernel_ms = ms;
  res->meas_seconds = cfg->ops_per_thread ? (double)(c[C_T_END] - c[C_T0]) * 1e-9 : cfg->duration_ms * 1e-3;
  res->threads_launched = r.threads; res->blocks = r.blocks; res->blocks_per_sm = r.blocks_per_sm;
  res->pool_exhausted = (uint32_t)(c[C_POOL] != 0);
  return 0;
}

// ---- debug / fault-injection builds (include/gq/detail/debug.cuh); in the product build these return GQ_E_INVAL
extern "C" int gq_dbg_sites(unsigned long long* out80) {
#ifdef GQ_DBG_SITES
  if (!out80) return GQ_E_INVAL;
  CU(cudaMemcpyFromSymbol(out80, gq::detail::g_dbg, 80 * 8));
  unsigned long long z[80] = {0};
  CU(cudaMemcpyToSymbol(gq::detail::g_dbg, z, sizeof z));
  return 0;
#else
  (void)out80; return GQ_E_INVAL;
#endif
}
extern "C" int gq_dbg_trace(void* out, uint64_t max_records, uint64_t* n_out) {
#ifdef GQ_DBG_SITES
  if (!out || !n_out) return GQ_E_INVAL;
  unsigned long long n = 0, zero = 0;
  CU(cudaMemcpyFromSymbol(&n, gq::detail::g_trace_n, 8));
  n = std::min<unsigned long long>(std::min<unsigned long long>(n, gq::detail::kTraceCap), max_records);
  if (n) CU(cudaMemcpyFromSymbol(out, gq::detail::g_trace, n * sizeof(gq::detail::TraceRec)));
  CU(cudaMemcpyToSymbol(gq::detail::g_trace_n, &zero, 8));
  *n_out = n;
  return 0;
#else
  (void)out; (void)max_records; (void)n_out; return GQ_E_INVAL;
#endif
}
extern "C" int gq_set_mutation(uint32_t id) {
#ifdef GQ_MUTANTS
  if (id >= gq::detail::MUT_COUNT) return GQ_E_INVAL;
  CU(cudaMemcpyToSymbol(gq::detail::g_mutation, &id, 4));
  return 0;
#else
  (void)id; return GQ_E_INVAL;
#endif
}
static void report_stuck() {
#ifdef GQ_DEBUG_STUCK
  unsigned long long h[2 + 16 * 6];
  if (cudaMemcpyFromSymbol(h, gq::detail::g_stuck, sizeof h) != cudaSuccess) return;
  if (!h[0]) return;
  std::fprintf(stderr, "[gq] livelock detector fired: %llu records\n", h[1]);
  for (unsigned i = 0; i < 16 && i < h[1]; ++i) {
    const unsigned long long* r = h + 2 + 6 * i;
    std::fprintf(stderr, "[gq]  loc=%#llx n=%llu tid=%llu a=%#llx b=%#llx c=%#llx d=%#llx\n", r[0] & 0xffffffffull, r[0] >> 32, r[1], r[2], r[3], r[4], r[5]);
  }
  std::memset(h, 0, sizeof h);
  cudaMemcpyToSymbol(gq::detail::g_stuck, h, sizeof h);
#endif
}

template <class Q>
static int run_bench_t(gq_queue* q, const Q& view, const gq_run_cfg* cfg, int mode, gq_run_result* res) {
  const bool per_lane = (q->opts.flags & GQ_F_PER_LANE_FAA) != 0;
  const bool hist = cfg->record_history != 0;
  if (hist && cfg->ops_per_thread == 0) return GQ_E_INVAL;
  if (!hist && cfg->ops_per_thread == 0 && cfg->duration_ms <= 0) return GQ_E_INVAL;
  const bool fused = mode == MODE_SPLIT && cfg->role_layout >= 2 && cfg->role_layout <= 4;       // mixed warps, one converged call (G-LFQ)
  if (fused && (q->kind != GQ_LFQ || per_lane)) return GQ_E_INVAL;
  if (hist && per_lane) return GQ_E_INVAL;                              // the per-thread-FAA ablation is a timing variant only
  const bool funnel = cfg->block_faa != 0;                              // block-level ticket funnels (D11): a kernel variant of its own
  if (funnel && (per_lane || fused)) return GQ_E_INVAL;
  void* fn = hist ? (void*)bench_kernel<Q, true, 1> : (per_lane ? (void*)bench_kernel<Q, false, 0> : (void*)bench_kernel<Q, false, 1>);
  if (funnel) fn = hist ? (void*)bench_kernel<Q, true, 2> : (void*)bench_kernel<Q, false, 2>;
  if constexpr (HasFused<Q>::value) {
    if (fused) fn = hist ? (void*)bench_kernel<Q, true, 1, true> : (void*)bench_kernel<Q, false, 1, true>;
  }
  Resolved r;
  int nb = 0;
  const uint32_t blk = cfg->block_threads ? cfg->block_threads : 256;
  if (blk % 32 || blk > 512) return GQ_E_INVAL;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, (int)blk, 0));
  int rc = resolve_launch(nb, cfg, q->max_threads, &r);
  if (rc) return rc;
  if (hist) {
    const uint64_t need = (uint64_t)r.threads * cfg->ops_per_thread * (mode == MODE_SPLIT ? 1 : 2);
    if (need > q->hist_cap) {
      if (q->d_hist) cudaFree(q->d_hist);
      q->d_hist = nullptr; q->hist_cap = 0;
      CU(cudaMalloc(&q->d_hist, need * sizeof(gq_hist_rec)));
      q->hist_cap = need;
    }
    q->hist_n = need;
  }
  CU(cudaMemset(q->d_ctr, 0, C_COUNT * sizeof(uint64_t)));
  BenchParams p = make_params(cfg, r, mode);
  Q v = view;
  set_nthreads(v, r.threads);          // help ring = the launched threads (reading W7)
  LaunchRes lr;
  if (mode == MODE_SPLIT && (cfg->role_layout == 1 || cfg->role_layout == 3)) {   // same seeded roles, producers first: homogeneous warps
    std::vector<uint32_t> perm; perm.reserve(r.threads);
    std::vector<uint32_t> cons; cons.reserve(r.threads);
    for (uint32_t t = 0; t < r.threads; ++t)
      ((uint64_t)gq::detail::mix32(p.seed * 0x9e3779b9u + t) < p.prod_threshold ? perm : cons).push_back(t);
    perm.insert(perm.end(), cons.begin(), cons.end());
    CU(cudaMalloc(&lr.scratch, (size_t)r.threads * 4));
    CU(cudaMemcpy(lr.scratch, perm.data(), (size_t)r.threads * 4, cudaMemcpyHostToDevice));
    p.perm = static_cast<const uint32_t*>(lr.scratch);
    if (cfg->role_layout == 3) p.fused = 1;          // homogeneous warps through the fused operation (diagnostic)
  } else if (mode == MODE_SPLIT && (cfg->role_layout == 2 || cfg->role_layout == 4)) {
    p.fused = cfg->role_layout == 2 ? 1 : 2;           // 2: enqueue_or_dequeue_step (waits handed back), 4: the blocking enqueue_or_dequeue
  } else if (cfg->role_layout != 0 && mode == MODE_SPLIT) {
    return GQ_E_INVAL;
  }
  uint64_t* ctr = q->d_ctr; gq_hist_rec* h = q->d_hist;
  void* args[] = {&v, &p, &ctr, &h};
  rc = lr.create();
  if (rc) return rc;
  CU(cudaEventRecord(lr.e0, nullptr));
  cudaError_t le = cudaLaunchCooperativeKernel(fn, dim3(r.blocks), dim3(r.block), args, 0, nullptr);
  if (le != cudaSuccess) return le == cudaErrorCooperativeLaunchTooLarge ? GQ_E_RESIDENCY : cuda_fail(le, "launch");
  CU(cudaEventRecord(lr.e1, nullptr));
  rc = wait_event(lr.e1, (cfg->warmup_ms + cfg->duration_ms) * 1e-3 + watchdog_slack_s());
  if (rc == GQ_E_TIMEOUT) { lr.abandon(); return rc; }
  if (rc == 0) rc = finish_run(q->d_ctr, lr.e0, lr.e1, cfg, r, res);
  if (rc == 0) report_stuck();
  if (rc == 0) rc = collect_stats(q, res);
  if (rc == 0 && res->pool_exhausted) return GQ_E_POOL;
  return rc;
}

static int run_bench(gq_queue* q, const gq_run_cfg* cfg, int mode, gq_run_result* res) {
  if (!q || !cfg || !res) return GQ_E_INVAL;
  q->fresh = false;
  return dispatch(q, [&](auto& view) { return run_bench_t(q, view, cfg, mode, res); });
}
extern "C" int run_balanced(gq_queue* q, const gq_run_cfg* cfg, gq_run_result* res) { return run_bench(q, cfg, MODE_BALANCED, res); }
extern "C" int run_split(gq_queue* q, const gq_run_cfg* cfg, gq_run_result* res) { return run_bench(q, cfg, MODE_SPLIT, res); }

// ------------------------------------------------------------------------------- ceilings
template <class K, class... A>
static int run_ceiling(K kernel, const gq_run_cfg* cfg, gq_run_result* res, uint64_t* d_ctr, void** args) {
  int nb = 0;
  const uint32_t blk = cfg->block_threads ? cfg->block_threads : 256;
  if (blk % 32 || blk > 512) return GQ_E_INVAL;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, (int)blk, 0));
  Resolved r;
  int rc = resolve_launch(nb, cfg, 0xFFFFFFFFu, &r);
  if (rc) return rc;
  BenchParams p = make_params(cfg, r, MODE_BALANCED);
  args[2] = &p;
  LaunchRes lr;
  rc = lr.create();
  if (rc) return rc;
  CU(cudaEventRecord(lr.e0, nullptr));
  cudaError_t le = cudaLaunchCooperativeKernel((void*)kernel, dim3(r.blocks), dim3(r.block), args, 0, nullptr);
  if (le != cudaSuccess) return cuda_fail(le, "launch");
  CU(cudaEventRecord(lr.e1, nullptr));
  rc = wait_event(lr.e1, (cfg->warmup_ms + cfg->duration_ms) * 1e-3 + watchdog_slack_s());
  if (rc == GQ_E_TIMEOUT) { lr.abandon(); return rc; }
  if (rc == 0) rc = finish_run(d_ctr, lr.e0, lr.e1, cfg, r, res);
  return rc;
}

extern "C" int run_faa_ceiling(const gq_run_cfg* cfg, uint32_t n_counters, gq_run_result* res) {
  const bool per_lane = (n_counters & GQ_CEILING_PER_LANE) != 0;
  n_counters &= ~(uint32_t)GQ_CEILING_PER_LANE;
  if (!cfg || !res || n_counters < 1 || n_counters > 8) return GQ_E_INVAL;
  if (cfg->ops_per_thread == 0 && cfg->duration_ms <= 0) return GQ_E_INVAL;
  uint64_t *d_counters = nullptr, *d_ctr = nullptr;
  CU(cudaMalloc(&d_counters, 8 * 1024));
  cudaError_t e = cudaMalloc(&d_ctr, C_COUNT * 8);
  if (e != cudaSuccess) { cudaFree(d_counters); return cuda_fail(e, "cudaMalloc"); }
  cudaMemset(d_counters, 0, 8 * 1024); cudaMemset(d_ctr, 0, C_COUNT * 8);
  void* args[4] = {&d_counters, &n_counters, nullptr, &d_ctr};
  int rc = per_lane ? run_ceiling(faa_ceiling_kernel<false>, cfg, res, d_ctr, args)
                    : run_ceiling(faa_ceiling_kernel<true>, cfg, res, d_ctr, args);
  if (rc != GQ_E_TIMEOUT) { cudaFree(d_counters); cudaFree(d_ctr); }
  return rc;
}

extern "C" int run_slot_atomic_ceiling(const gq_run_cfg* cfg, uint64_t slots, gq_run_result* res) {
  if (!cfg || !res || slots < 32) return GQ_E_INVAL;
  if (cfg->ops_per_thread == 0 && cfg->duration_ms <= 0) return GQ_E_INVAL;
  uint64_t *d_buf = nullptr, *d_ctr = nullptr;
  CU(cudaMalloc(&d_buf, slots * 8));
  cudaError_t e = cudaMalloc(&d_ctr, C_COUNT * 8);
  if (e != cudaSuccess) { cudaFree(d_buf); return cuda_fail(e, "cudaMalloc"); }
  cudaMemset(d_buf, 0, slots * 8); cudaMemset(d_ctr, 0, C_COUNT * 8);
  void* args[4] = {&d_buf, &slots, nullptr, &d_ctr};
  int rc = run_ceiling(slot_ceiling_kernel, cfg, res, d_ctr, args);
  if (rc != GQ_E_TIMEOUT) { cudaFree(d_buf); cudaFree(d_ctr); }
  return rc;
}

static int faa_probe(uint32_t threads, uint32_t rounds, uint64_t seed, uint32_t funnel_mode, uint32_t window_ns,
                     uint64_t* tickets_out, uint64_t* final_counter, uint64_t* sum_out) {
  if (!threads || !rounds || !final_counter) return GQ_E_INVAL;
  if (device_sms() <= 0) { std::snprintf(g_err, sizeof g_err, "no CUDA device"); return GQ_E_CUDA; }
  uint64_t *d_c = nullptr, *d_t = nullptr;
  const size_t n = (size_t)threads * rounds;
  CU(cudaMalloc(&d_c, 32));
  cudaError_t e = tickets_out ? cudaMalloc(&d_t, n * 8) : cudaSuccess;
  if (e != cudaSuccess) { cudaFree(d_c); return cuda_fail(e, "cudaMalloc"); }
  cudaMemset(d_c, 0, 32);
  LaunchRes lr;
  int rc = lr.create();
  if (rc == 0) {
    warp_faa_probe_kernel<<<(threads + 255) / 256, 256>>>(d_c, threads, rounds, (uint32_t)seed, d_t, funnel_mode, window_ns,
                                                          reinterpret_cast<unsigned long long*>(d_c + 1));
    cudaEventRecord(lr.e1, nullptr);
    rc = wait_event(lr.e1, watchdog_slack_s());
  }
  if (rc == GQ_E_TIMEOUT) { lr.abandon(); return rc; }
  uint64_t h[3] = {0, 0, 0};
  if (rc == 0) {
    e = cudaMemcpy(h, d_c, 24, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && tickets_out) e = cudaMemcpy(tickets_out, d_t, n * 8, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) rc = cuda_fail(e, "warp_faa_probe");
  }
  cudaFree(d_c); if (d_t) cudaFree(d_t);
  if (rc) return rc;
  *final_counter = h[0];
  if (sum_out) { sum_out[0] = h[1]; sum_out[1] = h[2]; }
  return 0;
}
extern "C" int run_warp_faa_probe(uint32_t threads, uint32_t rounds, uint64_t seed, uint64_t* tickets_out, uint64_t* final_counter) {
  if (!tickets_out) return GQ_E_INVAL;
  return faa_probe(threads, rounds, seed, 0, 0, tickets_out, final_counter, nullptr);
}
extern "C" int run_funnel_probe(uint32_t threads, uint32_t rounds, uint64_t seed, uint32_t funnel_window_ns, uint64_t* tickets_out,
                                uint64_t* final_counter, uint64_t* sum_count_out) {
  return faa_probe(threads, rounds, seed, 1, funnel_window_ns, tickets_out, final_counter, sum_count_out);
}

// ------------------------------------------------------------------------------- prefill / drain / script / history
template <class Q>
static int prefill_t(const Q& view, const uint32_t* host_vals, uint64_t count, cudaStream_t st, uint32_t serial, uint32_t lanes) {
  uint32_t* d_vals = nullptr; uint64_t* d_n = nullptr;
  CU(cudaMalloc(&d_vals, std::max<uint64_t>(count, 1) * 4));
  cudaError_t e = cudaMalloc(&d_n, 8);
  if (e != cudaSuccess) { cudaFree(d_vals); return cuda_fail(e, "cudaMalloc"); }
  uint64_t n_ok = 0;
  e = cudaMemcpyAsync(d_vals, host_vals, count * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) { prefill_kernel<Q><<<1, 32, 0, st>>>(view, d_vals, count, d_n, serial, lanes); e = cudaGetLastError(); }
  if (e == cudaSuccess) e = cudaMemcpyAsync(&n_ok, d_n, 8, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_vals); cudaFree(d_n);
  if (e != cudaSuccess) return cuda_fail(e, "prefill");
  return n_ok == count ? 0 : GQ_E_STATE;
}
extern "C" int queue_prefill(gq_queue* q, const uint32_t* host_vals, uint64_t count, void* stream) {
  if (!q || (!host_vals && count)) return GQ_E_INVAL;
  if (count == 0) return 0;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // Lanes enqueue side by side only where ticket order is certain to be lane order: a freshly
  // formatted queue on its fast path.  Anywhere else (holes left by abandoned tickets after a
  // concurrent run, all-slow builds) the lanes take turns.
  const uint32_t serial = !q->fresh || (q->kind != GQ_LFQ && q->kind != GQ_LFQ_DIRECT && q->opts.enq_patience == GQ_PATIENCE_ZERO);
  q->fresh = false;
  const uint32_t lanes = std::min(32u, q->max_threads);
  return dispatch(q, [&](auto& view) { return prefill_t(view, host_vals, count, st, serial, lanes); });
}

template <class Q>
static int drain_t(const Q& view, uint32_t* host_out, uint64_t max, uint64_t* n_out, cudaStream_t st, uint32_t lanes) {
  uint32_t* d_out = nullptr; uint64_t* d_n = nullptr;
  CU(cudaMalloc(&d_out, std::max<uint64_t>(max, 1) * 4));
  cudaError_t e = cudaMalloc(&d_n, 8);
  if (e != cudaSuccess) { cudaFree(d_out); return cuda_fail(e, "cudaMalloc"); }
  uint64_t n = 0;
  drain_kernel<Q><<<1, 32, 0, st>>>(view, d_out, max, d_n, lanes);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(&n, d_n, 8, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e == cudaSuccess && n) e = cudaMemcpy(host_out, d_out, n * 4, cudaMemcpyDeviceToHost);
  cudaFree(d_out); cudaFree(d_n);
  if (e != cudaSuccess) return cuda_fail(e, "drain");
  *n_out = n;
  return 0;
}
extern "C" int queue_drain(gq_queue* q, uint32_t* host_out, uint64_t max, uint64_t* n_out, void* stream) {
  if (!q || !n_out || (!host_out && max)) return GQ_E_INVAL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  q->fresh = false;
  const uint32_t lanes = std::min(32u, q->max_threads);
  return dispatch(q, [&](auto& view) { return drain_t(view, host_out, max, n_out, st, lanes); });
}

// ---- queue_drain_noalloc: the same drain for callers that must not allocate (gq.h) ------------------------------------
// The staging memory of queue_drain (item count + items) in a file-scope device array instead of two cudaMalloc'ed blocks.
// Every device that loads libgq.so holds these 256 B + 256 KiB until the process exits.  In HOST code the name
// g_drain_scratch is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress, once per
// device, with that device current.  All calls share the array (it keeps the last call's contents; the count word is
// cleared before each launch): calls that overlap on one GPU race.
static __device__ __align__(256) unsigned char g_drain_scratch[256 + (size_t)GQ_DRAIN_NOALLOC_MAX * 4];
static int drain_scratch_address(unsigned char** out) {
  constexpr int kMaxDevices = 64;
  static unsigned char* addr[kMaxDevices] = {};
  int dev = 0;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { gq_set_error("queue_drain_noalloc: device index beyond 63"); return GQ_E_INVAL; }
  if (!addr[dev]) {
    void* p = nullptr;
    CU(cudaGetSymbolAddress(&p, g_drain_scratch));       // resolves against the current device
    addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = addr[dev];
  return 0;
}
template <class Q>
static int drain_noalloc_t(const Q& view, unsigned char* scratch, uint32_t* host_out, uint64_t max, uint64_t* n_out, cudaStream_t st, uint32_t lanes) {
  uint64_t* d_n = reinterpret_cast<uint64_t*>(scratch);
  uint32_t* d_out = reinterpret_cast<uint32_t*>(scratch + 256);
  uint64_t n = 0;
  CU(cudaMemsetAsync(d_n, 0, 8, st));                    // the array keeps the last call's contents
  drain_kernel<Q><<<1, 32, 0, st>>>(view, d_out, max, d_n, lanes);
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(&n, d_n, 8, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  if (n > max) { gq_set_error("queue_drain_noalloc: count beyond max"); return GQ_E_STATE; }
  if (n) CU(cudaMemcpy(host_out, d_out, n * 4, cudaMemcpyDeviceToHost));
  *n_out = n;
  return 0;
}
extern "C" int queue_drain_noalloc(gq_queue* q, uint32_t* host_out, uint64_t max, uint64_t* n_out, void* stream) {
  if (!q || !n_out || (!host_out && max)) return GQ_E_INVAL;
  if (max > GQ_DRAIN_NOALLOC_MAX) {
    std::snprintf(g_err, sizeof g_err, "queue_drain_noalloc: max = %llu items exceeds GQ_DRAIN_NOALLOC_MAX = %u (static scratch); drain in pieces or use queue_drain",
                  (unsigned long long)max, (unsigned)GQ_DRAIN_NOALLOC_MAX);
    return GQ_E_INVAL;
  }
  unsigned char* scratch = nullptr;
  int rc = drain_scratch_address(&scratch);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  q->fresh = false;
  const uint32_t lanes = std::min(32u, q->max_threads);
  return dispatch(q, [&](auto& view) { return drain_noalloc_t(view, scratch, host_out, max, n_out, st, lanes); });
}

template <class Q>
static int script_t(const Q& view, const uint32_t* op, const uint32_t* arg, uint64_t count, uint32_t tid, uint32_t* st_out, uint32_t* val_out) {
  uint32_t* d = nullptr;
  CU(cudaMalloc(&d, count * 16));
  uint32_t *d_op = d, *d_arg = d + count, *d_st = d + 2 * count, *d_val = d + 3 * count;
  cudaError_t e = cudaMemcpy(d_op, op, count * 4, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d_arg, arg, count * 4, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) { script_kernel<Q><<<1, 1>>>(view, d_op, d_arg, count, tid, d_st, d_val); e = cudaDeviceSynchronize(); }
  if (e == cudaSuccess) e = cudaMemcpy(st_out, d_st, count * 4, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(val_out, d_val, count * 4, cudaMemcpyDeviceToHost);
  cudaFree(d);
  return e == cudaSuccess ? 0 : cuda_fail(e, "script");
}
extern "C" int queue_run_script(gq_queue* q, const uint32_t* host_op, const uint32_t* host_arg, uint64_t count,
                                uint32_t tid, uint32_t* host_status, uint32_t* host_val) {
  if (!q || !host_op || !host_arg || !host_status || !host_val || tid >= q->max_threads) return GQ_E_INVAL;
  if (count == 0) return 0;
  q->fresh = false;
  return dispatch(q, [&](auto& view) { return script_t(view, host_op, host_arg, count, tid, host_status, host_val); });
}

extern "C" int history_dump(gq_queue* q, gq_hist_rec* host_out, uint64_t max, uint64_t* n_out) {
  if (!q || !n_out || (!host_out && max)) return GQ_E_INVAL;
  const uint64_t n = std::min(max, q->hist_n);
  if (n) CU(cudaMemcpy(host_out, q->d_hist, n * sizeof(gq_hist_rec), cudaMemcpyDeviceToHost));
  *n_out = n;
  return 0;
}
