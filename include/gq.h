/* gq.h — C ABI of the B200-native concurrent-queue library (libgq.so).
 *
 * Implements the three linearizable bounded GPU queues of "Scalable Concurrent Queues for
 * GPU" (arxiv 2606.01693; cited below as P:Lnnn = reference/PAPER.md line nnn):
 *   GQ_LFQ      G-LFQ      lock-free sCQ-style ring, warp-batched FAA     P:L86-228  §III-B, Alg. 1
 *   GQ_WFQ      G-WFQ      + bounded wait-free slow path, 64-bit CAS only P:L230-331 §III-C, Alg. 2
 *   GQ_WFQ_YMC  G-WFQ-YMC  Yang/Mellor-Crummey queue on a preallocated pool P:L80-84 §III-A
 *
 * The queue operation itself (enqueue / dequeue issued by every resident thread) is a
 * __device__ API: include/gq/queue.cuh.  This header is the host boundary: plain pointers
 * and sizes, no C++ or torch types.  Every step runs in the library's own CUDA kernels;
 * there is no CPU fallback: without a CUDA device every compute entry point returns
 * GQ_E_CUDA.
 *
 * Conventions
 *  - Every function returns int: 0 = success, negative = error (below).  Out-parameters are
 *    written only on success (run_* also fill *res on GQ_E_POOL with the partial counters).
 *  - "host" / "device" is stated for every pointer.  Streams are cudaStream_t passed as
 *    void* (NULL = default stream).  Calls are synchronous on that stream.
 *  - Ownership: queue_create allocates device memory owned by the handle until
 *    queue_destroy.  With gq_opts.storage the caller (e.g. torch) owns the device block and
 *    the library only formats it.  Caller buffers stay the caller's.
 *    Every call returns only after its device work has completed, so work of two calls never overlaps, whatever
 *    streams they name.  run_* / queue_run_script / the ceilings take no stream: they launch on the default stream.
 *  - GQ_E_TIMEOUT (watchdog, GQ_WATCHDOG_S): the kernel is still running; its device buffers are deliberately not
 *    freed (that would block on it).  The context is unusable until the process ends or the device is reset.
 *  - A handle is not safe for concurrent host calls.
 */
#ifndef GQ_H_
#define GQ_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { GQ_LFQ = 0, GQ_WFQ = 1, GQ_WFQ_YMC = 2,                /* kind: the paper's three queues */
       GQ_LFQ_DIRECT = 3 };  /* ablation (not in the paper): G-LFQ without the index indirection of P:L88: one ring whose
                                entries carry the uint32 payload; half the atomics per operation, capacity bound soft:
                                at most capacity + (participating threads) items (include/gq/dlfq.cuh) */
enum { GQ_OK = 0, GQ_FULL = 1, GQ_EMPTY = 2 };               /* device-op status */
enum { GQ_E_INVAL = -1, GQ_E_NOMEM = -2, GQ_E_CUDA = -3, GQ_E_RESIDENCY = -4,
       GQ_E_TIMEOUT = -5, GQ_E_STATE = -6, GQ_E_POOL = -7 };
enum { GQ_OP_ENQ = 0, GQ_OP_DEQ = 1 };                       /* op=0 ENQ, op=1 DEQ */

#define GQ_PATIENCE_ZERO 0xFFFFFFFFu   /* patience value meaning "no fast attempts": every op takes the slow path */

typedef struct gq_queue gq_queue;      /* opaque host handle */

/* All fields 0 = default. */
typedef struct {
  uint32_t max_threads;     /* k upper bound: sizes per-thread records and the ring parameter
                               N = max(capacity, pow2ceil(max_threads)) (reading G1);
                               default = full co-residency of the benchmark kernel */
  uint32_t enq_patience;    /* G-WFQ / YMC fast attempts before the slow path; default 64 / 10 */
  uint32_t deq_patience;    /* default 64 / 10 */
  uint32_t help_delay;      /* D: inspect one peer record every D operations; default 64 */
  uint64_t ymc_pool_cells;  /* G-WFQ-YMC preallocated cells; default 2^26 */
  void*    storage;         /* optional caller-owned DEVICE block of >= queue_storage_bytes() bytes, 256 B aligned */
  size_t   storage_bytes;
  uint32_t layout;          /* ring entry stride: 0 = dense 8 B (default), 1 = 32 B sector, 2 = 128 B line */
  uint32_t flags;           /* GQ_F_* */
  uint32_t park_ns;         /* longest wait of a dequeuer on its own vacant slot before it gives the slot up
                               (D2); default 250000 */
  uint32_t park_nap_ns;     /* longest single __nanosleep between two looks at a parked slot (D2); default 128;
                               values below 32 = no sleep at all (pure re-reading of the slot) */
  uint32_t park_spin_ns;    /* a parked dequeuer re-reads its slot without any nap for this long before it starts the nap ladder
                               (D2); default 2000; GQ_PARK_SPIN_NONE = ladder from the first look */
  uint32_t reserved;        /* must be 0 */
} gq_opts;
#define GQ_PARK_SPIN_NONE 0xFFFFFFFFu
enum { GQ_F_PER_LANE_FAA = 1u,  /* ablation: one FAA per thread instead of the warp-batched one ("naive") */
       GQ_F_NO_PROBE = 2u,      /* ablation: no read-only emptiness probe before a ticket is claimed (D1) */
       GQ_F_NO_DEQ_SPIN = 4u,   /* ablation: dequeuer invalidates a vacant slot at once, no parking (D2) */
       GQ_F_NO_OPT_CAS = 8u,    /* ablation: TRYENQ loads the slot before its CAS (Alg. 1 L148 as written) instead of
                                   issuing the CAS against the predicted steady-state entry first (D3) */
       GQ_F_PLAIN_THR_STORE = 16u /* ablation: Threshold reset = plain store per enqueue instead of load-compare-store
                                   (measured 50x slower on B200: same-address stores serialise at L2) */,
       GQ_F_THR_FIRST = 32u,    /* ablation: read and test Threshold before the Head ticket is drawn, as listed in
                                   Alg. 1, instead of overlapping the two (D4) */
       GQ_F_NO_PAIRED_FAA = 64u,/* ablation: G-LFQ dequeue reserves its FQ tail ticket only after the payload load has
                                   returned, instead of behind it (D5) */
       GQ_F_THR_RED_MAX = 128u, /* variant: Threshold reset = one red.max by the warp leader instead of load-compare-store
                                   (measured slower on B200: it doubles the same-address atomic load) */
       GQ_F_EAGER_EMPTY = 512u, /* polling consumers (BFS, tracer): a dequeuer that sees Tail <= Head returns EMPTY at once
                                   and parks (D2) only for an enqueuer that already holds its ticket; the default waits
                                   in line for future enqueues, which is what the fixed-duration benchmarks want */
       GQ_F_NO_CELL_PREFETCH = 1024u, /* ablation: G-WFQ-YMC enqueue does not prefetch the pool cells of the next ticket wave into L2 */
       GQ_F_NO_FULL_TEST = 2048u, /* G-LFQ-D only: the caller guarantees that the queue never holds `capacity` items (a BFS
                                   frontier queue of nv slots, a work queue of all items): enqueue skips the FULL test, which is
                                   the two hot-word loads that make G-LFQ-D slow at scale */
       GQ_F_NO_REPAIR = 4096u,  /* ablation: a waiting dequeuer does not re-arm a slot that was marked unsafe (D9) */
       GQ_F_FENCED_PAYLOAD = 256u /* G-LFQ: order the payload against the index hand-over with release fences in front of
                                   both installing CAS (the paper's implicit scheme) instead of the payload-cell
                                   handshake (D6) */ };

/* Device bytes queue_create_ex would need for (kind, capacity, opts). */
size_t queue_storage_bytes(int kind, uint64_t capacity, const gq_opts* opts);
/* Create a queue of logical capacity n = `capacity` uint32 payloads ("logical capacity n").
   capacity >= 1.  GQ_WFQ_YMC: capacity does not throttle, the pool does (reading Y3). */
int queue_create   (int kind, uint64_t capacity, gq_queue** out);
int queue_create_ex(int kind, uint64_t capacity, const gq_opts* opts, gq_queue** out);
int queue_destroy  (gq_queue* q);
/* Back to the empty initial state (reading G4). */
int queue_reset    (gq_queue* q, void* stream);
/* Enqueue host_vals[0..count) in array order (one warp, so FIFO order = array order).
   Returns GQ_E_STATE if fewer than `count` fit.  host_vals: HOST. */
int queue_prefill  (gq_queue* q, const uint32_t* host_vals, uint64_t count, void* stream);
/* Dequeue until EMPTY or `max` items, in FIFO order, into host_out (HOST). */
int queue_drain    (gq_queue* q, uint32_t* host_out, uint64_t max, uint64_t* n_out, void* stream);
/* queue_drain for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
   cudaMalloc): same arguments, same result, but the staging memory is a static device array inside the library instead of
   two cudaMalloc'ed blocks; the call makes no cudaMalloc / cudaFree.  max > GQ_DRAIN_NOALLOC_MAX returns GQ_E_INVAL with a
   message in gq_last_cuda_error() (drain in pieces, or use queue_drain).  All calls on one GPU share that array: calls that
   overlap on the GPU (two host threads, two streams) race. */
#define GQ_DRAIN_NOALLOC_MAX 65536u
int queue_drain_noalloc(gq_queue* q, uint32_t* host_out, uint64_t max, uint64_t* n_out, void* stream);
/* Copy the POD device view (gq::LfqView / WfqView / YmcView of include/gq/queue.cuh) that user
   kernels take by value.  view_out: HOST, view_bytes must be >= sizeof(view). */
int queue_device_view(const gq_queue* q, void* view_out, size_t view_bytes);
int queue_kind(const gq_queue* q);
/* Read-back of the hot words of a QUIESCENT queue (synchronises the device first).  out16: HOST, 16 words:
   G-LFQ / G-WFQ: [0] AQ.Head, [1] AQ.Tail (ticket counters, decoded from the packed word), [2] AQ.Threshold (signed), [3] FQ.Head,
   [4] FQ.Tail, [5] FQ.Threshold; G-LFQ-D: Head, Tail, Threshold; G-WFQ-YMC: H, T.  [6] = ring parameter N, [7] = max_threads.
   G-WFQ also: slow-path rounds since the last reset, summed over the threads that performed them (Lemma III.7):
   [8] AQ.Tail increments <c,NULL> -> <c+1,tid> won, [9] INC bits cleared on local tails (completed rounds), [10], [11] the same
   for AQ.Head; [12..15] the same four for FQ. */
int queue_debug_counters(gq_queue* q, uint64_t* out16);
/* Largest thread count the benchmark kernel of this kind can keep co-resident (occupancy
   API x SM count): the forward-progress assumption of Thm III.10. */
int queue_max_coresident_threads(int kind, int block_threads, uint32_t* out);

typedef struct {
  uint32_t threads;            /* participating threads k (<= max co-resident; 0 = full co-residency) */
  uint32_t block_threads;      /* 0 = 256 */
  double   warmup_ms;          /* P:L359 "warmup interval followed by a measurement interval" */
  double   duration_ms;        /* t_meas of P:L355 */
  double   producer_fraction;  /* run_split: P(thread is a producer) */
  uint64_t seed;               /* roles, jitter */
  uint32_t record_history;     /* 1: log {proc,op,arg,ret,call,end} per op; needs ops_per_thread > 0 */
  uint32_t ops_per_thread;     /* > 0: fixed-op mode (iterations per thread) instead of fixed duration */
  uint32_t jitter_ns;          /* random __nanosleep in [0, jitter_ns] before each op (history runs) */
  uint32_t fail_backoff_ns;    /* harness sleeps up to this long after a FULL/EMPTY return (0 = none) */
  uint64_t value_base;         /* first payload value (split: prefill size).  Payload of (thread t, iteration i): value_base +
                                  (t << 16 | i) in history runs of at most 65536 threads x 65536 iterations (BASELINE.json
                                  configs[0]), else value_base + t + i * threads; unique in both cases */
  uint32_t role_layout;        /* run_split: 0 = logical thread t runs on physical thread t (mixed warps, the default);
                                  1 = same seeded roles, but the logical threads are placed so that producers fill the
                                  first physical threads and consumers the rest: warps are homogeneous (at most one mixed);
                                  2 = layout 0, but each iteration is ONE converged call of the fused operation
                                  gq::enqueue_or_dequeue_step (G-LFQ only): the two roles of a mixed warp overlap, and a
                                  lane that has to wait in line hands the wait back instead of holding up its warp (D12);
                                  4 = the same with the blocking gq::enqueue_or_dequeue; 3 = layout 1 through the fused
                                  operation (diagnostic: homogeneous warps, one address group) */
  uint32_t converged;          /* 1: the lanes of a warp start every iteration of the benchmark loop together (one ballot per
                                  iteration), as a lock-step wavefront would; 0: a lane starts its next operation as soon as its
                                  last one returns */
  uint32_t block_faa;          /* 1: the warps of a block combine their ticket requests per hot counter in shared memory: one global
                                  FAA per batch instead of one per warp (block-level funnel, D11; include/gq/queue.cuh) */
  uint32_t funnel_window_ns;   /* block_faa: a batch stays open this long so that more warps can join (0 = closed at once) */
} gq_run_cfg;

typedef struct {
  uint64_t succ_enq, succ_deq, full, empty;      /* inside the measurement window */
  uint64_t tot_enq, tot_deq, tot_full, tot_empty;/* whole kernel, for conservation */
  uint64_t sum_enq, sum_deq;                     /* sums of OK payloads, mod 2^64, whole kernel */
  uint64_t slow_enq, slow_deq, helps, retries;   /* G-WFQ / YMC slow-path entries, helps given, ring retries */
  double   meas_seconds;                         /* t_meas (fixed-op mode: kernel device time) */
  double   kernel_ms;                            /* CUDA-event time of the benchmark kernel */
  uint32_t threads_launched, blocks, blocks_per_sm, pool_exhausted;
} gq_run_result;

/* P:L349 balanced kernel: every thread loops { enqueue(unique v); dequeue() }.  The queue is
   NOT reset first.  Fixed-op mode runs cfg->ops_per_thread iterations per thread. */
int run_balanced(gq_queue* q, const gq_run_cfg* cfg, gq_run_result* res);
/* P:L349 split kernel: thread is a pure producer iff mix32(seed, tid) < producer_fraction * 2^32. */
int run_split   (gq_queue* q, const gq_run_cfg* cfg, gq_run_result* res);
/* Ceiling C1: bare warp-batched FAA (Alg. 1 WAVEFAA) on one counter, nothing else.
   res->succ_enq = tickets taken inside the window.  n_counters in {1,4}: 4 = each warp cycles
   over four padded counters (the like-for-like ceiling for one enqueue+dequeue pair). */
#define GQ_CEILING_PER_LANE 0x100u   /* OR into n_counters: one FAA per thread (the "naive" loop of P:L95) instead of WAVEFAA */
int run_faa_ceiling(const gq_run_cfg* cfg, uint32_t n_counters, gq_run_result* res);
/* Ceiling C2: coalesced stream of 64-bit CAS + red.or over a ring-sized L2-resident buffer. */
int run_slot_atomic_ceiling(const gq_run_cfg* cfg, uint64_t slots, gq_run_result* res);

/* Lemma III.1 probe: `threads` threads call the warp-batched FAA `rounds` times inside
   seeded divergent control flow; tickets_out (HOST, threads*rounds entries, UINT64_MAX = lane did
   not participate that round); *final_counter = counter value at the end. */
int run_warp_faa_probe(uint32_t threads, uint32_t rounds, uint64_t seed, uint64_t* tickets_out, uint64_t* final_counter);

/* The same probe with the tickets drawn through a block-level funnel (D11; blocks of 256 threads, one funnel per
   block): Lemma III.1 must hold batch-wise.  tickets_out may be NULL (long runs); sum_count_out (HOST, 2 words, may be NULL)
   = sum of all tickets handed out and their number: with distinct tickets 0..m-1 the sum is m(m-1)/2. */
int run_funnel_probe(uint32_t threads, uint32_t rounds, uint64_t seed, uint32_t funnel_window_ns, uint64_t* tickets_out,
                     uint64_t* final_counter, uint64_t* sum_count_out);

/* Single-thread script: op[i] in {GQ_OP_ENQ, GQ_OP_DEQ}, arg[i] payload; results to HOST arrays.
   `tid` = the thread_ctx id used (exercises per-thread records). */
int queue_run_script(gq_queue* q, const uint32_t* host_op, const uint32_t* host_arg, uint64_t count,
                     uint32_t tid, uint32_t* host_status, uint32_t* host_val);

typedef struct { uint32_t proc, op, arg, ret_status, ret_val, _pad; uint64_t call_ns, end_ns; } gq_hist_rec;
/* Records of the last record_history run, thread-major.  host_out: HOST. */
int history_dump(gq_queue* q, gq_hist_rec* host_out, uint64_t max, uint64_t* n_out);

/* Level-synchronous BFS with two alternating frontier queues ("At each level, the current
   frontier is dequeued, outgoing neighbors are examined, and newly visited vertices are marked and
   are enqueued into the next frontier.  We alternate between two queues across BFS levels until the
   next frontier is empty").  One persistent cooperative launch; grid-wide barriers between levels.
   d_rowptr (nv+1 uint64), d_col (uint32 ids), d_dist (nv int32, OUTPUT: hop distance, -1 =
   unreachable): DEVICE, caller-owned.  stats_out: HOST.  The two queues (capacity pow2ceil(nv)) are
   created and destroyed inside the call; stats.ms is the CUDA-event time of the BFS kernel alone,
   stats.total_ms the whole call (queue creation, dist fill, kernel).  Errors: GQ_E_INVAL (src >=
   nv, bad kind), GQ_E_POOL (G-WFQ-YMC pool exhausted), GQ_E_STATE (a frontier queue reported FULL). */
typedef struct {
  uint32_t threads;        /* participating threads (P:L365 sweeps 2^9..2^13); 0 = full co-residency */
  uint32_t block_threads;  /* 0 = 256 */
  uint32_t huge_degree;    /* adjacency lists at least this long are expanded by the whole grid; 0 = 64 (also the minimum) */
  uint32_t flags;          /* GQ_F_* for the two queues */
} gq_bfs_opts;
typedef struct { uint32_t levels; uint32_t threads; uint64_t edges_scanned, vertices_visited, queue_ops; double ms, total_ms; } gq_bfs_stats;
int bfs_run(int kind, const uint64_t* d_rowptr, const uint32_t* d_col, uint32_t nv, uint32_t src,
            int32_t* d_dist, gq_bfs_stats* stats_out, void* stream);
int bfs_run_ex(int kind, const uint64_t* d_rowptr, const uint32_t* d_col, uint32_t nv, uint32_t src,
               int32_t* d_dist, const gq_bfs_opts* opts, gq_bfs_stats* stats_out, void* stream);

/* Tile-based persistent wavefront path tracer driven by ONE work queue of tile items ("a
   persistent tracing kernel repeatedly dequeues work, traces rays, shades hits, and re-enqueues
   reflective bounces ... until no work remains"; BASELINE.json config 5: "work queue of tile ids",
   "secondary-ray batches are re-enqueued per bounce").  Item = tile | sample << 20 | bounce << 26;
   one warp advances the 16x16 pixel-paths of an item by one bounce.  Arithmetic, camera, RNG and
   shading constants: DESIGN.md section 6 (fp32, no FMA contraction).  d_rgb: DEVICE, height*width*3
   floats, row-major, OUTPUT.  stats.ms = CUDA-event time of the tracing + resolve kernels. */
typedef struct { uint32_t width, height, spp, max_bounce, n_spheres, threads; uint64_t seed;
                 const float* d_spheres; /* DEVICE, n_spheres x 8: cx,cy,cz,r, ar,ag,ab, emissive(0/1) */ } gq_rt_scene;
typedef struct { uint64_t rays, queue_ops; double ms, total_ms; uint32_t threads, items; } gq_rt_stats;
int rt_render(int kind, const gq_rt_scene* scene, float* d_rgb /* DEVICE H*W*3 */, gq_rt_stats* stats_out, void* stream);
/* The same image through the paper's own work distribution ("each tile owns its own queue"): mode 1 creates one queue
   per 16x16 tile, items are RAYS (pixel in tile | sample << 8 | bounce << 14).  Every thread block owns the tiles b, b + blocks,
   ...; its warps pull rays from those queues, 8 lanes per queue and 4 queues per instruction (the address-matched WAVEFAA,
   gq::enqueue / dequeue with kUniform = false), trace them and re-enqueue the bounce into the queue of the same tile.  The
   image is bit-identical to mode 0 (same per-path arithmetic, RNG keyed by pixel, sample and bounce).  GQ_LFQ and
   GQ_LFQ_DIRECT only (the kinds with per-thread records would need tiles x threads of them): others return GQ_E_INVAL. */
typedef struct { uint32_t mode;      /* 0 = one work queue of tile items (rt_render), 1 = one queue per tile, items = rays */
                 uint32_t reserved; } gq_rt_opts;
int rt_render_ex(int kind, const gq_rt_scene* scene, float* d_rgb, const gq_rt_opts* opts, gq_rt_stats* stats_out, void* stream);

/* Debug and fault-injection builds only (include/gq/detail/debug.cuh; paper_2606_01693_b200/build.py variants "dbg"
   and "mutants").  In the product build all three return GQ_E_INVAL and do nothing.
   gq_dbg_sites : out80 (HOST, 80 words) = event counters [0,32), latency-probe cycle sums [32,48) and sample counts
                  [48,64) since the last call; clears them.
   gq_dbg_trace : the first events of the launches since the last call, 64 B each {ns, site | tid << 32, ticket,
                  entry, Head, Tail, Threshold, aux}; out: HOST; clears the ring.
   gq_set_mutation : arm fault `id` (0 = none) for the following launches (SURVEY section 4 "mutation tests"). */
int gq_dbg_sites(unsigned long long* out80);
int gq_dbg_trace(void* out, uint64_t max_records, uint64_t* n_out);
int gq_set_mutation(uint32_t id);

const char* gq_last_cuda_error(void);   /* text of the last CUDA error seen by this thread */
const char* gq_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GQ_H_ */
