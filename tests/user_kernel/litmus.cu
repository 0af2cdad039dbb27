// A USER kernel of the library: includes only the public __device__ header (include/gq/queue.cuh), gets the queue as the POD
// view that queue_device_view() (gq.h) hands out, and is compiled on its own (tests/user_kernel/build.py), not into libgq.so.
//
// Hand-over litmus (reading G15; SURVEY section 8(c.2) G15 pin: "producers write a second word of
// payload-dependent data").  A producer writes side[v] = f(v) with a plain store and then enqueues v; the consumer that
// dequeues v reads side[v] with a plain load and compares.  What the queue promises (include/gq/queue.cuh):
//   - the payload itself always arrives intact (every build);
//   - memory OTHER than the payload is published with the item when the producer issues __threadfence() before enqueue
//     (`fences` = 1 here; the dequeue's entry load is an acquire), or when the queue was created with GQ_F_FENCED_PAYLOAD
//     (installing CAS = release), with no fence in the user code (`fences` = 0).
#include <cuda_runtime.h>

#include <cstdint>
#include <cstring>

#include "gq/queue.cuh"

using namespace gq;

__device__ __forceinline__ uint32_t f_of(uint32_t v) { return (v * 0x9E3779B1u) | 1u; }

template <class Q>
__global__ void litmus_kernel(Q q, uint32_t* side, uint32_t threads, uint32_t n_prod, uint32_t ops, uint32_t fences,
                              unsigned long long* ctr /* [0] consumed, [1] mismatches, [2] foreign values */) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= threads) return;
  thread_ctx ctx{tid};
  ctx.help_peer = tid + 1;
  const unsigned long long total = (unsigned long long)n_prod * ops;
  if (tid < n_prod) {
    for (uint32_t i = 0; i < ops; ++i) {
      const uint32_t v = tid * ops + i;
      side[v] = f_of(v);                              // plain store, before the item is published
      if (fences) __threadfence();
      uint32_t nap = 32;
      while (enqueue(q, ctx, v) != OK) { __nanosleep(nap); nap = nap < 1024 ? nap * 2 : 1024; }   // FULL: try again
    }
  } else {
    uint32_t nap = 32;
    for (;;) {
      if (*reinterpret_cast<volatile unsigned long long*>(&ctr[0]) >= total) break;
      uint32_t v = 0;
      if (dequeue(q, ctx, &v) != OK) { __nanosleep(nap); nap = nap < 1024 ? nap * 2 : 1024; continue; }
      nap = 32;
      if (v >= total) { atomicAdd(&ctr[2], 1ull); atomicAdd(&ctr[0], 1ull); continue; }
      const uint32_t x = side[v];                     // plain load, after the item was received
      if (x != f_of(v)) atomicAdd(&ctr[1], 1ull);
      atomicAdd(&ctr[0], 1ull);
    }
  }
}

template <class Q>
static int run_t(const void* view, size_t view_bytes, uint32_t threads, uint32_t n_prod, uint32_t ops, uint32_t fences, uint64_t* out3) {
  if (view_bytes < sizeof(Q)) return -1;
  Q q;
  std::memcpy(&q, view, sizeof q);
  const uint32_t block = 128, blocks = (threads + block - 1) / block;
  int nb = 0, dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, litmus_kernel<Q>, (int)block, 0) != cudaSuccess) return -3;
  if (blocks > (uint32_t)(nb * sms)) return -4;       // consumers spin: every block must be resident
  uint32_t* side = nullptr;
  unsigned long long* ctr = nullptr;
  const size_t n = (size_t)n_prod * ops;
  if (cudaMalloc(&side, n * 4 + 4) != cudaSuccess || cudaMalloc(&ctr, 32) != cudaSuccess) return -2;
  cudaMemset(side, 0, n * 4 + 4);
  cudaMemset(ctr, 0, 32);
  litmus_kernel<Q><<<blocks, block>>>(q, side, threads, n_prod, ops, fences, ctr);
  cudaError_t e = cudaDeviceSynchronize();
  unsigned long long h[4] = {0, 0, 0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(h, ctr, 32, cudaMemcpyDeviceToHost);
  cudaFree(side); cudaFree(ctr);
  if (e != cudaSuccess) return -3;
  out3[0] = h[0]; out3[1] = h[1]; out3[2] = h[2];
  return 0;
}

// kind: GQ_LFQ 0, GQ_WFQ 1, GQ_WFQ_YMC 2, GQ_LFQ_DIRECT 3 (gq.h); view: HOST copy of the device view
extern "C" int litmus_run(int kind, const void* view, size_t view_bytes, uint32_t threads, uint32_t n_prod, uint32_t ops,
                          uint32_t fences, uint64_t* out3) {
  if (!view || !out3 || n_prod == 0 || n_prod >= threads || (uint64_t)n_prod * ops >= (1ull << 31)) return -1;
  switch (kind) {
    case 0: return run_t<LfqView>(view, view_bytes, threads, n_prod, ops, fences, out3);
    case 1: return run_t<WfqView>(view, view_bytes, threads, n_prod, ops, fences, out3);
    case 2: return run_t<YmcView>(view, view_bytes, threads, n_prod, ops, fences, out3);
    case 3: return run_t<DlfqView>(view, view_bytes, threads, n_prod, ops, fences, out3);
    default: return -1;
  }
}
