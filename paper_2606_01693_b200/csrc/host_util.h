// Host helpers shared by the translation units of libgq.so (defined in capi.cu; not exported).
#pragma once
#include <cuda_runtime.h>

#include "gq.h"

#define GQ_HIDDEN __attribute__((visibility("hidden")))

GQ_HIDDEN int gq_cuda_fail(cudaError_t e, const char* what);      // records the text for gq_last_cuda_error()
GQ_HIDDEN void gq_set_error(const char* text);
GQ_HIDDEN int gq_device_sms();
GQ_HIDDEN double gq_watchdog_slack_s();                            // GQ_WATCHDOG_S or 60
GQ_HIDDEN int gq_wait_event(cudaEvent_t ev, double budget_s);      // 0, GQ_E_TIMEOUT or GQ_E_CUDA

// count queues of one shape in one device block (capi.cu); G-LFQ / G-LFQ-D
GQ_HIDDEN int gq_create_many(int kind, uint64_t capacity, const gq_opts* opts, uint32_t count, gq_queue** out, void** block_out, cudaStream_t st);
GQ_HIDDEN void gq_destroy_many(gq_queue** qs, uint32_t count, void* block);

#define CU(call)                                             \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return gq_cuda_fail(e_, #call);   \
  } while (0)
