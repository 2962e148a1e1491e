// Shared plumbing of libdriftsched.so (CUDA path only; the oracle never includes this).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/driftsched.h"

namespace ds {

// sticky device status word (DS_DEV_* bits): lives in api.cu, kernels get its device address as an argument
// (one word per device: the address is looked up for the calling thread's current device)
unsigned int* status_ptr();  // nullptr if the symbol address cannot be obtained
int num_sms();               // SM count of the current device (148 on a B200), 0 on a CUDA error
// true exactly once per (device, which): the caller then sets that kernel's cudaFuncAttributeMaxDynamicSharedMemorySize
enum { DS_ATTR_K1 = 0, DS_ATTR_K3_HIST = 1, DS_ATTR_K3_LAT = 2 };
bool attr_needed(int which);

// host side bookkeeping (api.cu)
void note_launch(int n = 1);
int cuda_fail(cudaError_t e);  // records the message, returns DS_ECUDA

#define DS_CUDA(expr)                                   \
  do {                                                  \
    cudaError_t _e = (expr);                            \
    if (_e != cudaSuccess) return ::ds::cuda_fail(_e);  \
  } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr int kNumSMsB200 = 148;  // what the per-SM tuning constants below were measured on; grids use num_sms()

}  // namespace ds
