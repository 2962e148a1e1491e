// Shared plumbing of libdriftsched.so (CUDA path only; the oracle never includes this).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/driftsched.h"

namespace ds {

// sticky device status word (DS_DEV_* bits): lives in api.cu, kernels get its device address as an argument
unsigned int* status_ptr();  // nullptr if the symbol address cannot be obtained

// host side bookkeeping (api.cu)
void note_launch(int n = 1);
int cuda_fail(cudaError_t e);  // records the message, returns DS_ECUDA

#define DS_CUDA(expr)                                   \
  do {                                                  \
    cudaError_t _e = (expr);                            \
    if (_e != cudaSuccess) return ::ds::cuda_fail(_e);  \
  } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr int kNumSMs = 148;  // B200

}  // namespace ds
