// ds_estimation_error — estimation-fidelity reductions: job classes of Eq. 3-4
// (PAPER.md:135, 154), token-estimation error of Tables IV / X and queue wait by job class
// of Table IX. All outputs are exact integer sums, so any reduction order is bit-exact; the caller
// derives MAE = sum|err|/n, RMSE = sqrt(sum err^2/n), mean bias = sum P / sum est in fp64.
#include "common.cuh"

namespace ds {
namespace k4 {

constexpr int kFields = 11;   // n, sum|err|, sum err^2, sum est, sum P, n_short, n_medium, n_long, sum qdelay per class x3

__global__ void __launch_bounds__(256) esterr_kernel(const int64_t* __restrict__ trace_off, const int64_t* __restrict__ arrival,
                                                     const int32_t* __restrict__ tokens, const int32_t* __restrict__ out_len,
                                                     const ds_instance* __restrict__ inst,
                                                     long long n_inst, const int64_t* __restrict__ out_off,
                                                     const int64_t* __restrict__ arr_ov, const int64_t* __restrict__ est, const int64_t* __restrict__ start,
                                                     const int32_t* __restrict__ group, int n_groups, unsigned long long* out,
                                                     int32_t* __restrict__ class_seg, unsigned int* status) {
  const int lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  // one warp per instance (an instance belongs to one group): lane-local sums, shuffle reduction, 11 atomics per instance
  for (long long ii = (long long)blockIdx.x * nwarp + (threadIdx.x >> 5); ii < n_inst; ii += (long long)gridDim.x * nwarp) {
    const int t = inst[ii].trace;
    const long long lo = trace_off[t], n = trace_off[t + 1] - lo, oo = out_off[ii];
    const int g = group ? group[ii] : 0;
    if (g < 0 || g >= n_groups) { if (lane == 0) atomicOr(status, DS_DEV_BAD_INSTANCE); continue; }
    const bool with_out = inst[ii].estimator >= DS_BUDGET_SPLIT;     // budget estimators predict input + output tokens (Eq. 1)
    const int64_t* __restrict__ ap = arr_ov ? arr_ov + oo : arrival + lo;   // closed loop: the instance's own arrival ticks
    unsigned long long acc[kFields];
#pragma unroll
    for (int k = 0; k < kFields; ++k) acc[k] = 0ull;
    for (long long r = lane; r < n; r += 32) {
      const long long e = est[oo + r], P = (long long)tokens[lo + r] + (with_out ? (long long)out_len[lo + r] : 0ll), err = e - P;
      const int cls = e <= 128 ? 0 : (e <= 512 ? 1 : 2);                     // Eq. 4
      const unsigned long long qd = start ? (unsigned long long)(start[oo + r] - ap[r]) : 0ull;
      acc[0] += 1ull; acc[1] += (unsigned long long)(err < 0 ? -err : err); acc[2] += (unsigned long long)(err * err);
      acc[3] += (unsigned long long)e; acc[4] += (unsigned long long)P;
#pragma unroll
      for (int c = 0; c < 3; ++c) { acc[5 + c] += cls == c ? 1ull : 0ull; acc[8 + c] += cls == c ? qd : 0ull; }
      if (class_seg) class_seg[oo + r] = 3 * g + cls;
    }
#pragma unroll
    for (int k = 0; k < kFields; ++k) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);   // wrap-around adds: exact mod 2^64
    }
    if (lane < kFields) {
      unsigned long long v = 0ull;
#pragma unroll
      for (int k = 0; k < kFields; ++k) if (lane == k) v = acc[k];
      if (v) atomicAdd(out + (size_t)g * kFields + lane, v);
    }
  }
}

}  // namespace k4
}  // namespace ds

extern "C" int ds_estimation_error(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                                   const int64_t* arrival_override, const int64_t* est, const int64_t* start_tick, const int32_t* group, int32_t n_groups,
                                   int64_t* out, int32_t* class_seg, void* stream) {
  using namespace ds;
  if (!tr || n_inst < 0 || n_groups < 1 || !out) return DS_EINVAL;
  if (n_inst > 0 && (!inst || !out_off || !est || !tr->trace_off || !tr->tokens || !tr->out_len || (start_tick && !arrival_override && !tr->arrival_tick))) return DS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  unsigned int* status = status_ptr();
  if (!status) return cuda_fail(cudaGetLastError());
  DS_CUDA(cudaMemsetAsync(out, 0, sizeof(int64_t) * k4::kFields * (size_t)n_groups, s));
  if (n_inst == 0) return DS_OK;
  long long blocks = (n_inst + 7) / 8;
  if (blocks > num_sms() * 8) blocks = num_sms() * 8;
  k4::esterr_kernel<<<(unsigned)blocks, 256, 0, s>>>(tr->trace_off, tr->arrival_tick, tr->tokens, tr->out_len, inst, n_inst, out_off, arrival_override, est, start_tick,
                                                    group, n_groups, (unsigned long long*)out, class_seg, status);
  note_launch();
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}
