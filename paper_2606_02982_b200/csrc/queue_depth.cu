// ds_queue_depth — per-tenant queue depth over time (Fig. 8).
//   depth[i][j][k] = #{requests r of instance i with tier k : arrival_r <= t_j < start_r},  t_j = t0 + j*dt.
// Counting form used here: depth(t_j) = #{arrival <= t_j} - #{start <= t_j}. Every request adds +1 at the first sample
// at or after its arrival and -1 at the first sample at or after its admission (integer atomics into the output, which
// therefore first holds the difference sequence), then one warp per instance turns the differences into depths with an
// in-place prefix sum over the samples of each tier. All integer: any order is bit-exact.
#include "common.cuh"

namespace ds {
namespace k5 {

// first j >= 0 with t0 + j*dt >= x, clamped to n
__device__ __forceinline__ long long first_sample(long long x, long long t0, long long dt, long long n) {
  const long long d = x - t0;
  if (d <= 0) return 0;
  const unsigned long long q = ((unsigned long long)d + (unsigned long long)dt - 1ull) / (unsigned long long)dt;
  return q > (unsigned long long)n ? n : (long long)q;
}

__global__ void __launch_bounds__(256) diff_kernel(const int64_t* __restrict__ trace_off, const int64_t* __restrict__ arrival,
                                                   const uint8_t* __restrict__ tier, const ds_instance* __restrict__ inst,
                                                   long long n_inst, const int64_t* __restrict__ out_off,
                                                   const int64_t* __restrict__ arr_ov, const int64_t* __restrict__ start, long long t0, long long dt,
                                                   long long n_samples, int* __restrict__ depth) {
  const int lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  for (long long ii = (long long)blockIdx.x * nwarp + (threadIdx.x >> 5); ii < n_inst; ii += (long long)gridDim.x * nwarp) {
    const int t = inst[ii].trace;
    const long long lo = trace_off[t], n = trace_off[t + 1] - lo, oo = out_off[ii];
    int* row = depth + ii * n_samples * 3;
    const int64_t* __restrict__ ap = arr_ov ? arr_ov + oo : arrival + lo;   // closed loop: the instance's own arrival ticks
    for (long long r = lane; r < n; r += 32) {
      const int k = tier[lo + r];
      if (k > 2) continue;                                  // (ds_simulate reports bad tiers)
      const long long ja = first_sample(ap[r], t0, dt, n_samples);
      const long long js = first_sample(start[oo + r], t0, dt, n_samples);
      if (ja < js) {
        atomicAdd(row + ja * 3 + k, 1);
        if (js < n_samples) atomicAdd(row + js * 3 + k, -1);
      }
    }
  }
}

__global__ void __launch_bounds__(256) scan_kernel(long long n_inst, long long n_samples, int* __restrict__ depth) {
  const int lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  for (long long ii = (long long)blockIdx.x * nwarp + (threadIdx.x >> 5); ii < n_inst; ii += (long long)gridDim.x * nwarp) {
    int* row = depth + ii * n_samples * 3;
    int c0 = 0, c1 = 0, c2 = 0;                             // running depth per tier
    for (long long base = 0; base < n_samples; base += 32) {
      const long long j = base + lane;
      const bool in = j < n_samples;
      int v0 = in ? row[j * 3 + 0] : 0, v1 = in ? row[j * 3 + 1] : 0, v2 = in ? row[j * 3 + 2] : 0;
#pragma unroll
      for (int s = 1; s < 32; s <<= 1) {
        const int y0 = __shfl_up_sync(0xffffffffu, v0, s), y1 = __shfl_up_sync(0xffffffffu, v1, s), y2 = __shfl_up_sync(0xffffffffu, v2, s);
        if (lane >= s) { v0 += y0; v1 += y1; v2 += y2; }
      }
      v0 += c0; v1 += c1; v2 += c2;
      if (in) { row[j * 3 + 0] = v0; row[j * 3 + 1] = v1; row[j * 3 + 2] = v2; }
      c0 = __shfl_sync(0xffffffffu, v0, 31); c1 = __shfl_sync(0xffffffffu, v1, 31); c2 = __shfl_sync(0xffffffffu, v2, 31);
    }
  }
}

}  // namespace k5
}  // namespace ds

extern "C" int ds_queue_depth(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                              const int64_t* arrival_override, const int64_t* start_tick, int64_t t0, int64_t dt, int64_t n_samples, int32_t* depth, void* stream) {
  using namespace ds;
  if (!tr || n_inst < 0 || dt < 1 || n_samples < 0) return DS_EINVAL;
  if (n_inst == 0 || n_samples == 0) return DS_OK;
  if (!inst || !out_off || !start_tick || !depth || !tr->trace_off || (!arrival_override && !tr->arrival_tick) || !tr->tier) return DS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  DS_CUDA(cudaMemsetAsync(depth, 0, sizeof(int32_t) * 3 * (size_t)n_samples * (size_t)n_inst, s));
  long long blocks = (n_inst + 7) / 8;
  if (blocks > num_sms() * 8) blocks = num_sms() * 8;
  k5::diff_kernel<<<(unsigned)blocks, 256, 0, s>>>(tr->trace_off, tr->arrival_tick, tr->tier, inst, n_inst, out_off, arrival_override, start_tick, t0, dt,
                                                  n_samples, depth);
  k5::scan_kernel<<<(unsigned)blocks, 256, 0, s>>>(n_inst, n_samples, depth);
  note_launch(2);
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}
