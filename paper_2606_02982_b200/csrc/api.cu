// libdriftsched.so: error handling, status word, workspace sizes (include/driftsched.h).
#include <atomic>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "common.cuh"

namespace ds {

__device__ unsigned int g_status_word = 0;

static thread_local char t_cuda_err[256] = "";
static std::atomic<long long> g_launches{0};

// Per-DEVICE state (a process may drive several devices, one after the other or from several threads): the status word's
// address, the SM count and which kernels already have their dynamic-shared-memory attribute set on that device.
namespace {
struct DeviceState { unsigned int* status = nullptr; int num_sms = 0; unsigned attr_mask = 0; bool init = false; };
constexpr int kMaxDevices = 64;
DeviceState g_dev[kMaxDevices];
std::mutex g_dev_mu;
DeviceState* device_state() {   // state of the calling thread's current device, nullptr on a CUDA error
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= kMaxDevices) return nullptr;
  std::lock_guard<std::mutex> lk(g_dev_mu);
  DeviceState& st = g_dev[d];
  if (!st.init) {
    void* q = nullptr;
    if (cudaGetSymbolAddress(&q, g_status_word) != cudaSuccess) return nullptr;
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, d) != cudaSuccess || n < 1) return nullptr;
    st.status = (unsigned int*)q; st.num_sms = n; st.init = true;
  }
  return &st;
}
}  // namespace

unsigned int* status_ptr() { DeviceState* st = device_state(); return st ? st->status : nullptr; }
int num_sms() { DeviceState* st = device_state(); return st ? st->num_sms : 0; }
bool attr_needed(int which) {
  DeviceState* st = device_state();
  if (!st) return true;
  std::lock_guard<std::mutex> lk(g_dev_mu);
  const bool need = !(st->attr_mask & (1u << which));
  st->attr_mask |= 1u << which;
  return need;
}

void note_launch(int n) { g_launches += n; }

int cuda_fail(cudaError_t e) {
  snprintf(t_cuda_err, sizeof(t_cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
  cudaGetLastError();  // clear non-sticky error state
  return DS_ECUDA;
}

// sizes shared with the kernels' own layouts (kept in one place: each .cu exposes its need)
size_t ws_characterize(int64_t n_bytes, int64_t n_prompts);
size_t ws_simulate(int64_t total_requests, int64_t n_inst);
size_t ws_tail_stats(int64_t n_segments, int64_t n_pct);
size_t ws_latency_stage(int64_t n_total);
size_t ws_simulate_traces(int64_t n_requests);

}  // namespace ds

extern "C" {

size_t ds_workspace_bytes(int which, int64_t n, int64_t m) {
  size_t b = 0;
  if (n < 0) n = 0;
  if (m < 0) m = 0;
  switch (which) {
    case DS_WS_CHARACTERIZE: b = ds::ws_characterize(n, m); break;
    case DS_WS_SIMULATE: b = ds::ws_simulate(n, m); break;
    case DS_WS_TAIL_STATS: b = ds::ws_tail_stats(n, m); break;
    case DS_WS_LATENCY_STAGE: b = ds::ws_latency_stage(n); break;
    case DS_WS_SIMULATE_TRACES: b = ds::ws_simulate_traces(n); break;
    default: b = 0;
  }
  return b < 256 ? 256 : b;
}

int ds_device_status(void* stream) {
  unsigned int* p = ds::status_ptr();
  if (!p) return ds::cuda_fail(cudaGetLastError());
  unsigned int h = 0, zero = 0;
  cudaStream_t s = (cudaStream_t)stream;
  DS_CUDA(cudaStreamSynchronize(s));
  DS_CUDA(cudaMemcpyAsync(&h, p, sizeof(h), cudaMemcpyDeviceToHost, s));
  DS_CUDA(cudaMemcpyAsync(p, &zero, sizeof(zero), cudaMemcpyHostToDevice, s));
  DS_CUDA(cudaStreamSynchronize(s));
  return (int)h;
}

const char* ds_strerror(int code) {
  switch (code) {
    case DS_OK: return "ok";
    case DS_EINVAL: return "invalid argument";
    case DS_ECUDA: return "CUDA runtime error";
    case DS_ENOMEM: return "workspace too small";
    case DS_ELIMIT: return "size beyond the built-in scratch of a *_static entry point";
    default: return "unknown error";
  }
}

const char* ds_last_cuda_error(void) { return ds::t_cuda_err; }

int64_t ds_launch_count(void) { return ds::g_launches.load(); }

}  // extern "C"
