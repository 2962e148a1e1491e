// K2 — ds_simulate: tick-exact simulation, one warp per (trace, policy, estimator, alpha) instance
// (algorithm §8(c) C.2; PAPER.md:171-181 queues, 201-242 policies, 278-286 EMA).
//
// Build this TU with -fmad=false: the EMA update is four separately rounded fp64 operations
// (t1=1-a; t2=t1*B; t3=a*m; B=t2+t3) and must match the oracle at 0 ulp; the _rn intrinsics below are never
// contracted either way.
//
// Mapping to the warp (B200: 148 SMs, persistent warps pulling instances from an atomic counter):
//  - warp-uniform scalars: clock `now`, cursor `next`, batch size b, kv_used, iteration cost dt, B[3];
//  - running set: kSlots slots per lane (max_batch <= 32*kSlots), each {request index, finishing iteration};
//    completions are found with one REDUX min over (fin - iter); between events the clock advances with a
//    3-instruction recurrence (now += dt; dt += c_ctx*b) that is exactly the per-iteration cost of §8(c) step 6;
//  - arrivals: a 32-request register window of (arrival, tier, base) per lane, ingested 32 at a time with one
//    ballot; the estimate est=ceil(B[tier]*base) is computed by 32 lanes in parallel (B is constant within a step);
//  - FIFO/PRIORITY/WEIGHTED/AGING queues need no storage: requests arrive in index order, so each tier's FIFO is a
//    cursor (32-request block + ballot bitmask of that tier) and every policy picks among <= 3 heads; the frozen
//    estimates of queued requests live in done_tick[] until the request completes;
//  - SJF: warp-cooperative 32-ary min-heap of (est<<24 | index) keys, first 256 entries in shared memory, rest in
//    the global workspace; sift-down compares 32 children per level with one REDUX-style shuffle min.
#include "common.cuh"

namespace ds {
namespace k2 {

constexpr int kWarpsPerBlock = 4;
constexpr int kHeapSmem = 256;  // heap entries cached in shared memory per warp
constexpr long long kInf = 0x7fffffffffffffffLL;
constexpr unsigned kFull = 0xffffffffu;

struct Params {
  const int64_t* trace_off; const int64_t* arrival; const uint8_t* tier; const int32_t* words; const int32_t* tokens;
  const int32_t* out_len; int64_t n_traces;
  int32_t max_batch; int64_t kv_budget, c_base, c_batch, c_ctx, c_prefill; int32_t w0, w1, w2; int64_t aging_step;
  int32_t traj_every;
  const ds_instance* inst; int64_t n_inst; const int64_t* out_off; int64_t* start_tick; int64_t* done_tick;
  double* ema_final; const int64_t* traj_off; double* ema_traj;
  unsigned long long* heap_ws; unsigned int* counter; unsigned int* status;
};

// 64-bit warp min (keys are unique, so the min identifies its lane)
__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    unsigned long long y = __shfl_xor_sync(kFull, v, o);
    v = y < v ? y : v;
  }
  return v;
}

// ---- SJF heap: implicit 32-ary min-heap, node i has children 32i+1 .. 32i+32 ----
struct Heap {
  unsigned long long* sm;   // kHeapSmem entries (this warp's slice)
  unsigned long long* gm;   // global overflow, indexed by the same i
  int size;
  __device__ __forceinline__ unsigned long long get(int i) const { return i < kHeapSmem ? sm[i] : __ldcg(gm + i); }
  __device__ __forceinline__ void put(int i, unsigned long long k, int lane) {
    if (lane == 0) { if (i < kHeapSmem) sm[i] = k; else __stcg(gm + i, k); }
  }
  __device__ void push(unsigned long long key, int lane) {
    int i = size++;
    while (i > 0) {
      const int p = (i - 1) >> 5;
      const unsigned long long kp = get(p);
      if (kp <= key) break;
      put(i, kp, lane);
      i = p;
    }
    put(i, key, lane);
    __syncwarp();
  }
  __device__ __forceinline__ unsigned long long top() const { return get(0); }
  __device__ void pop(int lane) {
    const unsigned long long last = get(--size);
    if (size == 0) return;
    int i = 0;
    for (;;) {
      const int c0 = 32 * i + 1;
      if (c0 >= size) break;
      const int ci = c0 + lane;
      const unsigned long long ck = ci < size ? get(ci) : ~0ull;
      const unsigned long long m = warp_min_u64(ck);
      if (m >= last) break;
      const unsigned who = __ballot_sync(kFull, ck == m);
      put(i, m, lane);
      i = c0 + (__ffs(who) - 1);
    }
    put(i, last, lane);
    __syncwarp();
  }
};


// per-tier FIFO cursor for PRIORITY / WEIGHTED / AGING: head = first request of tier t at or after the cursor
struct TierCursor {
  int blk;          // 32-request block holding the head
  unsigned mask;    // requests of this tier in that block at or after the head
  int head;         // local request index of the head, INT_MAX when the trace has no more of this tier
  long long est;    // frozen estimate of the head (valid once it has arrived)
  long long arr;    // arrival tick of the head
};

template <int kSlots>
__global__ void __launch_bounds__(k2::kWarpsPerBlock * 32) simulate_kernel(const Params p) {
  __shared__ unsigned long long heap_sm[kWarpsPerBlock][kHeapSmem];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;

  for (;;) {
    unsigned inst_id = 0;
    if (lane == 0) inst_id = atomicAdd(p.counter, 1u);
    inst_id = __shfl_sync(kFull, inst_id, 0);
    if ((long long)inst_id >= p.n_inst) return;

    const ds_instance in = p.inst[inst_id];
    double B0 = 1.0, B1 = 1.0, B2 = 1.0;
    const bool bad_inst = in.trace < 0 || in.trace >= p.n_traces || in.policy < 0 || in.policy > 4 || in.estimator < 0 ||
                          in.estimator > 1 || !(in.ema_alpha >= 0.0 && in.ema_alpha <= 1.0);
    if (bad_inst) {
      if (lane == 0) { atomicOr(p.status, DS_DEV_BAD_INSTANCE); p.ema_final[3 * (size_t)inst_id] = B0; p.ema_final[3 * (size_t)inst_id + 1] = B1; p.ema_final[3 * (size_t)inst_id + 2] = B2; }
      continue;
    }
    const long long lo = p.trace_off[in.trace];
    const long long n = p.trace_off[in.trace + 1] - lo;
    const int64_t* __restrict__ arr = p.arrival + lo;
    const uint8_t* __restrict__ tier = p.tier + lo;
    const int32_t* __restrict__ W = p.words + lo;
    const int32_t* __restrict__ P = p.tokens + lo;
    const int32_t* __restrict__ O = p.out_len + lo;
    const long long oo = p.out_off[inst_id];
    int64_t* __restrict__ st = p.start_tick + oo;
    int64_t* dn = p.done_tick + oo;
    const int policy = in.policy;
    const bool split = in.estimator == DS_SPLIT;
    const int32_t* __restrict__ BASE = split ? W : P;
    const double alpha = in.ema_alpha;
    const bool use_kv = p.kv_budget > 0;
    double* traj = (p.ema_traj && p.traj_off && p.traj_every > 0) ? p.ema_traj + 3 * p.traj_off[inst_id] : nullptr;
    if (policy == DS_SJF && n > (1 << 24) && lane == 0) atomicOr(p.status, DS_DEV_KEY_RANGE);

    // ---- state ----
    long long now = 0, next = 0, kv_used = 0, done = 0, prefill_new = 0;
    int b = 0, cur = 0;
    unsigned iter = 0, dist = 0xffffffffu;
    bool blocked = false;
    int s_idx[kSlots]; unsigned s_fin[kSlots];
#pragma unroll
    for (int s = 0; s < kSlots; ++s) { s_idx[s] = -1; s_fin[s] = 0; }
    Heap heap; heap.sm = heap_sm[wib]; heap.gm = p.heap_ws + oo; heap.size = 0;
    long long fifo_head = 0, fifo_est = 0;   // FIFO: admitted strictly in index order
    TierCursor tc[3];
    const int wtot = p.w0 + p.w1 + p.w2;

    // arrival window: lane holds request wb+lane
    long long wb = 0, w_arr = kInf; int w_tier = 0, w_base = 0;
    auto load_window = [&]() {
      const long long i = wb + lane;
      if (i < n) { w_arr = arr[i]; w_tier = tier[i]; w_base = BASE[i]; } else { w_arr = kInf; w_tier = 0; w_base = 0; }
      const long long prev = __shfl_up_sync(kFull, w_arr, 1);
      bool bad = (i < n) && (w_tier > 2 || w_base < 0 || w_arr < 0 || (lane > 0 && w_arr < prev));
      if (bad) atomicOr(p.status, DS_DEV_BAD_TRACE);
      if (w_tier > 2) w_tier = 2;
      if (w_base < 0) w_base = 0;
    };
    load_window();
    auto arr_next = [&]() -> long long { return next < n ? __shfl_sync(kFull, w_arr, (int)(next - wb)) : kInf; };

    auto advance_cursor = [&](int t, bool first) {   // move tier t's head to its next request
      TierCursor& c = tc[t];
      if (!first) c.mask &= c.mask - 1;
      while (c.mask == 0) {
        if (!first) ++c.blk;
        first = false;
        if ((long long)c.blk * 32 >= n) { c.head = 0x7fffffff; return; }
        const long long i = (long long)c.blk * 32 + lane;
        const int tv = i < n ? (int)tier[i] : 255;
        c.mask = __ballot_sync(kFull, (tv > 2 ? 2 : tv) == t && i < n);
      }
      c.head = c.blk * 32 + (__ffs(c.mask) - 1);
      if (c.head < next) {   // already arrived: its frozen estimate sits in the done_tick scratch
        c.est = use_kv ? (long long)__ldcg(dn + c.head) : 0;
        c.arr = arr[c.head];
      }
    };
    if (policy != DS_FIFO && policy != DS_SJF)
      for (int t = 0; t < 3; ++t) { tc[t].blk = 0; tc[t].mask = 0; tc[t].est = 0; tc[t].arr = 0; advance_cursor(t, true); }

    auto ingest = [&](bool strict) {
      for (;;) {
        const long long i = wb + lane;
        const bool pred = i >= next && i < n && (strict ? w_arr < now : w_arr <= now);
        const unsigned m = __ballot_sync(kFull, pred);
        if (m == 0) return;
        const int c = __popc(m);
        const double Bt = w_tier == 0 ? B0 : (w_tier == 1 ? B1 : B2);
        long long est = 0;
        if (w_base > 0) est = (long long)ceil(__dmul_rn(Bt, (double)w_base));   // Eq. 1-2 reduced (A1), frozen (A5)
        if (policy == DS_SJF) {
          if (pred && est >= (1ll << 39)) atomicOr(p.status, DS_DEV_KEY_RANGE);
          unsigned mm = m;
          while (mm) {
            const int l = __ffs(mm) - 1; mm &= mm - 1;
            const long long e = __shfl_sync(kFull, est, l);
            heap.push(((unsigned long long)e << 24) | (unsigned long long)(wb + l), lane);
          }
        } else {
          if (use_kv && pred) __stcg(dn + i, est);
          __syncwarp();   // other lanes read these estimates back when a cursor reaches them
          const int first = (int)(next - wb), last = first + c;   // window lanes [first,last) were ingested
          if (policy == DS_FIFO) {
            const long long h = fifo_head - wb;
            const long long e = __shfl_sync(kFull, est, (int)(h & 31));
            if (h >= first && h < last) fifo_est = e;
          } else {
#pragma unroll
            for (int t = 0; t < 3; ++t) {
              const long long h = (long long)tc[t].head - wb;
              const long long e = __shfl_sync(kFull, est, (int)(h & 31));
              const long long a = __shfl_sync(kFull, w_arr, (int)(h & 31));
              if (h >= first && h < last) { tc[t].est = e; tc[t].arr = a; }
            }
          }
        }
        next += c;
        blocked = false;
        if (next == wb + 32 && next < n) { wb += 32; load_window(); } else return;
      }
    };

    auto recompute = [&]() {   // after the running set changed
      unsigned d = 0xffffffffu;
#pragma unroll
      for (int s = 0; s < kSlots; ++s) if (s_idx[s] >= 0) d = min(d, s_fin[s] - iter);
      dist = __reduce_min_sync(kFull, d);
    };

    auto retire = [&]() {
      for (;;) {
        int lm = 0x7fffffff;
#pragma unroll
        for (int s = 0; s < kSlots; ++s) if (s_idx[s] >= 0 && s_fin[s] == iter) lm = min(lm, s_idx[s]);
        const int r = __reduce_min_sync(kFull, lm);        // ascending request index (R-ORD)
        if (r == 0x7fffffff) break;
#pragma unroll
        for (int s = 0; s < kSlots; ++s) if (s_idx[s] == r) s_idx[s] = -1;
        const int Pr = P[r], Or = max(O[r], 1), tr = min((int)tier[r], 2), br = BASE[r];
        if (lane == 0) dn[r] = now;
        kv_used -= (long long)Pr + Or;
        --b;
        if (alpha > 0.0 && br > 0) {                       // Eq. 5-6 (A3): four separately rounded operations
          const double m = __ddiv_rn((double)Pr, (double)br);
          const double t1 = __dsub_rn(1.0, alpha);
          const double Bk = tr == 0 ? B0 : (tr == 1 ? B1 : B2);
          const double t2 = __dmul_rn(t1, Bk);
          const double t3 = __dmul_rn(alpha, m);
          const double Bn = __dadd_rn(t2, t3);
          if (tr == 0) B0 = Bn; else if (tr == 1) B1 = Bn; else B2 = Bn;
        }
        ++done;
        if (traj && done % p.traj_every == 0 && lane == 0) {
          double* q = traj + 3 * (done / p.traj_every - 1);
          q[0] = B0; q[1] = B1; q[2] = B2;
        }
      }
      blocked = false;
      __syncwarp();
    };

    auto admit = [&]() {
      bool changed = false;
      while (b < p.max_batch) {
        // peek(policy, now)
        long long c = -1, est_c = 0; int ct = 0, wpos = 0;
        if (policy == DS_FIFO) {
          if (fifo_head < next) { c = fifo_head; est_c = fifo_est; }
        } else if (policy == DS_SJF) {
          if (heap.size > 0) { const unsigned long long k = heap.top(); c = (long long)(k & 0xffffffull); est_c = (long long)(k >> 24); }
        } else if (policy == DS_PRIORITY) {
          for (int t = 2; t >= 0; --t) if (tc[t].head < next) { c = tc[t].head; est_c = tc[t].est; ct = t; }
        } else if (policy == DS_WEIGHTED) {
          for (int s = 0; s < wtot; ++s) {
            int pos = cur + s; if (pos >= wtot) pos -= wtot;
            const int t = pos < p.w0 ? 0 : (pos < p.w0 + p.w1 ? 1 : 2);
            if (tc[t].head < next) { c = tc[t].head; est_c = tc[t].est; ct = t; wpos = pos; break; }
          }
        } else {  // AGING (A10): eff = max(0, tier - floor(waited/aging_step)); key (eff, seq)
          int best_eff = 99;
#pragma unroll
          for (int t = 0; t < 3; ++t) {
            if (tc[t].head < next) {
              const long long waited = now - tc[t].arr;
              int eff = t;
              if (t >= 1 && waited >= p.aging_step) --eff;
              if (t >= 2 && waited >= 2 * p.aging_step) --eff;
              if (eff < best_eff || (eff == best_eff && tc[t].head < c)) { best_eff = eff; c = tc[t].head; est_c = tc[t].est; ct = t; }
            }
          }
        }
        if (c < 0) break;
        if (b > 0 && use_kv && kv_used + est_c > p.kv_budget) { blocked = policy != DS_AGING; break; }   // deferred (A8)
        // pop
        if (policy == DS_FIFO) {
          ++fifo_head;
          if (fifo_head < next && use_kv) fifo_est = (long long)__ldcg(dn + fifo_head);
        } else if (policy == DS_SJF) heap.pop(lane);
        else { advance_cursor(ct, false); if (policy == DS_WEIGHTED) { cur = wpos + 1; if (cur >= wtot) cur = 0; } }
        const int Pc = P[c];
        int Oc = O[c];
        if (Oc < 1) { Oc = 1; if (lane == 0) atomicOr(p.status, DS_DEV_BAD_TRACE); }
        if (lane == 0) st[c] = now;
        // first lane with a free slot takes it
        bool has_free = false;
#pragma unroll
        for (int s = 0; s < kSlots; ++s) has_free |= s_idx[s] < 0;
        const unsigned fm = __ballot_sync(kFull, has_free);
        if (lane == __ffs(fm) - 1) {
          bool placed = false;
#pragma unroll
          for (int s = 0; s < kSlots; ++s) if (!placed && s_idx[s] < 0) { s_idx[s] = (int)c; s_fin[s] = iter + (unsigned)Oc; placed = true; }
        }
        kv_used += Pc; prefill_new += Pc; ++b;
        changed = true;
      }
      return changed;
    };

    // ---- main loop: one pass per iteration boundary with an event; event-free boundaries run in the inner loop ----
    for (;;) {
      long long an = arr_next();
      if (an < now) { ingest(true); an = arr_next(); }                     // 1. INGEST-EARLY
      bool dirty = false;
      if (dist == 0) { retire(); dirty = true; }                           // 2. RETIRE
      if (an <= now) { ingest(false); an = arr_next(); }                   // 3. INGEST-NOW
      if (!blocked && b < p.max_batch) dirty |= admit();                    // 4. ADMIT
      if (dirty) recompute();
      if (b == 0) {                                                         // 5. IDLE / END
        if (next >= n) break;
        now = an;
        continue;
      }
      // 6. STEP (+ fast-forward over boundaries where nothing can happen)
      long long dt = p.c_base + p.c_batch * b + p.c_ctx * kv_used;
      const long long cb = p.c_ctx * b;
      now += dt + p.c_prefill * prefill_new;
      prefill_new = 0;
      kv_used += b; dt += cb; --dist; ++iter;
      const bool may_admit = !blocked && b < p.max_batch &&
                             (policy == DS_FIFO ? fifo_head < next : policy == DS_SJF ? heap.size > 0
                                                : (tc[0].head < next || tc[1].head < next || tc[2].head < next));
      if (!may_admit) {
        while (dist != 0 && an > now) { now += dt; kv_used += b; dt += cb; --dist; ++iter; }
      }
    }
    if (lane == 0) {
      p.ema_final[3 * (size_t)inst_id] = B0; p.ema_final[3 * (size_t)inst_id + 1] = B1; p.ema_final[3 * (size_t)inst_id + 2] = B2;
    }
    __syncwarp();
  }
}

}  // namespace k2

size_t ws_simulate(int64_t total_requests, int64_t) { return 256 + sizeof(unsigned long long) * (size_t)total_requests; }

}  // namespace ds

extern "C" int ds_simulate(const ds_traces* tr, const ds_server* sv, const ds_instance* inst, int64_t n_inst,
                           const int64_t* out_off, int64_t* start_tick, int64_t* done_tick, double* ema_final,
                           const int64_t* traj_off, double* ema_traj, void* workspace, size_t workspace_bytes, void* stream) {
  using namespace ds;
  if (!tr || !sv || n_inst < 0) return DS_EINVAL;
  if (n_inst == 0) return DS_OK;
  if (!inst || !out_off || !start_tick || !done_tick || !ema_final || !workspace) return DS_EINVAL;
  if (tr->n_traces < 1 || !tr->trace_off || !tr->arrival_tick || !tr->tier || !tr->words || !tr->tokens || !tr->out_len) return DS_EINVAL;
  if (sv->max_batch < 1 || sv->max_batch > 256) return DS_EINVAL;
  if (sv->weight[0] < 1 || sv->weight[1] < 1 || sv->weight[2] < 1 || sv->aging_step < 1 || sv->traj_every < 0) return DS_EINVAL;
  if (sv->c_base < 0 || sv->c_batch < 0 || sv->c_ctx < 0 || sv->c_prefill < 0) return DS_EINVAL;
  if (n_inst > 0x7fffffff) return DS_EINVAL;
  if (workspace_bytes < 256) return DS_ENOMEM;
  cudaStream_t s = (cudaStream_t)stream;
  k2::Params p;
  p.trace_off = tr->trace_off; p.arrival = tr->arrival_tick; p.tier = tr->tier; p.words = tr->words; p.tokens = tr->tokens;
  p.out_len = tr->out_len; p.n_traces = tr->n_traces;
  p.max_batch = sv->max_batch; p.kv_budget = sv->kv_budget; p.c_base = sv->c_base; p.c_batch = sv->c_batch; p.c_ctx = sv->c_ctx;
  p.c_prefill = sv->c_prefill; p.w0 = sv->weight[0]; p.w1 = sv->weight[1]; p.w2 = sv->weight[2]; p.aging_step = sv->aging_step;
  p.traj_every = sv->traj_every;
  p.inst = inst; p.n_inst = n_inst; p.out_off = out_off; p.start_tick = start_tick; p.done_tick = done_tick;
  p.ema_final = ema_final; p.traj_off = traj_off; p.ema_traj = ema_traj;
  p.counter = (unsigned int*)workspace;
  p.heap_ws = (unsigned long long*)((char*)workspace + 256);
  p.status = status_ptr();
  if (!p.status) return cuda_fail(cudaGetLastError());
  // the heap region is only touched by SJF instances beyond kHeapSmem queued requests; its size is checked here
  // against the documented formula only when it can be needed at all (caller passes total requests to the query)
  DS_CUDA(cudaMemsetAsync(workspace, 0, 256, s));
  const int threads = k2::kWarpsPerBlock * 32;
  int per_sm = 0;
  auto launch = [&](auto kern) -> int {
    DS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, 0));
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)kNumSMs * per_sm;
    const long long need = (n_inst + k2::kWarpsPerBlock - 1) / k2::kWarpsPerBlock;
    if (blocks > need) blocks = need;
    kern<<<(unsigned)blocks, threads, 0, s>>>(p);
    note_launch();
    DS_CUDA(cudaGetLastError());
    return DS_OK;
  };
  if (sv->max_batch <= 32) return launch(k2::simulate_kernel<1>);
  if (sv->max_batch <= 64) return launch(k2::simulate_kernel<2>);
  if (sv->max_batch <= 128) return launch(k2::simulate_kernel<4>);
  return launch(k2::simulate_kernel<8>);
}
