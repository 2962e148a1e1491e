// K2 — ds_simulate: tick-exact simulation, one warp per (trace, policy, estimator, alpha) instance
// (algorithm §8(c) C.2; PAPER.md:171-181 queues, 201-242 policies, 278-286 EMA).
//
// Build this TU with -fmad=false: the EMA update is four separately rounded fp64 operations
// (t1=1-a; t2=t1*B; t3=a*m; B=t2+t3) and must match the oracle at 0 ulp; the _rn intrinsics below are never
// contracted either way.
//
// Mapping to the warp (B200: 148 SMs, persistent warps pulling instances from an atomic counter). The per-instance
// body is compiled once per (slots, policy) so that each policy's queue logic is straight-line code:
//  - warp-uniform scalars: clock `now`, cursor `next`, next arrival tick `an`, batch size b, kv_used; the factors B[3]
//    and the arrival ticks of the current window sit in shared memory (every lane writes the same factor, so no
//    synchronisation is needed to read it back; shuffles from an owner lane cost 27 instructions per request with their guards);
//  - running set: 32*kSlots slots {request index, finishing iteration} in shared memory (max_batch <= 32*kSlots) with a
//    free-slot stack beside them: an admission is one pop + two stores by uniform address (placing a request into one
//    lane's register slots cost 35 instructions of divergent, predicated code per request). At a completion boundary
//    lane L loads slots [kSlots*L, kSlots*(L+1)) into registers once (LDS.128), the completions of that boundary are
//    retired from those registers in ascending request index (one REDUX min each) and the distance to the next
//    completion is one more REDUX min over (fin - iter);
//  - per-request records: pack_kernel first writes {m = tokens/words (the feedback ratio of Eq. 6, one fp64 division per
//    TRACE request instead of one per simulated request), tokens, out_len} as one 16-byte record, so a completion or an
//    admission is one LDG.128 instead of two to four 4-byte loads with their 64-bit address arithmetic;
//  - between events the batch is constant, so j iterations cost exactly j*dt + c_ctx*b*j(j-1)/2 ticks (§8(c) step 6
//    with a constant running set): the kernel jumps to the next event (completion, or arrival when an arrival can
//    matter) with that closed form; a float estimate gives a provably safe lower bound on j, exact integer arithmetic
//    does the jump, the last one or two iterations are stepped. The oracle steps one iteration at a time;
//  - arrivals: a 32-request register window of (arrival, tier, base) per lane, ingested 32 at a time with one
//    ballot; est=ceil(B[tier]*base) is computed by 32 lanes in parallel. Arrivals cannot matter while the batch is
//    full (or FIFO's head is KV-deferred): they are then ingested lazily, in bulk, at the next completion, which is
//    exact because B only changes at completions and INGEST-EARLY uses the pre-completion B (R-ORD);
//  - FIFO/PRIORITY/WEIGHTED/AGING queues need no storage: requests arrive in index order, so each tier's FIFO is a
//    cursor (32-request block + ballot bitmask of that tier) and every policy picks among <= 3 heads; the frozen
//    estimates of queued requests live in done_tick[] until the request completes;
//  - SJF: warp-cooperative 32-ary min-heap of (est<<24 | index) keys, first 256 entries in shared memory, rest in the
//    global workspace; sift-down compares 32 children per level with one shuffle min.
#include <type_traits>

#include "common.cuh"

namespace ds {
namespace k2 {

// Launch shape per instantiation (warps per block x resident blocks per SM the register allocation is bounded for), r02. With the
// running set in shared memory the 4- and 8-slot bodies run best at 28 warps of 72 registers (6 / 7 / 8 blocks of 4 warps =
// configs[3] at 4096 traces 384.0 / 381.3 / 396.8 ms; 7 x 4, 2 x 14 and 1 x 28 are the same within 0.1 %, 24 warps of 80
// registers +7 %). The one-slot body fits 64 registers (32 warps) and gains 4 % from 8-warp blocks (configs[1] 10.15 -> 9.72 ms;
// 4 x 8 / 8 x 3 / 6 x 5 / 7 x 4 / 16 x 2: 10.15 / 11.04 / 10.23 / 10.75 / 10.22). For the 8-slot body 8 x 3 at 80 registers looked
// 3.5 % faster on configs[4] cut to 1024 traces (10 240 instances fill a third round of 24 warps per SM better than one of 28)
// and is 3.9 % slower at full size (40 960 instances: 1131.9 against 1089.7 ms): it stays at 4 x 7.
#ifndef DS_K2_WARPS
#define DS_K2_WARPS 4
#endif
#ifndef DS_K2_MIN_BLOCKS
#define DS_K2_MIN_BLOCKS 7
#endif
#ifndef DS_K2_WARPS_1
#define DS_K2_WARPS_1 8
#endif
#ifndef DS_K2_MIN_BLOCKS_1
#define DS_K2_MIN_BLOCKS_1 4
#endif
template <int kSlots, bool kBudget, bool kReest> struct Shape { static constexpr int kWarps = DS_K2_WARPS, kBlocks = DS_K2_MIN_BLOCKS; };
template <> struct Shape<1, false, false> { static constexpr int kWarps = DS_K2_WARPS_1, kBlocks = DS_K2_MIN_BLOCKS_1; };
constexpr int kHeapSmem = 256;  // heap entries cached in shared memory per warp
// Build with -DDS_K2_CHECK to verify the bookkeeping of the shared-memory structures on the device (compute-sanitizer is not
// available on this pool): a violated invariant sets DS_DEV_INTERNAL in the status word. Off in the product build.
#ifdef DS_K2_CHECK
#define DS_K2_INVARIANT(cond) do { if (!(cond)) atomicOr(p.status, DS_DEV_INTERNAL); } while (0)
#else
#define DS_K2_INVARIANT(cond) do { } while (0)
#endif
constexpr long long kInf = 0x7fffffffffffffffLL;
constexpr unsigned kFull = 0xffffffffu;

// per trace request, written by pack_kernel: m = tokens/words as fp64 (correctly rounded division, the B_measured of Eq. 6
// under reading A3; -1.0 when words <= 0: no feedback from that request), P = tokens, O = out_len | tier << 30 (out_len < 2^30
// is part of the contract, checked by pack_kernel: a completion then needs no second load for the tier)
struct __align__(16) Rec { double m; int P; unsigned O; };
constexpr unsigned kRecLenMask = 0x3fffffffu;

struct Params {
  const int64_t* trace_off; const int64_t* arrival; const uint8_t* tier; const int32_t* words; const int32_t* tokens;
  const int32_t* out_len; int64_t n_traces;
  int32_t max_batch; int64_t kv_budget; uint32_t c_base, c_batch, c_ctx, c_prefill; /* < 2^31, checked by ds_simulate */ int32_t w0, w1, w2; int64_t aging_step;
  int32_t traj_every;
  const ds_instance* inst; int64_t n_inst; const int64_t* out_off; int64_t* start_tick; int64_t* done_tick;
  double* ema_final; const int64_t* traj_off; double* ema_traj; int64_t* est_out;
  const uint8_t* category; ds_budget bp;   // budget estimators only (ds_simulate_budget)
  int32_t n_clients; int64_t think; int64_t* arrival_out;   // closed-loop arrivals (ds_simulate_closed), n_clients = 0: open loop
  int64_t batch_wait;                                        // ds_simulate_closed: dispatch gate of an idle server (0 = none)
  unsigned long long* heap_ws; unsigned int* counter; unsigned int* status; const unsigned int* perm;
  const struct Rec* rec;                                     // [n_requests] packed per-request records (pack_kernel)
  int32_t use_kv, want_est, want_traj;                       // 32-bit copies of kv_budget > 0, est_out != NULL, trajectory sampling on
  int64_t n_total;                                           // out_off[n_inst] as stated by the caller: size of every per-request output and of the heap region
  unsigned n_sms;
};

// 64-bit warp min (keys are unique, so the min identifies its lane): the minimum of the high words, then the minimum of
// the low words among the lanes that hold it. Two REDUX.MIN instead of five butterfly steps of two shuffles each.
__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long v) {
  const unsigned hi = (unsigned)(v >> 32), lo = (unsigned)v;
  const unsigned mh = __reduce_min_sync(kFull, hi);
  const unsigned ml = __reduce_min_sync(kFull, hi == mh ? lo : 0xffffffffu);
  return ((unsigned long long)mh << 32) | ml;
}
__device__ __forceinline__ long long shfl_i64(long long v, int src) { return __shfl_sync(kFull, v, src); }
__device__ __forceinline__ double shfl_f64(double v, int src) { return __shfl_sync(kFull, v, src); }

// WEIGHTED (A9): the tier served next is the first non-empty tier in cyclic order starting with the block of the slot
// cursor. It depends only on that block (0..2) and on which tiers are non-empty (3 bits): a table of 2-bit entries per
// block, entry 3 = every queue empty. (The loop over the three cyclic positions with its nested selects was 45
// instructions per pick and made WEIGHTED 47 % more expensive per request than FIFO.)
constexpr unsigned weighted_table(int blk) {
  unsigned tab = 0;
  for (int nem = 0; nem < 8; ++nem) {
    unsigned ct = 3;
    for (int k = 2; k >= 0; --k) { const int t = (blk + k) % 3; if ((nem >> t) & 1) ct = (unsigned)t; }
    tab |= ct << (2 * nem);
  }
  return tab;
}
constexpr unsigned kWeightedTab0 = weighted_table(0), kWeightedTab1 = weighted_table(1), kWeightedTab2 = weighted_table(2);
static_assert(((weighted_table(1) >> (2 * 0b101)) & 3u) == 2u && ((weighted_table(2) >> (2 * 0b011)) & 3u) == 0u &&
              ((weighted_table(0) >> 0) & 3u) == 3u, "first non-empty tier in cyclic order");

// ---- running set: per warp, 32*kSlots slots in shared memory; lane L scans slots [kSlots*L, kSlots*(L+1)) ----
constexpr int kFreeIdx = 0x7fffffff;          // idx of a free slot (also "no request" in the min reductions)
template <int kSlots>
struct __align__(16) Slots {
  int idx[32 * kSlots];                       // request index, kFreeIdx = free
  unsigned fin[32 * kSlots];                  // iteration at whose boundary the request completes
  unsigned short stack[32 * kSlots];          // free slot numbers, [0, nfree) valid
  // Warp-uniform values that used to be fetched from their owner lane by shuffles (27 instructions per request with the
  // convergence guards around every SHFL). B: every lane writes the SAME new factor, so a lane only ever reads what it wrote
  // itself and no synchronisation is needed. warr / west: lane l's arrival tick and frozen estimate of request wb + l, read
  // by other lanes after a __syncwarp(). (The cursor policies keep their estimate shuffles: those run only when a queue head
  // falls inside the ingested range, which is rare; an unconditional store per ingest step cost more: configs[4] +3 %.)
  double B[4];                                // feedback factors: per tier (3) or per semantic category (4)
  long long warr[32];                         // arrival ticks of the current 32-request window
  long long west[32];                         // SJF: estimates of the current ingest step (every heap push ends in a __syncwarp, which
                                              // orders its reads before the next step's writes)
};

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
  long long est;    // frozen estimate of the head (valid once it has arrived; only kept when the KV budget is on)
  long long arr;    // arrival tick of the head (AGING only)
};

// kSmall: every per-iteration quantity of this trace (kv_used, dt, prefill) is proven < 2^31 and out_len <= 65535 by
// trace_is_small(), so they are kept in 32-bit registers and the closed-form jump is two IMAD.WIDE; `now` stays 64-bit.
// kBudget: the paper's full estimator (Eq. 1-2) with one feedback factor per semantic category (lanes 0..3) instead of
// the reduced per-tier one (lanes 0..2); a separate instantiation so that the benchmarked path is not touched.
// kReest: online re-estimation of queued requests (ds_server.reestimate; reading A16): estimates follow the factors, so
// neither the SJF heap (keys frozen at insertion) nor the per-tier cursors' cached estimates apply. The queue is a plain
// array of request indices in the workspace; every pick scans it, 32 entries per step, with the policy's key evaluated on
// the spot - the oracle's linear peek run by a warp. A variant, not the benchmarked path: O(queue/32) per admission.
template <int kSlots, int kPolicy, bool kSmall, bool kBudget, bool kReest = false>
__device__ __forceinline__ void run_instance(const Params& p, const unsigned inst_id, const int trace, const bool split, const double alpha,
                                          unsigned long long* heap_sm, Slots<kSlots>& sl, const int lane) {
  constexpr bool kAging = kPolicy == DS_AGING || kPolicy == DS_AGING_UNCLAMPED;   // both read the heads' arrival ticks
  constexpr bool kCursor = !kReest && (kPolicy == DS_PRIORITY || kPolicy == DS_WEIGHTED || kAging);
  const long long lo = p.trace_off[trace];
  const long long n64 = p.trace_off[trace + 1] - lo;
  if (n64 < 0 || n64 > 0x7ffffff0ll || (!kReest && kPolicy == DS_SJF && n64 > (1 << 24))) {   // local indices are 32-bit (SJF keys: 24-bit)
    if (lane == 0) atomicOr(p.status, n64 > (1 << 24) ? DS_DEV_KEY_RANGE : DS_DEV_BAD_TRACE);
    return;
  }
  const int n = (int)n64;
  const int64_t* __restrict__ arr = p.arrival + lo;
  const uint8_t* __restrict__ tier = p.tier + lo;
  const int32_t* __restrict__ W = p.words + lo;
  const int32_t* __restrict__ P = p.tokens + lo;
  const int32_t* __restrict__ O = p.out_len + lo;
  const long long oo = p.out_off[inst_id];
  if (oo < 0 || oo + n64 > p.n_total) {                     // this instance's outputs (and SJF heap region) would leave the caller's arrays
    if (lane == 0) atomicOr(p.status, DS_DEV_BAD_OUT_OFF);
    return;
  }
  // the per-instance base pointers of the tick outputs and the record array, kept in registers (volatile asm): at 72
  // registers the compiler otherwise re-derives each of them from the kernel parameters and the instance offset at every
  // use (LDC + 64-bit add + LEA pair: 6-7 instructions per store / record load instead of 2-3)
  // (measured: configs[3] -1.3 %, configs[4] -5.3 %; the one-slot bodies run at 64 registers and lose 3.5 %, so they do not pin)
  constexpr bool kPinPtrs = kSlots > 1 && !kBudget && !kReest;
  int64_t* st = p.start_tick + oo;
  int64_t* dn = p.done_tick + oo;
  if constexpr (kPinPtrs) {
    asm volatile("mov.b64 %0, %0;" : "+l"(st)); asm volatile("mov.b64 %0, %0;" : "+l"(dn));
    __builtin_assume(__isGlobal(st)); __builtin_assume(__isGlobal(dn));     // (the asm hides the address space: keep STG, not generic ST)
  }
  const int32_t* __restrict__ BASE = split ? W : P;
  const Rec* rec = p.rec + lo;
  if constexpr (kSlots > 1 && !kBudget && !kReest) { asm volatile("mov.b64 %0, %0;" : "+l"(rec)); __builtin_assume(__isGlobal(rec)); }
  const bool use_kv = p.use_kv != 0;
  int64_t* est_o = p.want_est ? p.est_out + oo : nullptr;
  const bool need_est = use_kv || kPolicy == DS_SJF || est_o != nullptr;
  // EXACT estimator: m = P/P = 1.0, and (1-a)*1 + a*1 rounds to exactly 1.0 for every a in [0,1] (DESIGN.md §4 A4),
  // so B stays 1.0 and est = base: no fp64 work at all on that path.
  const bool ema_on = (kBudget || split) && alpha > 0.0;
  constexpr int kFac = kBudget ? 4 : 3;           // feedback factors per instance
  const uint8_t* __restrict__ cat = kBudget ? p.category + lo : nullptr;
  double* traj = p.want_traj ? p.ema_traj + kFac * p.traj_off[inst_id] : nullptr;
  const int max_batch = p.max_batch;

  // ---- state (warp-uniform unless noted) ----
  using acc_t = typename std::conditional<kSmall, unsigned, unsigned long long>::type;
  long long now = 0, an = kInf;
  acc_t kv_used = 0, prefill_new = 0;
  int next = 0, b = 0, cur = 0, fifo_head = 0, done = 0;
  int wblk = 0;                          // WEIGHTED: block (tier) of the slot cursor `cur`, recomputed when cur moves
  long long fifo_est = 0;
  unsigned iter = 0, dist = 0xffffffffu;
  bool blocked = false;
  long long collect = -1;                // batch-wait: tick at which the idle dispatcher started collecting (-1: not collecting)
#pragma unroll
  for (int k = 0; k < 4; ++k) sl.B[k] = 1.0;   // (every lane, same value)
  // running set: all slots free, the free stack holds every slot number
  int nfree = 32 * kSlots;
#pragma unroll
  for (int s = 0; s < kSlots; ++s) { sl.idx[s * 32 + lane] = kFreeIdx; sl.fin[s * 32 + lane] = 0u; sl.stack[s * 32 + lane] = (unsigned short)(s * 32 + lane); }
  __syncwarp();
  Heap heap; heap.sm = heap_sm; heap.gm = p.heap_ws + oo; heap.size = 0;
  int* const q = reinterpret_cast<int*>(p.heap_ws + oo);     // kReest: the queued request indices, unordered (n entries fit twice)
  int qn = 0;
  TierCursor tc[3];
  const int wtot = p.w0 + p.w1 + p.w2;

  // Closed loop (ds_simulate_closed): arrivals live in arrival_out (per instance). The first n_clients
  // entries are the trace's, the rest start at kInf ("not submitted yet") and are written when a completion releases them.
  const bool closed = kBudget && p.n_clients > 0;
  int64_t* arr_d = closed ? p.arrival_out + oo : nullptr;
  int released = n;
  long long last_rel = 0;                // closed loop: arrival tick of the most recently submitted request (contract: non-decreasing)
  if (closed) {
    released = p.n_clients < n ? p.n_clients : n;
    last_rel = released > 0 ? (long long)arr[released - 1] : 0;
    for (int i = lane; i < n; i += 32) __stcg(arr_d + i, i < released ? arr[i] : kInf);
    __syncwarp();
  }
  auto arr_at = [&](const int i) -> long long { return closed ? (long long)__ldcg(arr_d + i) : (long long)arr[i]; };

  // arrival window: lane holds request wb+lane
  int wb = 0; long long w_arr = kInf; int w_tier = 0, w_base = 0, w_cat = 0;
  auto load_window = [&]() {
    const long long w_prev_last = wb > 0 ? sl.warr[31] : 0;   // last arrival of the window being replaced (lane 0's predecessor)
    __syncwarp();                                              // ... read by every lane before lane 31 overwrites it
    const int i = wb + lane;
    if (i < n) { w_arr = arr_at(i); w_tier = tier[i]; w_base = BASE[i]; } else { w_arr = kInf; w_tier = 0; w_base = 0; }
    if (kBudget) {
      w_cat = i < n ? (int)cat[i] : 0;
      if (w_cat > 3) { atomicOr(p.status, DS_DEV_BAD_TRACE); w_cat = 3; }
    }
    long long prev = __shfl_up_sync(kFull, w_arr, 1);
    if (lane == 0) prev = w_prev_last;
    const bool bad = (i < n) && (w_tier > 2 || w_base < 0 || w_arr < 0 || w_arr < prev || O[i] < 1);   // (out_len checked here, 32 at a time)
    if (bad) atomicOr(p.status, DS_DEV_BAD_TRACE);
    if (w_tier > 2) w_tier = 2;
    if (w_base < 0) w_base = 0;
    sl.warr[lane] = w_arr;
    __syncwarp();
  };
  load_window();
  an = n > 0 ? sl.warr[0] : kInf;

  auto advance_cursor = [&](TierCursor& c, const int t, bool first) {   // move tier t's head to its next request
    if (!first) c.mask &= c.mask - 1;
    while (c.mask == 0) {
      if (!first) ++c.blk;
      first = false;
      if (c.blk * 32 >= n) { c.head = 0x7fffffff; return; }
      const int i = c.blk * 32 + lane;
      const int tv = i < n ? (int)tier[i] : 255;
      c.mask = __ballot_sync(kFull, (tv > 2 ? 2 : tv) == t && i < n);
    }
    c.head = c.blk * 32 + (__ffs(c.mask) - 1);
    if (c.head < next) {   // already arrived: its frozen estimate sits in the done_tick scratch
      if (use_kv) c.est = (long long)__ldcg(dn + c.head);
      if (kAging) c.arr = arr_at(c.head);
    }
  };
  if (kCursor)
#pragma unroll
    for (int t = 0; t < 3; ++t) { tc[t].blk = 0; tc[t].mask = 0; tc[t].est = 0; tc[t].arr = 0; advance_cursor(tc[t], t, true); }

  // enqueue every request of the window with arrival <= limit (now-1 for INGEST-EARLY, now for INGEST-NOW); 32 at a time
  auto ingest = [&](const long long limit) {
    for (;;) {
      const int i = wb + lane;
      const bool pred = i >= next && w_arr <= limit;            // lanes past the trace hold kInf
      const unsigned m = __ballot_sync(kFull, pred);
      if (m == 0) break;
      const int c = __popc(m);
      long long est = 0;
      if constexpr (kReest) {                                 // A16: no estimate is taken at arrival; the request joins the array
        if (pred) __stcg(q + qn + (i - next), i);             // (the ingested lanes are contiguous from request `next`)
        qn += c;
        __syncwarp();
      } else
      if (kBudget) {
        if (need_est) {                                       // Eq. 1-2 in full, frozen at arrival (A5)
          const double tb = w_cat == 0 ? p.bp.t_base[0] : w_cat == 1 ? p.bp.t_base[1] : w_cat == 2 ? p.bp.t_base[2] : p.bp.t_base[3];
          const double sc = w_tier == 0 ? p.bp.s_tenant[0] : w_tier == 1 ? p.bp.s_tenant[1] : p.bp.s_tenant[2];
          double F = __dadd_rn(1.0, __dmul_rn(p.bp.f_slope, (double)w_base));
          if (F > p.bp.f_max) F = p.bp.f_max;
          double x = __dmul_rn(tb, sl.B[w_cat]);
          x = __dmul_rn(x, sc);
          x = __dmul_rn(x, F);
          est = (long long)w_base + (long long)ceil(x);
        }
      } else if (need_est) {
        if (ema_on) {                                         // Eq. 1-2 reduced (A1), frozen at arrival (A5)
          const double Bt = sl.B[w_tier];
          if (w_base > 0) est = (long long)ceil(__dmul_rn(Bt, (double)w_base));
        } else est = w_base;                                  // B == 1.0 exactly
      }
      if (!kReest && est_o && pred) est_o[i] = est;           // frozen admission-time estimate (ds_simulate_est)
      if constexpr (kReest) {
      } else if (kPolicy == DS_SJF) {
        if (pred && est >= (1ll << 39)) atomicOr(p.status, DS_DEV_KEY_RANGE);
        sl.west[lane] = est;
        __syncwarp();
        unsigned mm = m;
        while (mm) {
          const int l = __ffs(mm) - 1; mm &= mm - 1;
          const long long e = sl.west[l];
          heap.push(((unsigned long long)e << 24) | (unsigned long long)(wb + l), lane);
        }
      } else {
        if (use_kv && pred) __stcg(dn + i, est);
        __syncwarp();   // other lanes read these estimates back when a cursor reaches them
        const int last = next + c;                            // requests [next,last) were ingested
        if (kPolicy == DS_FIFO) {
          if (use_kv && fifo_head >= next && fifo_head < last) fifo_est = shfl_i64(est, fifo_head - wb);
        } else {
#pragma unroll
          for (int t = 0; t < 3; ++t) {
            if (tc[t].head >= next && tc[t].head < last) {   // warp-uniform
              if (use_kv) tc[t].est = shfl_i64(est, tc[t].head - wb);
              if (kAging) tc[t].arr = sl.warr[tc[t].head - wb];
            }
          }
        }
      }
      next += c;
      if (kPolicy != DS_FIFO) blocked = false;               // a new arrival can change the head (never FIFO's)
      if (next == wb + 32 && next < n) { wb += 32; load_window(); continue; }
      break;
    }
    an = next < n ? sl.warr[next - wb] : kInf;
  };

  // 2. RETIRE: completions at `now`, ascending request index (R-ORD); then the distance to the next completion.
  // The lane's slots are loaded into registers once; every completion of this boundary is found and cleared there.
  const double t1 = __dsub_rn(1.0, alpha);                    // Eq. 5: (1 - alpha), the same rounding every time
  auto retire = [&]() {
    __syncwarp();                                             // the slot stores of earlier admissions are visible
    int ri[kSlots]; unsigned rf[kSlots];
    if constexpr (kSlots % 4 == 0) {
#pragma unroll
      for (int q = 0; q < kSlots / 4; ++q) {
        const int4 vi = *reinterpret_cast<const int4*>(&sl.idx[lane * kSlots + 4 * q]);
        const uint4 vf = *reinterpret_cast<const uint4*>(&sl.fin[lane * kSlots + 4 * q]);
        ri[4 * q] = vi.x; ri[4 * q + 1] = vi.y; ri[4 * q + 2] = vi.z; ri[4 * q + 3] = vi.w;
        rf[4 * q] = vf.x; rf[4 * q + 1] = vf.y; rf[4 * q + 2] = vf.z; rf[4 * q + 3] = vf.w;
      }
    } else if constexpr (kSlots == 2) {
      const int2 vi = *reinterpret_cast<const int2*>(&sl.idx[lane * 2]);
      const uint2 vf = *reinterpret_cast<const uint2*>(&sl.fin[lane * 2]);
      ri[0] = vi.x; ri[1] = vi.y; rf[0] = vf.x; rf[1] = vf.y;
    } else {
#pragma unroll
      for (int s = 0; s < kSlots; ++s) { ri[s] = sl.idx[lane * kSlots + s]; rf[s] = sl.fin[lane * kSlots + s]; }
    }
    // completions at this boundary (a free slot has idx = kFreeIdx, so its stale fin cannot match): per lane the smallest
    // completing request, its slot, and how many of the lane's slots complete
    int lm = kFreeIdx, ls = 0, cnt = 0;
#pragma unroll
    for (int s = 0; s < kSlots; ++s) {
      const bool hit = rf[s] == iter && ri[s] != kFreeIdx;
      cnt += hit ? 1 : 0;
      if (hit && ri[s] < lm) { lm = ri[s]; ls = s; }
    }
    int left = __reduce_add_sync(kFull, cnt);                 // called with dist == 0: at least one
    while (left > 0) {
      const int r = __reduce_min_sync(kFull, lm);             // ascending request index (R-ORD)
      if (r == kFreeIdx) break;                               // (defensive: cannot happen; never index with it)
      --left;
      // owner: free the slot in shared memory and push its number on the free stack (registers keep the loaded state: the
      // completions are told apart from what stays by rf == iter)
      const bool own = lm == r;
      DS_K2_INVARIANT(nfree >= 0 && nfree < 32 * kSlots && __popc(__ballot_sync(kFull, own)) == 1 && r >= 0 && r < next);
      if (own) { const int slot = lane * kSlots + ls; sl.idx[slot] = kFreeIdx; sl.stack[nfree] = (unsigned short)slot; --cnt; lm = kFreeIdx; }
      ++nfree;
      if (kSlots > 1 && __any_sync(kFull, own && cnt > 0)) {  // rare: the owner holds another completion; its next candidate
#pragma unroll
        for (int s = 0; s < kSlots; ++s)
          if (own && rf[s] == iter && ri[s] != kFreeIdx && ri[s] > r && ri[s] < lm) { lm = ri[s]; ls = s; }
      }
      const Rec rr = rec[r];                                   // one 16-byte load: m, tokens, out_len
      const int Pr = rr.P, Or = max((int)(rr.O & kRecLenMask), 1);
      dn[r] = now;                                            // every lane, same address and value: one store, no branch
      kv_used -= (acc_t)Pr + (acc_t)Or;
      --b;
      if (kBudget) {
        if (ema_on) {                                         // Eq. 5-6 as printed: T_actual = observed output length, per category
          const int cr = min((int)cat[r], 3);
          const double tb = cr == 0 ? p.bp.t_base[0] : cr == 1 ? p.bp.t_base[1] : cr == 2 ? p.bp.t_base[2] : p.bp.t_base[3];
          if (tb > 0.0) {
            const double m = __ddiv_rn((double)Or, tb);
            const double t2 = __dmul_rn(t1, sl.B[cr]);
            const double t3 = __dmul_rn(alpha, m);
            sl.B[cr] = __dadd_rn(t2, t3);                       // every lane: same address, same value
          }
        }
      } else if (ema_on) {                                    // Eq. 5-6 (A3): four separately rounded operations; m = P/W came
        const int tr = (int)(rr.O >> 30);                     // rounded from pack_kernel (the same correctly rounded division)
        if (rr.m >= 0.0) {                                    // words > 0
          const double t2 = __dmul_rn(t1, sl.B[tr]);
          const double t3 = __dmul_rn(alpha, rr.m);
          sl.B[tr] = __dadd_rn(t2, t3);                         // every lane: same address, same value
        }
      }
      ++done;
      if (kBudget && closed && released < n) {                // the client whose request completed submits the next one
        const long long t_new = now + p.think;
        if (t_new < last_rel && lane == 0) atomicOr(p.status, DS_DEV_BAD_TRACE);   // a client's start tick lies after this release
        last_rel = t_new;
        if (lane == 0) __stcg(arr_d + released, t_new);
        if (lane == released - wb) { w_arr = t_new; sl.warr[lane] = t_new; }   // (released >= next >= wb; read back after the __syncwarp below)
        if (released == next) an = t_new;
        ++released;
        __syncwarp();
      }
      if (traj && done % p.traj_every == 0 && lane < kFac) traj[kFac * (done / p.traj_every - 1) + lane] = sl.B[lane];
    }
    // distance to the next completion: the occupied slots that did not complete now
    unsigned d = 0xffffffffu;
#pragma unroll
    for (int s = 0; s < kSlots; ++s) d = (ri[s] != kFreeIdx && rf[s] != iter) ? min(d, rf[s] - iter) : d;
    dist = __reduce_min_sync(kFull, d);
    blocked = false;
    __syncwarp();
  };

  auto queue_nonempty = [&]() -> bool {
    if (kReest) return qn > 0;
    if (kPolicy == DS_FIFO) return fifo_head < next;
    if (kPolicy == DS_SJF) return heap.size > 0;
    return tc[0].head < next || tc[1].head < next || tc[2].head < next;
  };

  // 4. ADMIT: while a slot is free, peek(policy, now); KV check on the estimate (A8); pop
  auto admit = [&]() {
    // batch-wait gate (reading B6): an idle server with a queued request collects for at most batch_wait
    // ticks from `collect` (the first boundary at which it is idle with a non-empty queue) and dispatches as soon as
    // max_batch requests are queued. Idle => everything started has completed, so next - done requests are queued.
    if (kBudget && p.batch_wait > 0 && b == 0) {
      if (collect < 0) collect = now;
      if (next - done < max_batch && now < collect + p.batch_wait) return;
      collect = -1;
    }
    while (b < max_batch) {
      int c = -1, ct = 0, wpos = 0; long long est_c = 0;
      int qpos = 0;
      if constexpr (kReest) {
        if (qn > 0) {
          const double B0 = sl.B[0], B1 = sl.B[1], B2 = sl.B[2];   // the factors as they are now
          auto est_now = [&](const int r, const int tr) -> long long {   // Eq. 1-2 reduced (A1) with the current factor (A16)
            const int base = max((int)BASE[r], 0);
            if (!ema_on) return base;                           // B == 1.0 exactly
            const double Bt = tr == 0 ? B0 : tr == 1 ? B1 : B2;
            return base > 0 ? (long long)ceil(__dmul_rn(Bt, (double)base)) : 0ll;
          };
          long long bk = kInf; int br = kFreeIdx, bp = 0;       // lane-best key (k0, request index) and its position in q
          int tmin[3] = {kFreeIdx, kFreeIdx, kFreeIdx}, tpos[3] = {0, 0, 0};   // WEIGHTED: oldest queued request per tier
          for (int j0 = 0; j0 < qn; j0 += 32) {
            const int j = j0 + lane;
            if (j < qn) {
              const int r = __ldcg(q + j);
              const int tr = min((int)tier[r], 2);
              if (kPolicy == DS_WEIGHTED) {
#pragma unroll
                for (int t = 0; t < 3; ++t) if (tr == t && r < tmin[t]) { tmin[t] = r; tpos[t] = j; }
              } else {
                long long k0 = 0;                               // FIFO: key = seq
                if (kPolicy == DS_PRIORITY) k0 = tr;
                else if (kPolicy == DS_SJF) k0 = est_now(r, tr);
                else if (kAging) {
                  const long long lv = (now - arr_at(r)) / p.aging_step;
                  k0 = (long long)tr - lv;
                  if (kPolicy == DS_AGING && k0 < 0) k0 = 0;    // A10: clamped at Premium's level
                }
                if (k0 < bk || (k0 == bk && r < br)) { bk = k0; br = r; bp = j; }
              }
            }
          }
          if (kPolicy == DS_WEIGHTED) {                         // slot pattern (A9): first non-empty tier in block order from cur's block
            const int m0 = __reduce_min_sync(kFull, tmin[0]), m1 = __reduce_min_sync(kFull, tmin[1]), m2 = __reduce_min_sync(kFull, tmin[2]);
            const int t0 = cur < p.w0 ? 0 : (cur < p.w0 + p.w1 ? 1 : 2);
            const unsigned nem = (m0 != kFreeIdx ? 1u : 0u) | (m1 != kFreeIdx ? 2u : 0u) | (m2 != kFreeIdx ? 4u : 0u);
            ct = -1;
#pragma unroll
            for (int k = 2; k >= 0; --k) {
              int t = t0 + k; if (t >= 3) t -= 3;
              if ((nem >> t) & 1u) { ct = t; wpos = k == 0 ? cur : (t == 0 ? 0 : (t == 1 ? p.w0 : p.w0 + p.w1)); }
            }
            c = ct == 0 ? m0 : ct == 1 ? m1 : m2;
            const int mine = ct == 0 ? tmin[0] : ct == 1 ? tmin[1] : tmin[2], mp = ct == 0 ? tpos[0] : ct == 1 ? tpos[1] : tpos[2];
            const unsigned own = __ballot_sync(kFull, mine == c);
            qpos = __shfl_sync(kFull, mp, __ffs(own) - 1);
          } else {
            const unsigned long long kb = warp_min_u64((unsigned long long)bk ^ 0x8000000000000000ull);   // signed order
            const int cand = ((unsigned long long)bk ^ 0x8000000000000000ull) == kb ? br : kFreeIdx;
            c = __reduce_min_sync(kFull, cand);
            const unsigned own = __ballot_sync(kFull, cand == c);
            qpos = __shfl_sync(kFull, bp, __ffs(own) - 1);
          }
          ct = min((int)tier[c], 2);
          est_c = est_now(c, ct);
        }
      } else
      if (kPolicy == DS_FIFO) {
        if (fifo_head < next) { c = fifo_head; est_c = fifo_est; }
      } else if (kPolicy == DS_SJF) {
        if (heap.size > 0) { const unsigned long long k = heap.top(); c = (int)(k & 0xffffffull); est_c = (long long)(k >> 24); }
      } else if (kPolicy == DS_PRIORITY) {
#pragma unroll
        for (int t = 2; t >= 0; --t) if (tc[t].head < next) { c = tc[t].head; est_c = tc[t].est; ct = t; }
      } else if (kPolicy == DS_WEIGHTED) {
        // slot pattern w0 x Premium, w1 x Standard, w2 x Batch scanned cyclically from `cur` (A9): the first non-empty
        // tier in block order starting with cur's own block; position = cur itself or that block's first slot
        const unsigned nem = (tc[0].head < next ? 1u : 0u) | (tc[1].head < next ? 2u : 0u) | (tc[2].head < next ? 4u : 0u);
        const unsigned tab = wblk == 0 ? kWeightedTab0 : wblk == 1 ? kWeightedTab1 : kWeightedTab2;
        ct = (int)((tab >> (2u * nem)) & 3u);                  // 3: every queue empty
        wpos = ct == wblk ? cur : (ct == 0 ? 0 : (ct == 1 ? p.w0 : p.w0 + p.w1));   // cur itself, or the first slot of that tier's block
        if (ct == 0) { c = tc[0].head; est_c = tc[0].est; }
        else if (ct == 1) { c = tc[1].head; est_c = tc[1].est; }
        else if (ct == 2) { c = tc[2].head; est_c = tc[2].est; }
      } else if (kPolicy == DS_AGING_UNCLAMPED) {  // A15: eff = tier - floor(waited/aging_step), not clamped; key (eff, seq)
        long long best_eff = 0;
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          if (tc[t].head < next) {                 // a head has the longest wait of its tier, so the minimum is among the heads
            const long long eff = (long long)t - (now - tc[t].arr) / p.aging_step;
            if (c < 0 || eff < best_eff || (eff == best_eff && tc[t].head < c)) { best_eff = eff; c = tc[t].head; est_c = tc[t].est; ct = t; }
          }
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
      if (b > 0 && use_kv && (long long)kv_used + est_c > p.kv_budget) { blocked = !kAging; break; }   // deferred (A8)
      // pop
      if constexpr (kReest) {
        if (lane == 0) { const int lastv = __ldcg(q + qn - 1); __stcg(q + qpos, lastv); }   // order in q is irrelevant: every pick scans all of it
        --qn;
        __syncwarp();
        if (kPolicy == DS_WEIGHTED) { cur = wpos + 1; if (cur >= wtot) cur = 0; wblk = cur < p.w0 ? 0 : (cur < p.w0 + p.w1 ? 1 : 2); }
        if (est_o) est_o[c] = est_c;                           // the estimate in force at admission to the batch (A16)
      } else
      if (kPolicy == DS_FIFO) {
        ++fifo_head;
        if (use_kv && fifo_head < next) fifo_est = (long long)__ldcg(dn + fifo_head);
      } else if (kPolicy == DS_SJF) heap.pop(lane);
      else {
#pragma unroll
        for (int t = 0; t < 3; ++t) if (t == ct) advance_cursor(tc[t], t, false);
        if (kPolicy == DS_WEIGHTED) { cur = wpos + 1; if (cur >= wtot) cur = 0; wblk = cur < p.w0 ? 0 : (cur < p.w0 + p.w1 ? 1 : 2); }
      }
      const Rec rc = rec[c];                                   // one 16-byte load: tokens, out_len (m unused here)
      const int Pc = rc.P;
      const int Oc = max((int)(rc.O & kRecLenMask), 1);        // (a bad out_len was reported when its window was loaded)
      st[c] = now;                                             // every lane, same address and value
      DS_K2_INVARIANT(nfree >= 1 && nfree <= 32 * kSlots && c >= 0 && c < next);
      const int slot = sl.stack[--nfree];                      // b < max_batch <= 32*kSlots: a free slot exists
      DS_K2_INVARIANT(slot >= 0 && slot < 32 * kSlots && sl.idx[slot] == kFreeIdx);
      sl.idx[slot] = c; sl.fin[slot] = iter + (unsigned)Oc;    // (uniform address and value)
      kv_used += (acc_t)Pc; prefill_new += (acc_t)Pc; ++b;
      dist = min(dist, (unsigned)Oc);
    }
  };

  // ---- main loop: one pass per iteration boundary that has an event; event-free boundaries are jumped over ----
  for (;;) {
    DS_K2_INVARIANT(b >= 0 && b <= max_batch && max_batch <= 32 * kSlots && nfree + b == 32 * kSlots);   // one slot per running request
    DS_K2_INVARIANT(next >= 0 && next <= n && done >= 0 && done <= next && wb >= 0 && wb <= next && next - wb <= 32);
    DS_K2_INVARIANT(kPolicy != DS_SJF || kReest || (heap.size >= 0 && heap.size <= next - done));
    DS_K2_INVARIANT(!kReest || (qn >= 0 && qn <= next - done));
    // 1.-3. Two inlined copies of ingest() instead of one in a two-trip loop: the loop's carried state cost ~35 instructions
    // per request in register moves (measured: configs[3] -4.8 %, configs[1] -6.7 % simulate time).
    if (dist == 0) {
      if (an < now) ingest(now - 1);                                      // 1. INGEST-EARLY: arrivals before this tick's completions
      retire();                                                           // 2. RETIRE
    }
    if (an <= now) ingest(now);                                           // 3. INGEST-NOW (without a completion at `now`: every arrival up to it)
    // 4. ADMIT. admit() returns with the batch full, the queue empty or (every policy but AGING) `blocked` set, so
    // afterwards something can still be admitted at the next boundary only under AGING (levels change with time)
    bool can_admit = !blocked && b < max_batch && queue_nonempty();
    if (can_admit) {
      admit();
      can_admit = kAging && !blocked && b < max_batch && queue_nonempty();
    }
    if (b == 0) {                                                         // 5. IDLE / END
      if (kBudget && p.batch_wait > 0) {
        // the gate's closed form: first queued (or next arriving) request q0 -> dispatch at min(arrival[q0] + wait,
        // arrival of the request that fills the batch); unsubmitted requests of a closed loop read as +inf
        const int qc = next - done;                                       // queued (gated) requests
        if (qc == 0) { if (next >= n) break; collect = an; }              // collection starts at the first arrival
        long long t = collect + p.batch_wait;
        const int kf = next + (max_batch - qc) - 1;                       // the arrival that fills the batch
        if (kf < n) { const long long tf = arr_at(kf); if (tf < t) t = tf; }
        now = t > now ? t : now;
        continue;
      }
      if (next >= n) break;
      now = an;
      continue;
    }
    // 6. STEP: the iteration that carries the prefill of the newly admitted requests
    acc_t dt = (acc_t)p.c_base + (acc_t)p.c_batch * (unsigned)b + kv_used * p.c_ctx;
    const acc_t cb = (acc_t)p.c_ctx * (unsigned)b;
    now += (long long)(dt + prefill_new * p.c_prefill);
    prefill_new = 0;
    kv_used += (unsigned)b; dt += cb; --dist; ++iter;
    // boundaries at which nothing can happen: no completion, and no arrival that could be admitted
    if (dist != 0 && !can_admit) {
      const bool arrivals_matter = b < max_batch && !(kPolicy == DS_FIFO && blocked) && next < n;
      // tick of the last boundary before the completion boundary: the stepping loop "while (an > now) step" runs all
      // `dist` iterations iff an > t_last
      const unsigned dm1 = dist - 1;
      const acc_t tri = (acc_t)dm1 * (acc_t)(dm1 - 1) / 2;               // kSmall: dist <= 65535, fits 32 bits
      const long long t_last = now + (long long)((unsigned long long)dm1 * dt + (unsigned long long)cb * tri);
      if (!arrivals_matter || an > t_last) {                              // next event is the completion: exact jump
        now = t_last + (long long)dt + (long long)((unsigned long long)dm1 * cb);
        kv_used += (acc_t)dist * (unsigned)b;
        iter += dist; dist = 0;
      } else {
        // next event is an arrival. Lower bound on the stepping loop's trip count: every one of the first `cap`
        // iterations costs at most dt + cb*cap ticks, where cap >= the true count because the true count is at most
        // ceil(G/dt). Float rounding (2^-22 relative with MUFU.RCP) is covered by the 1e-4 margins.
        unsigned j = 0;
        if (an > now && dt > 0) {
          const float G = (float)(an - now), fdt = (float)dt;
          const float cap = fminf(__fdividef(G, fdt) * 1.0001f + 1.0f, (float)dist);
          const float q = __fdividef(G, fdt + (float)cb * cap) * 0.9999f;
          j = q >= (float)dist ? dist : (unsigned)q;
          if (j > dist) j = dist;
        }
        if (j) {                                                          // j iterations at once, exact
          const acc_t trj = (acc_t)j * (acc_t)(j - 1) / 2;
          now += (long long)((unsigned long long)j * dt + (unsigned long long)cb * trj);
          kv_used += (acc_t)j * (unsigned)b;
          dt += (acc_t)j * cb;
          dist -= j; iter += j;
        }
        while (dist != 0 && an > now) { now += (long long)dt; kv_used += (unsigned)b; dt += cb; --dist; ++iter; }
      }
    }
  }
  if (lane < kFac) p.ema_final[kFac * (size_t)inst_id + lane] = sl.B[lane];
  __syncwarp();
}

// One 16-byte record per TRACE request (shared by all instances of the trace): the feedback ratio m = tokens/words of Eq. 6
// (reading A3) as a correctly rounded fp64 division - bit-identical to dividing at every completion - and the two lengths.
__global__ void __launch_bounds__(256) pack_kernel(const int32_t* __restrict__ W, const int32_t* __restrict__ P, const int32_t* __restrict__ O,
                                                   const uint8_t* __restrict__ tier, long long n, Rec* __restrict__ rec, unsigned int* status) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int w = W[i], pt = P[i], o = O[i];
    if (o > (int)kRecLenMask) atomicOr(status, DS_DEV_BAD_TRACE);     // (out_len < 1, tier > 2: reported when the window is loaded)
    Rec r;
    r.m = w > 0 ? __ddiv_rn((double)pt, (double)w) : -1.0;
    r.P = pt; r.O = ((unsigned)max(o, 0) & kRecLenMask) | ((unsigned)min((int)tier[i], 2) << 30);
    rec[i] = r;
  }
}

// true iff kv_used, the iteration cost (with prefill) and c_ctx*b of every reachable state of this trace stay below
// 2^31 and every out_len is <= 65535: kv_used <= max_batch*(maxP+maxO) since a running request holds P+g <= P+O tokens.
__device__ __forceinline__ bool trace_is_small(const Params& p, const int trace, const int lane) {
  const long long lo = p.trace_off[trace], n = p.trace_off[trace + 1] - lo;
  int mp = 0, mo = 0, mn = 0;
  for (long long i = lane; i < n; i += 32) {
    const int P = p.tokens[lo + i], O = p.out_len[lo + i];
    mp = max(mp, P); mo = max(mo, O); mn = min(mn, P);
  }
  mp = __reduce_max_sync(kFull, mp); mo = __reduce_max_sync(kFull, mo); mn = __reduce_min_sync(kFull, mn);
  const unsigned long long mb = (unsigned long long)p.max_batch;
  const unsigned long long kvmax = mb * ((unsigned long long)mp + (unsigned long long)mo);
  const unsigned long long dtmax = p.c_base + p.c_batch * mb + p.c_ctx * kvmax + p.c_prefill * mb * (unsigned long long)mp;
  return mn >= 0 && mo <= 65535 && kvmax < (1ull << 31) && dtmax < (1ull << 31) && (unsigned long long)p.c_ctx * mb < (1ull << 31);
}

// Processing order: instances grouped by policy, most expensive policy first (SJF, AGING, WEIGHTED, PRIORITY, FIFO).
// Each policy is its own ~25 KB of straight-line code; running one policy at a time across the GPU keeps the
// instruction cache warm (trace-major order thrashed it: 26 of 27 issue-stall samples were "no instruction"), and
// longest-first shortens the tail. One block; n_inst is small next to the simulation itself.
__global__ void __launch_bounds__(1024) order_kernel(const ds_instance* __restrict__ inst, long long n_inst, unsigned int* perm,
                                                     unsigned int* hdr) {
  __shared__ unsigned int cnt[6], pos[6];
  if (threadIdx.x < 6) cnt[threadIdx.x] = 0;
  __syncthreads();
  auto bucket = [](int policy) { return policy == DS_SJF ? 0 : (policy == DS_AGING || policy == DS_AGING_UNCLAMPED) ? 1 : policy == DS_WEIGHTED ? 2 :
                                        policy == DS_PRIORITY ? 3 : policy == DS_FIFO ? 4 : 5; };
  for (long long i = threadIdx.x; i < n_inst; i += blockDim.x) atomicAdd(&cnt[bucket(inst[i].policy)], 1u);
  __syncthreads();
  if (threadIdx.x == 0) {   // hdr[0..5]: per-bucket work counters (zeroed by the host), hdr[8..14]: bucket starts in perm[]
    unsigned a = 0;
    for (int k = 0; k < 6; ++k) { pos[k] = a; hdr[8 + k] = a; a += cnt[k]; }
    hdr[14] = a;
  }
  __syncthreads();
  // stable within a bucket per 1024-chunk: warp-aggregated ranks keep neighbouring instances (same trace) together
  for (long long base = 0; base < n_inst; base += blockDim.x) {
    const long long i = base + threadIdx.x;
    const int bk = i < n_inst ? bucket(inst[i].policy) : -1;
    __shared__ unsigned int wcnt[32][6];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    unsigned rank = 0;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const unsigned m = __ballot_sync(0xffffffffu, bk == k);
      if (bk == k) rank = __popc(m & ((1u << l) - 1u));
      if (l == 0) wcnt[w][k] = __popc(m);
    }
    __syncthreads();
    if (bk >= 0) {
      unsigned off = pos[bk];
      for (int ww = 0; ww < w; ++ww) off += wcnt[ww][bk];
      perm[off + rank] = (unsigned)i;
    }
    __syncthreads();
    if (threadIdx.x < 6) { unsigned a = 0; for (int ww = 0; ww < 32; ++ww) a += wcnt[ww][threadIdx.x]; pos[threadIdx.x] += a; }
    __syncthreads();
  }
}

template <int kSlots, bool kBudget = false, bool kReest = false>
__global__ void __launch_bounds__(k2::Shape<kSlots, kBudget, kReest>::kWarps * 32, k2::Shape<kSlots, kBudget, kReest>::kBlocks)
simulate_kernel(const __grid_constant__ Params p) {   // (launch shape per instantiation: k2::Shape above)
  constexpr int kFac = kBudget ? 4 : 3;
  constexpr int kWarpsPerBlock = Shape<kSlots, kBudget, kReest>::kWarps;
  __shared__ unsigned long long heap_sm[kWarpsPerBlock][kHeapSmem];
  __shared__ Slots<kSlots> slots_sm[kWarpsPerBlock];
  // lane and warp-in-block through volatile asm: under register pressure the compiler otherwise re-derives them from
  // SR_TID.X (a 20-cycle S2R plus shifts and the shared-memory address arithmetic) at every use: 27 instructions per request
  int lane, wib;
  asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane));
  asm volatile("{\n.reg .u32 t;\nmov.u32 t, %%tid.x;\nshr.u32 %0, t, 5;\n}" : "=r"(wib));
  // Policy affinity per SM: every warp of an SM starts on the same bucket and, when it is empty, moves to the bucket
  // with the most instances left, so that an SM executes one policy's code at a time (instruction-cache locality).
  // Buckets: SJF, AGING, WEIGHTED, PRIORITY, FIFO, invalid. SMs are split 26/31/35/30/26 (measured relative cost of one
  // instance per policy on configs[1]); the split only sets the starting point, stealing evens out the rest.
  unsigned smid;
  asm("mov.u32 %0, %%smid;" : "=r"(smid));
  const unsigned sm148 = (smid % p.n_sms) * 148u / p.n_sms;      // position of this SM on the 148-SM scale the split was measured on
  int bucket = sm148 < 26 ? 0 : sm148 < 57 ? 1 : sm148 < 92 ? 2 : sm148 < 122 ? 3 : 4;
  for (;;) {
    unsigned k = 0;
    if (lane == 0) k = atomicAdd(p.counter + bucket, 1u);
    k = __shfl_sync(kFull, k, 0);
    const unsigned b0 = p.counter[8 + bucket], b1 = p.counter[9 + bucket];
    if (k >= b1 - b0) {                                    // bucket empty: go where most work is left
      int best = -1; unsigned best_left = 0;
      if (lane < 6) {
        const unsigned tot = p.counter[9 + lane] - p.counter[8 + lane];
        const unsigned taken = *(volatile unsigned int*)(p.counter + lane);
        best_left = taken < tot ? tot - taken : 0u;
      }
      const unsigned mx = __reduce_max_sync(kFull, best_left);
      if (mx == 0) return;
      best = __ffs(__ballot_sync(kFull, best_left == mx)) - 1;
      bucket = best;
      continue;
    }
    const unsigned inst_id = p.perm[b0 + k];
    const ds_instance in = p.inst[inst_id];
    const int est_lo = kBudget ? DS_BUDGET_SPLIT : DS_SPLIT;          // this kernel's pair of estimators
    const bool bad_inst = in.trace < 0 || in.trace >= p.n_traces || in.policy < 0 || in.policy > DS_AGING_UNCLAMPED || in.estimator < est_lo ||
                          in.estimator > est_lo + 1 || !(in.ema_alpha >= 0.0 && in.ema_alpha <= 1.0);
    if (bad_inst) {
      if (lane == 0) atomicOr(p.status, DS_DEV_BAD_INSTANCE);
      if (lane < kFac) p.ema_final[kFac * (size_t)inst_id + lane] = 1.0;
      continue;
    }
    const bool split = in.estimator == est_lo;                         // T_input = words (else tokens)
    if (lane < kFac) p.ema_final[kFac * (size_t)inst_id + lane] = 1.0;   // overwritten unless the trace is rejected
    const bool small = trace_is_small(p, in.trace, lane);
#define DS_RUN(POL)                                                                                             \
  if (small && !kReest) run_instance<kSlots, POL, true, kBudget, false>(p, inst_id, in.trace, split, in.ema_alpha, heap_sm[wib], slots_sm[wib], lane);    \
  else run_instance<kSlots, POL, false, kBudget, kReest>(p, inst_id, in.trace, split, in.ema_alpha, heap_sm[wib], slots_sm[wib], lane)
    switch (in.policy) {
      case DS_FIFO: DS_RUN(DS_FIFO); break;
      case DS_PRIORITY: DS_RUN(DS_PRIORITY); break;
      case DS_WEIGHTED: DS_RUN(DS_WEIGHTED); break;
      case DS_SJF: DS_RUN(DS_SJF); break;
      case DS_AGING: DS_RUN(DS_AGING); break;
      default: DS_RUN(DS_AGING_UNCLAMPED); break;
    }
#undef DS_RUN
  }
}

}  // namespace k2

static size_t perm_bytes(int64_t n_inst) { return align_up(sizeof(unsigned int) * (size_t)(n_inst > 0 ? n_inst : 1), 256); }
size_t ws_simulate(int64_t total_requests, int64_t n_inst) {
  return align_up(256 + perm_bytes(n_inst) + sizeof(unsigned long long) * (size_t)total_requests, 256);
}
size_t ws_simulate_traces(int64_t n_requests) { return align_up(sizeof(k2::Rec) * (size_t)(n_requests > 0 ? n_requests : 1), 256); }

}  // namespace ds
static int simulate_impl(const ds_traces* tr, const uint8_t* category, const ds_budget* bp, int32_t n_clients, int64_t think_ticks,
                         int64_t batch_wait, int64_t* arrival_out, const ds_server* sv, const ds_instance* inst, int64_t n_inst,
                         const int64_t* out_off, int64_t n_total, int64_t* start_tick, int64_t* done_tick, double* ema_final,
                         const int64_t* traj_off, double* ema_traj, int64_t* est_out, void* workspace, size_t workspace_bytes,
                         void* stream) {
  using namespace ds;
  if (!tr || !sv || n_inst < 0 || n_total < 0) return DS_EINVAL;
  if (n_inst == 0) return DS_OK;
  if (!inst || !out_off || !start_tick || !done_tick || !ema_final || !workspace) return DS_EINVAL;
  if (tr->n_traces < 1 || !tr->trace_off || !tr->arrival_tick || !tr->tier || !tr->words || !tr->tokens || !tr->out_len) return DS_EINVAL;
  if (sv->max_batch < 1 || sv->max_batch > 256) return DS_EINVAL;
  if (sv->weight[0] < 1 || sv->weight[1] < 1 || sv->weight[2] < 1 || sv->aging_step < 1 || sv->traj_every < 0) return DS_EINVAL;
  if (sv->c_base < 0 || sv->c_batch < 0 || sv->c_ctx < 0 || sv->c_prefill < 0) return DS_EINVAL;
  if ((sv->reestimate != 0 && sv->reestimate != 1) || (sv->reestimate && bp)) return DS_EINVAL;   // A16 is built for ds_simulate / ds_simulate_est
  if (sv->c_base > 0x7fffffff || sv->c_batch > 0x7fffffff || sv->c_ctx > 0x7fffffff || sv->c_prefill > 0x7fffffff) return DS_EINVAL;
  if (n_inst > 0x7fffffff) return DS_EINVAL;
  if (bp) {
    if (!category) return DS_EINVAL;
    for (int c = 0; c < 4; ++c) if (!(bp->t_base[c] >= 0.0)) return DS_EINVAL;
    for (int t = 0; t < 3; ++t) if (!(bp->s_tenant[t] > 0.0)) return DS_EINVAL;
    if (!(bp->f_slope >= 0.0) || !(bp->f_max >= 1.0)) return DS_EINVAL;
  }
  // the whole documented workspace is required: header + permutation + one SJF heap slot per simulated request (the heap
  // region is only touched by SJF instances with more than kHeapSmem requests queued, but which launch will need it is
  // not known on the host)
  if (tr->n_requests < 0) return DS_EINVAL;
  if (workspace_bytes < ws_simulate(n_total, n_inst) + ws_simulate_traces(tr->n_requests)) return DS_ENOMEM;
  const int n_sms = num_sms();
  if (n_sms < 1) return cuda_fail(cudaGetLastError());
  cudaStream_t s = (cudaStream_t)stream;
  k2::Params p;
  p.trace_off = tr->trace_off; p.arrival = tr->arrival_tick; p.tier = tr->tier; p.words = tr->words; p.tokens = tr->tokens;
  p.out_len = tr->out_len; p.n_traces = tr->n_traces;
  p.max_batch = sv->max_batch; p.kv_budget = sv->kv_budget; p.c_base = (uint32_t)sv->c_base; p.c_batch = (uint32_t)sv->c_batch; p.c_ctx = (uint32_t)sv->c_ctx;
  p.c_prefill = (uint32_t)sv->c_prefill; p.w0 = sv->weight[0]; p.w1 = sv->weight[1]; p.w2 = sv->weight[2]; p.aging_step = sv->aging_step;
  p.traj_every = sv->traj_every;
  p.inst = inst; p.n_inst = n_inst; p.out_off = out_off; p.start_tick = start_tick; p.done_tick = done_tick;
  p.ema_final = ema_final; p.traj_off = traj_off; p.ema_traj = ema_traj; p.est_out = est_out;
  p.category = category; p.n_clients = n_clients; p.think = think_ticks; p.arrival_out = arrival_out; p.batch_wait = batch_wait;
  if (batch_wait < 0 || n_clients < 0 || think_ticks < 0 || (n_clients > 0 && (!bp || !arrival_out))) return DS_EINVAL;
  if (bp) p.bp = *bp; else memset(&p.bp, 0, sizeof(p.bp));
  p.counter = (unsigned int*)workspace;
  unsigned int* perm = (unsigned int*)((char*)workspace + 256);
  p.perm = perm;
  p.heap_ws = (unsigned long long*)((char*)workspace + 256 + perm_bytes(n_inst));
  p.status = status_ptr();
  if (!p.status) return cuda_fail(cudaGetLastError());
  p.n_total = n_total; p.n_sms = (unsigned)n_sms;
  k2::Rec* recs = (k2::Rec*)((char*)workspace + ws_simulate(n_total, n_inst));
  p.rec = recs;
  p.use_kv = sv->kv_budget > 0; p.want_est = est_out != nullptr; p.want_traj = ema_traj && traj_off && sv->traj_every > 0;
  DS_CUDA(cudaMemsetAsync(workspace, 0, 256, s));
  k2::order_kernel<<<1, 1024, 0, s>>>(inst, n_inst, perm, (unsigned int*)workspace);
  if (tr->n_requests > 0) {
    long long pb = (tr->n_requests + 255) / 256;
    if (pb > (long long)n_sms * 16) pb = (long long)n_sms * 16;
    k2::pack_kernel<<<(unsigned)pb, 256, 0, s>>>(tr->words, tr->tokens, tr->out_len, tr->tier, tr->n_requests, recs, p.status);
    note_launch();
  }
  note_launch();
  int per_sm = 0;
  auto launch = [&](auto kern, int warps) -> int {
    const int threads = warps * 32;
    DS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, 0));
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)n_sms * per_sm;
    const long long need = (n_inst + warps - 1) / warps;
    if (blocks > need) blocks = need;
    kern<<<(unsigned)blocks, threads, 0, s>>>(p);
    note_launch();
    DS_CUDA(cudaGetLastError());
    return DS_OK;
  };
  if (sv->reestimate) return launch(k2::simulate_kernel<8, false, true>, k2::Shape<8, false, true>::kWarps);   // the variant's one instantiation serves every max_batch <= 256
  if (bp) {
    if (sv->max_batch <= 32) return launch(k2::simulate_kernel<1, true>, k2::Shape<1, true, false>::kWarps);
    if (sv->max_batch <= 64) return launch(k2::simulate_kernel<2, true>, k2::Shape<2, true, false>::kWarps);
    if (sv->max_batch <= 128) return launch(k2::simulate_kernel<4, true>, k2::Shape<4, true, false>::kWarps);
    return launch(k2::simulate_kernel<8, true>, k2::Shape<8, true, false>::kWarps);
  }
  if (sv->max_batch <= 32) return launch(k2::simulate_kernel<1>, k2::Shape<1, false, false>::kWarps);
  if (sv->max_batch <= 64) return launch(k2::simulate_kernel<2>, k2::Shape<2, false, false>::kWarps);
  if (sv->max_batch <= 128) return launch(k2::simulate_kernel<4>, k2::Shape<4, false, false>::kWarps);
  return launch(k2::simulate_kernel<8>, k2::Shape<8, false, false>::kWarps);
}

extern "C" int ds_simulate(const ds_traces* tr, const ds_server* sv, const ds_instance* inst, int64_t n_inst,
                           const int64_t* out_off, int64_t n_total, int64_t* start_tick, int64_t* done_tick, double* ema_final,
                           const int64_t* traj_off, double* ema_traj, void* workspace, size_t workspace_bytes, void* stream) {
  return simulate_impl(tr, nullptr, nullptr, 0, 0, 0, nullptr, sv, inst, n_inst, out_off, n_total, start_tick, done_tick, ema_final, traj_off, ema_traj, nullptr, workspace,
                       workspace_bytes, stream);
}

extern "C" int ds_simulate_est(const ds_traces* tr, const ds_server* sv, const ds_instance* inst, int64_t n_inst,
                               const int64_t* out_off, int64_t n_total, int64_t* start_tick, int64_t* done_tick, double* ema_final,
                               const int64_t* traj_off, double* ema_traj, int64_t* est_out, void* workspace,
                               size_t workspace_bytes, void* stream) {
  if (n_inst > 0 && !est_out) return DS_EINVAL;
  return simulate_impl(tr, nullptr, nullptr, 0, 0, 0, nullptr, sv, inst, n_inst, out_off, n_total, start_tick, done_tick, ema_final, traj_off, ema_traj, est_out, workspace,
                       workspace_bytes, stream);
}

extern "C" int ds_simulate_budget(const ds_traces* tr, const uint8_t* category, const ds_budget* bp, const ds_server* sv,
                                  const ds_instance* inst, int64_t n_inst, const int64_t* out_off, int64_t n_total, int64_t* start_tick,
                                  int64_t* done_tick, double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out,
                                  void* workspace, size_t workspace_bytes, void* stream) {
  if (!bp) return DS_EINVAL;
  return simulate_impl(tr, category, bp, 0, 0, 0, nullptr, sv, inst, n_inst, out_off, n_total, start_tick, done_tick, ema_final, traj_off, ema_traj,
                       est_out, workspace, workspace_bytes, stream);
}

extern "C" int ds_simulate_closed(const ds_traces* tr, const uint8_t* category, const ds_budget* bp, const ds_server* sv,
                                  int32_t n_clients, int64_t think_ticks, int64_t batch_wait_ticks, const ds_instance* inst,
                                  int64_t n_inst,
                                  const int64_t* out_off, int64_t n_total, int64_t* arrival_out, int64_t* start_tick, int64_t* done_tick,
                                  double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out, void* workspace,
                                  size_t workspace_bytes, void* stream) {
  if (!bp || n_clients < 1) return DS_EINVAL;
  return simulate_impl(tr, category, bp, n_clients, think_ticks, batch_wait_ticks, arrival_out, sv, inst, n_inst, out_off, n_total, start_tick, done_tick,
                       ema_final, traj_off, ema_traj, est_out, workspace, workspace_bytes, stream);
}
