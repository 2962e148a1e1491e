/* driftsched.h — C ABI of the B200-native DriftSched evaluation hot path (libdriftsched.so).
 *
 * The library evaluates LLM-serving scheduling policies in bulk, following the problem statement of
 * "DriftSched" (arxiv/paper_2606_02982; text in /root/reference/PAPER.md) as instantiated by
 * BASELINE.json and SURVEY.md §8:
 *   (a) ds_characterize : admission-time workload characterization of packed prompt text,
 *   (b) ds_simulate     : tick-exact simulation of tier queues x scheduling policy x continuous-batching
 *                         server model x per-tier EMA calibration, one instance per warp,
 *   (c) ds_latencies + ds_tail_stats (or the fused ds_latency_stats) : queue wait / end-to-end latency and their percentiles.
 *
 * Conventions (all entry points)
 *  - extern "C"; plain pointers and sizes; no C++/torch types.
 *  - Every function returns int: DS_OK (0) or a negative DS_E* code. No exception or abort crosses the ABI.
 *  - Unless a parameter says "host", every data pointer is a DEVICE pointer owned by the caller
 *    (allocate with cudaMalloc / torch). The library never frees or retains caller memory.
 *  - Descriptor structs (ds_traces, ds_server) are passed by HOST pointer and read during the call;
 *    the arrays they point to are device arrays.
 *  - Work is enqueued on the caller's stream (`stream` is a cudaStream_t passed as void*; NULL = default
 *    stream). Calls do not synchronise. Host-checkable arguments fail immediately with DS_EINVAL;
 *    device-side contract violations (non-monotone offsets, tier > 2, out_len < 1, decreasing arrivals,
 *    key overflow) set a sticky device status word, read (with a stream sync) by ds_device_status().
 *  - Scratch memory comes from a caller-supplied workspace; query its size with ds_workspace_bytes().
 *    Workspace contents are undefined on entry and exit; two calls in flight need two workspaces.
 *  - There is no CPU fallback: every function fails with DS_ECUDA if no CUDA device is usable.
 *  - Devices: every call works on the calling thread's current CUDA device (cudaSetDevice); pointers, stream and workspace
 *    must belong to it. The status word, the SM count used to size grids and the kernels' shared-memory attributes are
 *    kept per device, so one process may drive several devices (bench.py uses one process per GPU all the same).
 */
#ifndef DRIFTSCHED_H
#define DRIFTSCHED_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DS_OK 0
#define DS_EINVAL (-1) /* bad argument / host-checkable contract violation */
#define DS_ECUDA (-2)  /* CUDA runtime error (see ds_last_cuda_error) */
#define DS_ENOMEM (-3) /* workspace too small */
#define DS_ELIMIT (-4) /* size beyond the built-in scratch of a *_static entry point (use the workspace form of the call) */

/* bits of the device status word (ds_device_status) */
#define DS_DEV_BAD_OFFSETS 1u  /* ds_characterize: offsets not in [0,n_bytes] or decreasing */
#define DS_DEV_BAD_TRACE 2u    /* ds_simulate: tier > 2, out_len < 1, words/tokens < 0 or arrivals decreasing */
#define DS_DEV_KEY_RANGE 4u    /* ds_simulate: SJF key overflow (est >= 2^39 or trace longer than 2^24) */
#define DS_DEV_BAD_INSTANCE 8u /* ds_simulate: instance field out of range; ds_estimation_error: group out of range */
#define DS_DEV_INTERNAL 32u   /* ds_simulate built with -DDS_K2_CHECK only: an internal invariant of the kernel's bookkeeping failed */
#define DS_DEV_BAD_OUT_OFF 16u /* ds_simulate: out_off[i] < 0 or out_off[i] + trace length > n_total (instance skipped) */

/* ---------------------------------------------------------------------------------------------- (a)
 * Workload characterization ("whitespace-delimited word counts" vs
 * "tokenizer-aware" accounting; Table III). Definition: SURVEY.md §8(c) C.1.
 *   WS     = {0x09,0x0A,0x0B,0x0C,0x0D,0x20}  (Python bytes.split())
 *   PUNCT  = 0x21-0x2F, 0x3A-0x40, 0x5B-0x60, 0x7B-0x7E
 *   LETTER = every other byte value
 * For prompt i = bytes[offsets[i], offsets[i+1]) taken as an isolated string:
 *   words_out[i]  = number of maximal runs of non-WS bytes                      (the split() proxy)
 *   tokens_out[i] = sum over maximal LETTER runs of ceil(len/4) + number of PUNCT bytes
 *                   (BASELINE.json:configs[0] pseudo-token rule standing in for the model tokenizer)
 * bytes   [n_bytes]      device, any alignment (16-byte alignment is fastest). The kernel reads whole 16-byte-aligned
 *                        pieces: up to 15 bytes before bytes and after bytes + n_bytes are loaded (and ignored) when the
 *                        ends are not 16-byte aligned. Such a piece never leaves the 256-byte allocation granule that holds
 *                        a byte of the buffer, so any cudaMalloc / torch (sub-)allocation is safe; a buffer carved out of
 *                        a foreign mapping at finer granularity must be padded to 16-byte boundaries.
 * offsets [n_prompts+1]  device, 0 <= offsets[0], non-decreasing, offsets[n_prompts] <= n_bytes
 * words_out, tokens_out [n_prompts] device, overwritten.
 * workspace: ds_workspace_bytes(DS_WS_CHARACTERIZE, n_bytes, n_prompts).
 * Launches: 2 memsets (the two outputs) + 1 kernel. */
int ds_characterize(const uint8_t* bytes, int64_t n_bytes, const int64_t* offsets, int64_t n_prompts,
                    int32_t* words_out, int32_t* tokens_out, void* workspace, size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------- (b) */
typedef struct {              /* SoA request records, traces concatenated; HOST struct, DEVICE arrays */
  int64_t n_traces;
  const int64_t* trace_off;    /* [n_traces+1] request index range of each trace */
  const int64_t* arrival_tick; /* microsecond ticks, >= 0, non-decreasing inside a trace */
  const uint8_t* tier;         /* 0 Premium, 1 Standard, 2 Batch */
  const int32_t* words;        /* split() count, >= 0 */
  const int32_t* tokens;       /* pseudo-token count = true prompt length, >= 0 */
  const int32_t* out_len;      /* decode length, in [1, 2^30) */
  int64_t n_requests;          /* HOST copy of trace_off[n_traces]: requests over all traces = length of the five arrays above */
} ds_traces;

typedef struct {              /* continuous-batching server model, BASELINE.json:configs[0] */
  int32_t max_batch;           /* 1..256 */
  int64_t kv_budget;           /* tokens; <= 0 means unlimited */
  int64_t c_base, c_batch, c_ctx, c_prefill; /* each in [0, 2^31): iteration cost = c_base + c_batch*b + c_ctx*sum(ctx) + c_prefill*sum(P_new) */
  int32_t weight[3];           /* Weighted policy slots per tier, each >= 1: {4,2,1} configs, {5,3,2} PAPER.md:234 */
  int64_t aging_step;          /* ticks waited per promoted tier level, >= 1 */
  int32_t traj_every;          /* 0 = no EMA trajectory; k = sample B[0..2] every k completions */
  int32_t reestimate;          /* 0 = estimates frozen at arrival (reading A5, the measured path). 1 = online re-estimation of queued
                                  requests ("adaptive queue reordering, online workload
                                  reclassification"; A16): SJF's key and the KV admission check use ceil(B[tier]*base) with the
                                  factors current at the scheduling decision, est_out is the estimate in force when the request was
                                  admitted to the batch. ds_simulate / ds_simulate_est only (DS_EINVAL with the budget estimators); a
                                  variant that scans the queue at every pick, not tuned for throughput. */
} ds_server;

#define DS_FIFO 0
#define DS_PRIORITY 1
#define DS_WEIGHTED 2
#define DS_SJF 3
#define DS_AGING 4    /* PAPER.md:242; score max(0, tier - floor(waited/aging_step)) (A10) */
#define DS_AGING_UNCLAMPED 5 /* PAPER.md:242, variant (A15): score tier - floor(waited/aging_step), no clamp */
#define DS_SPLIT 0    /* estimate base = words  (split() proxy) */
#define DS_EXACT 1    /* estimate base = tokens (tokenizer-aware) */
#define DS_BUDGET_SPLIT 2 /* ds_simulate_budget only: full Eq. 1-2 estimator, T_input = words  */
#define DS_BUDGET_EXACT 3 /* ds_simulate_budget only: full Eq. 1-2 estimator, T_input = tokens */

typedef struct {
  int32_t trace;     /* index into ds_traces */
  int32_t policy;    /* DS_FIFO .. DS_AGING_UNCLAMPED */
  int32_t estimator; /* DS_SPLIT / DS_EXACT (ds_simulate, ds_simulate_est); DS_BUDGET_* (ds_simulate_budget) */
  int32_t _pad;
  double ema_alpha;  /* EMA learning rate in [0,1] (Eq. 5); 0 = BIAS OFF */
} ds_instance;

/* Simulate n_inst independent (trace, policy, estimator, alpha) instances, one warp each.
 * Algorithm: SURVEY.md §8(c) C.2 (LOOP steps 1-6, readings A1-A14, R-ORD), summarised in DESIGN.md §3.
 *   est = ceil(B[tier]*base) frozen at arrival (Eq. 1-2 reduced);
 *   EMA on completion: m=P/base; B = (1-a)*B + a*m in fp64, four separately rounded operations.
 * inst        [n_inst]            device
 * out_off     [n_inst+1]          device; instance i writes start/done at out_off[i] + local request index
 * n_total                         HOST value: out_off[n_inst] = number of simulated requests = length of every per-request
 *                                 output array; an instance whose range leaves [0, n_total) is skipped (DS_DEV_BAD_OUT_OFF)
 * start_tick, done_tick           device, int64, sized n_total; done_tick is also used as scratch
 *                                 for the frozen estimates while a request is queued
 * ema_final   [n_inst*3]          device, fp64 B[tier] at the end of the run
 * traj_off    [n_inst+1] nullable device; instance i owns trajectory samples [traj_off[i], traj_off[i+1]),
 *                                 floor(n_req_i / traj_every) of them
 * ema_traj    [traj_off[n_inst]*3] nullable device fp64
 * workspace: ds_workspace_bytes(DS_WS_SIMULATE, n_total, n_inst) + ds_workspace_bytes(DS_WS_SIMULATE_TRACES, tr->n_requests, 0)
 *   bytes are REQUIRED (DS_ENOMEM otherwise): header, instance permutation, one 8-byte SJF heap slot per simulated request
 *   (touched only by SJF instances with more than 256 requests queued, but always validated), then one packed 16-byte
 *   record per trace request (tokens/words ratio, tokens, out_len; written by a pre-pass of every call).
 * Contract checked on the device (DS_DEV_BAD_TRACE, outputs of that instance unspecified): tier <= 2, words/tokens >= 0,
 *   1 <= out_len < 2^30, arrival_tick >= 0 and non-decreasing over every pair of neighbouring requests of a trace.
 *   The check REPORTS, it does not stop the instance: with decreasing arrivals a request may be queued ahead of its turn or
 *   twice. What was verified on such inputs (randomised closed-loop cases under the -DDS_K2_CHECK build): every
 *   request index the kernel uses stays inside the trace, so start_tick / done_tick / est_out writes stay inside the
 *   instance's own ranges, and the running-set bookkeeping stays intact. What is NOT guaranteed: the SJF heap / re-estimation
 *   queue scratch and the trajectory samples of such an instance may run up to a few entries past its own share of the
 *   workspace / ema_traj. When DS_DEV_BAD_TRACE is set, treat every output of the CALL as invalid and validate the traces
 *   (sorted arrivals; for ds_simulate_closed: every client start tick <= the first release) before calling again.
 * Launches: 1 memset (work counter) + 3 kernels (policy-major ordering of the instances, request records, simulation). */
int ds_simulate(const ds_traces* tr, const ds_server* sv, const ds_instance* inst, int64_t n_inst,
                const int64_t* out_off, int64_t n_total, int64_t* start_tick, int64_t* done_tick, double* ema_final,
                const int64_t* traj_off, double* ema_traj, void* workspace, size_t workspace_bytes, void* stream);

/* ds_simulate that also returns the frozen admission-time estimate of every simulated request (reading A5):
 * est_out [out_off[n_inst]] int64 device, same indexing as start_tick. Everything else as ds_simulate. */
int ds_simulate_est(const ds_traces* tr, const ds_server* sv, const ds_instance* inst, int64_t n_inst,
                    const int64_t* out_off, int64_t n_total, int64_t* start_tick, int64_t* done_tick, double* ema_final,
                    const int64_t* traj_off, double* ema_traj, int64_t* est_out, void* workspace, size_t workspace_bytes,
                    void* stream);

/* The paper's estimator in full (Eq. 1-2 and Alg. 1; semantic categories
 * short_qa / summary / technical / report; one feedback factor per workload category):
 *   T_budget = T_input + ceil(((t_base[c] * B[c]) * s_tenant[tier]) * F_input),   F_input = min(f_max, 1 + f_slope * T_input)
 *   (fp64, the three products and F's multiply-add rounded separately, in that order), T_input = words (DS_BUDGET_SPLIT)
 *   or tokens (DS_BUDGET_EXACT), c = category[r]; frozen at arrival; used as the SJF key, by KV admission and as est_out.
 * Feedback on completion of r (Eq. 5-6 as printed: T_actual = observed output length, T_base = the
 * category baseline): if ema_alpha > 0 and t_base[c] > 0:  B[c] <- (1-a)*B[c] + a*(out_len[r] / t_base[c]), B[] = 1.0 initially.
 * Everything else (queues, policies, server model, same-tick ordering) is ds_simulate's. The paper prints none of the
 * constants; they are parameters (DESIGN.md §4 B1-B4).
 * category [same indexing as tr->tier] uint8 device, values 0..3 (larger: DS_DEV_BAD_TRACE); bp: HOST struct, t_base >= 0,
 * s_tenant > 0, f_slope >= 0, f_max >= 1 (DS_EINVAL otherwise); every instance must use DS_BUDGET_SPLIT or DS_BUDGET_EXACT
 * (DS_DEV_BAD_INSTANCE otherwise). ema_final [n_inst*4], ema_traj [samples][4] (one factor per category). est_out nullable. */
typedef struct {
  double t_base[4];   /* baseline output-token estimate per semantic category */
  double s_tenant[3]; /* tenant-aware safety scaling per tier */
  double f_slope;     /* prompt complexity scaling: F_input = min(f_max, 1 + f_slope * T_input) */
  double f_max;
} ds_budget;
int ds_simulate_budget(const ds_traces* tr, const uint8_t* category, const ds_budget* bp, const ds_server* sv,
                       const ds_instance* inst, int64_t n_inst, const int64_t* out_off, int64_t n_total, int64_t* start_tick,
                       int64_t* done_tick, double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out,
                       void* workspace, size_t workspace_bytes, void* stream);

/* ds_simulate_budget with CLOSED-LOOP arrivals ("50 concurrent clients",
 * 3000 requests per run): only the first n_clients requests of a trace arrive at their tr->arrival_tick; every completion
 * (in completion order: tick, then request index) lets the next request of the trace arrive at completion tick +
 * think_ticks. Same-tick order as everywhere (R-ORD): completions, then same-tick arrivals, which therefore see the updated
 * factors. n_clients >= 1, think_ticks >= 0 (host values; DS_EINVAL otherwise); n_clients >= trace length = the open loop.
 * Contract: the arrival sequence the loop produces must be non-decreasing in request index like every trace's, i.e. the
 * first n_clients arrival ticks (non-decreasing, like every trace) must not lie after the first release: staggered client
 * starts are fine as long as the last client starts no later than the first completion + think_ticks (they are all 0 when
 * the paper's clients start together). Every release is compared with the arrival before it; a violation sets
 * DS_DEV_BAD_TRACE and the instance's outputs are unspecified.
 * arrival_out [out_off[n_inst]] int64 device (written): the arrival tick of every simulated request - per instance,
 * because arrivals now depend on the policy; latencies are done_tick - arrival_out / start_tick - arrival_out.
 * batch_wait_ticks >= 0 ("batch wait interval of 0.01 seconds before dispatching"; 0 = none; reading B6): an
 * IDLE server does not start at the first queued request's arrival a but when max_batch requests are queued or at
 * a + batch_wait_ticks, whichever is first; a busy server admits at every iteration boundary as before.
 * Everything else as ds_simulate_budget. */
int ds_simulate_closed(const ds_traces* tr, const uint8_t* category, const ds_budget* bp, const ds_server* sv, int32_t n_clients,
                       int64_t think_ticks, int64_t batch_wait_ticks, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                       int64_t n_total, int64_t* arrival_out,
                       int64_t* start_tick, int64_t* done_tick, double* ema_final, const int64_t* traj_off, double* ema_traj,
                       int64_t* est_out, void* workspace, size_t workspace_bytes, void* stream);

/* Estimation fidelity: job classes of Eq. 3-4 (short est<=128, medium
 * est<=512, long otherwise), token-estimation error (Tables IV, X) and queue wait by job class
 * (Table IX), per reporting group g = group[instance] (nullable -> 0) in [0, n_groups).
 * out [n_groups*11] int64 device, exact integer sums over the group's simulated requests:
 *   { n, sum|est-P|, sum(est-P)^2, sum est, sum P, n_short, n_medium, n_long, sum qdelay_short, _medium, _long }
 *   with P = tokens (the observed length, reading A3; tokens + out_len for the DS_BUDGET_* estimators, which predict
 *   input + output tokens, Eq. 1) and qdelay = start_tick - arrival (0 if start_tick is NULL).
 *   MAE = out[1]/out[0], RMSE = sqrt(out[2]/out[0]), mean bias = out[4]/out[3] are left to the caller (fp64).
 * class_seg (nullable) [out_off[n_inst]] int32 device: 3*g + class, usable as seg_id for ds_tail_stats.
 * A group outside [0, n_groups) sets DS_DEV_BAD_INSTANCE. Launches: 1 memset + 1 kernel.
 * arrival_override (nullable; here and in ds_queue_depth, ds_latencies, ds_latency_stats): int64 device array indexed like
 *   start_tick (out_off[i] + local request index) holding the arrival tick of every simulated request; when given it is
 *   used instead of tr->arrival_tick. It is the arrival_out of ds_simulate_closed: in a closed loop (the
 *   setup behind Tables VI-IX and Fig. 8) arrivals depend on the instance's policy, so the trace's array does not hold them. */
int ds_estimation_error(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                        const int64_t* arrival_override, const int64_t* est, const int64_t* start_tick, const int32_t* group, int32_t n_groups,
                        int64_t* out, int32_t* class_seg, void* stream);

/* Queue depth per tenant tier over time (Fig. 8: "per-tenant queue depth"):
 * a request is queued from its arrival tick until the tick it is admitted to the batch (start_tick).
 *   depth[(i*n_samples + j)*3 + k] = #{requests r of instance i with tier k : arrival_r <= t0 + j*dt < start_tick_r}
 * depth [n_inst*n_samples*3] int32 device (written); t0 any tick, dt >= 1, n_samples >= 0 (host values).
 * Launches: 1 memset + 2 kernels. */
int ds_queue_depth(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                   const int64_t* arrival_override, const int64_t* start_tick, int64_t t0, int64_t dt, int64_t n_samples, int32_t* depth, void* stream);

/* ---------------------------------------------------------------------------------------------- (c)
 * Latency derivation (worker timestamps separate queueing from inference):
 *   e2e = done - arrival, qdelay = start - arrival, per simulated request (same indexing as start/done);
 *   arrival = tr->arrival_tick, or arrival_override (see ds_estimation_error) for closed-loop runs.
 * Segment ids for ds_tail_stats, with g = group[i] (nullable -> 0) and, if t_mid != NULL,
 *   g = 2*g + (arrival >= t_mid[trace]) (pre/post-drift phase, BASELINE.json:configs[4]):
 *   seg_tier = 3*g + tier (per-tier statistics), seg_all = g (overall). Either seg output may be NULL.
 * n_total = out_off[n_inst] must be passed by the caller (host value). Launches: 1 kernel. */
int ds_latencies(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off, int64_t n_total,
                 const int64_t* arrival_override, const int64_t* start_tick, const int64_t* done_tick, const int32_t* group, const int64_t* t_mid,
                 int64_t* e2e, int64_t* qdelay, int32_t* seg_tier, int32_t* seg_all, void* stream);

/* Segmented percentiles by MSB-first radix select (PAPER.md:436 P50/P95/P99; Tables VI-VIII).
 * For each segment s in [0,n_segments): the values[i] with seg_id[i]==s, sorted ascending; for each pct p the
 * nearest-rank element, rank = max(1, ceil(p*n_s/100)). seg_id outside [0,n_segments)
 * (e.g. -1) is skipped. out[s*n_pct+q] = -1 for an empty segment. count_out (nullable) [n_segments].
 * pct is a HOST array of n_pct values in [0,100], n_pct <= 8.
 * workspace: ds_workspace_bytes(DS_WS_TAIL_STATS, n_segments, n_pct). Launches: 1 memset + up to 9 x 2 kernels. */
int ds_tail_stats(const int64_t* values, const int32_t* seg_id, int64_t n, int32_t n_segments, const int32_t* pct,
                  int32_t n_pct, int64_t* out, int64_t* count_out, void* workspace, size_t workspace_bytes, void* stream);

/* ds_tail_stats WITHOUT a caller workspace, for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the scratch (header, counts, prefixes, ranks, radix histograms)
 * is one fixed device array inside the library, DS_TAIL_STATS_STATIC_BYTES (134 400) bytes, present on every GPU that
 * loads the library until the process exits. The call allocates nothing: no cudaMalloc, cudaFree or allocating library
 * routine; it enqueues memsets and kernels on `stream` exactly like ds_tail_stats and returns the same results, bit for bit.
 * Limit: n_segments <= DS_TAIL_STATS_STATIC_MAX_SEGPCT and n_segments * n_pct <= DS_TAIL_STATS_STATIC_MAX_SEGPCT (128);
 *   anything larger returns DS_ELIMIT ("size beyond the built-in scratch") and launches nothing. n is not limited.
 * Sharing: every call on a device uses the SAME array, which keeps the last call's contents; each call clears what it
 *   needs at its start (on `stream`), so calls that follow one another on one stream are independent. Calls that OVERLAP on
 *   the GPU (two streams, two host threads without ordering between their streams) RACE on the array and give undefined
 *   results: order them with events, or use ds_tail_stats with one workspace per call in flight.
 * Everything else (arguments, nearest-rank definition, pct as a HOST array, -1 for an empty segment) as ds_tail_stats. */
#define DS_TAIL_STATS_STATIC_MAX_SEGPCT 128
#define DS_TAIL_STATS_STATIC_BYTES 134400
int ds_tail_stats_static(const int64_t* values, const int32_t* seg_id, int64_t n, int32_t n_segments, const int32_t* pct,
                         int32_t n_pct, int64_t* out, int64_t* count_out, void* stream);

/* Fused form of ds_latencies + 4 x ds_tail_stats for the report the paper's tables need (Tables VI-VIII: percentiles of
 * end-to-end latency and queue wait per tenant tier and overall): nothing is materialised, every radix pass recomputes
 * value = tick - arrival from start_tick / done_tick. With G = n_groups * (t_mid ? 2 : 1) and g as in ds_latencies:
 *   e2e_out, qdelay_out [4*G*n_pct] int64 device (either may be NULL = not wanted): entries [(3*g+tier)*n_pct + q] are the
 *     per-(group, tier) percentiles, entries [(3*G + g)*n_pct + q] the per-group ("overall") percentiles; -1 = empty.
 *   count_out [4*G] nullable: segment sizes in the same order.
 * Same nearest-rank definition and results as the unfused calls (bit-exact). pct: HOST array, n_pct <= 8.
 * Requires 4*G*n_pct <= 200 histograms (shared memory); DS_EINVAL otherwise: use the unfused calls then.
 * workspace: ds_workspace_bytes(DS_WS_TAIL_STATS, 4*G, n_pct), optionally followed by a staging area of
 *   ds_workspace_bytes(DS_WS_LATENCY_STAGE, n_total, 0) bytes (n_total = out_off[n_inst]; 5 bytes per simulated request): when
 *   it is there, out_off tiles [0, n_total) in instance order and every latency is below 2^32 ticks, the count pass stages
 *   32-bit keys + segment codes and the digit passes stream those instead of recomputing tick - arrival (same results,
 *   bit-exact; any other case silently takes the unstaged passes). Launches per wanted metric: 2 memsets + 2 + up to 8 x 2 kernels. */
int ds_latency_stats(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                     const int64_t* arrival_override, const int64_t* start_tick, const int64_t* done_tick, const int32_t* group, int32_t n_groups,
                     const int64_t* t_mid, const int32_t* pct, int32_t n_pct, int64_t* e2e_out, int64_t* qdelay_out,
                     int64_t* count_out, void* workspace, size_t workspace_bytes, void* stream);

#define DS_WS_CHARACTERIZE 0
#define DS_WS_SIMULATE 1
#define DS_WS_TAIL_STATS 2
#define DS_WS_LATENCY_STAGE 3 /* n = simulated requests over all instances; m unused: optional staging area of ds_latency_stats */
#define DS_WS_SIMULATE_TRACES 4 /* n = tr->n_requests; m unused: second, mandatory part of the ds_simulate* workspace */
/* Workspace size in bytes for call `which` with the two size arguments named at that call. Never 0. */
size_t ds_workspace_bytes(int which, int64_t n, int64_t m);

/* Synchronises `stream`, returns the sticky device status word (0 = all contracts held) and clears it.
 * Negative on CUDA error. */
int ds_device_status(void* stream);

const char* ds_strerror(int code);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char* ds_last_cuda_error(void);
/* Number of kernel launches (memsets not counted) issued by the library in this process since load. */
int64_t ds_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* DRIFTSCHED_H */
