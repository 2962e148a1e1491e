/* CPU ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, single-threaded restatement of what the DriftSched hot path computes, written from
 * /root/reference/PAPER.md and SURVEY.md §8(c) (the binding readings of the paper; listed in
 * DESIGN.md §4). Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call anything in this directory. It shares no code, header,
 * table or constant generator with the CUDA path (paper_2606_02982_b200/csrc, include/): the
 * structs below are re-declared here on purpose.
 *
 * All pointers are HOST pointers. All time is int64 microsecond ticks. Return 0 on success,
 * -1 on a contract violation.
 */
#ifndef DRIFTSCHED_ORACLE_H
#define DRIFTSCHED_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int64_t n_traces;
  const int64_t* trace_off;    /* [n_traces+1] */
  const int64_t* arrival_tick; /* non-decreasing inside a trace */
  const uint8_t* tier;         /* 0 Premium 1 Standard 2 Batch */
  const int32_t* words;
  const int32_t* tokens;
  const int32_t* out_len;      /* >= 1 */
} oracle_traces;

typedef struct {
  int32_t max_batch;
  int64_t kv_budget;           /* <= 0: unlimited */
  int64_t c_base, c_batch, c_ctx, c_prefill;
  int32_t weight[3];
  int64_t aging_step;
  int32_t traj_every;
  int32_t reestimate;          /* 0: estimates frozen at arrival (A5); 1: online re-estimation of queued requests (A16) */
} oracle_server;

/* policy: 0 FIFO, 1 PRIORITY, 2 WEIGHTED, 3 SJF, 4 AGING (score clamped at Premium's level, A10),
 *         5 AGING_UNCLAMPED (A15: score = tier - floor(waited/aging_step), no clamp) */
typedef struct { int32_t trace, policy, estimator, _pad; double ema_alpha; } oracle_instance;

/* Budget estimators (estimator 2: T_input = words, 3: T_input = tokens), Eq. 1-2 of the paper in full. */
typedef struct {
  double t_base[4];    /* baseline output-token estimate per semantic category short_qa/summary/technical/report */
  double s_tenant[3];  /* tenant-aware safety scaling per tier */
  double f_slope, f_max; /* prompt complexity scaling F_input = min(f_max, 1 + f_slope * T_input) */
} oracle_budget;

/* PAPER.md:35,114 (split() proxy vs tokenizer-aware count); SURVEY.md §8(c) C.1. */
int oracle_characterize(const uint8_t* bytes, int64_t n_bytes, const int64_t* offsets, int64_t n_prompts,
                        int32_t* words_out, int32_t* tokens_out);

/* PAPER.md:171-181 (tier queues), 201-242 (policies), 278-286 (Eq. 5/6 EMA); SURVEY.md §8(c) C.2. */
int oracle_simulate(const oracle_traces* tr, const oracle_server* sv, const oracle_instance* inst, int64_t n_inst,
                    const int64_t* out_off, int64_t* start_tick, int64_t* done_tick,
                    double* ema_final /*[n_inst*3]*/,
                    const int64_t* traj_off /*nullable; [n_inst+1] sample ranges*/, double* ema_traj /*nullable; [samples][3]*/,
                    int64_t* est_out /*nullable; frozen admission-time estimate per simulated request*/);

/* Same loop with the paper's full estimator (Eq. 1-2, Alg. 1) and per-category feedback (Eq. 5-6 as printed,
 * PAPER.md:276-286): est = T_input + ceil(((t_base[c]*B[c])*s_tenant[tier])*F_input); on completion
 * B[c] <- (1-a)*B[c] + a*(out_len / t_base[c]). category: per request, 0..3. ema_final [n_inst*4], ema_traj [samples][4]. */
int oracle_simulate_budget(const oracle_traces* tr, const uint8_t* category, const oracle_budget* bp, const oracle_server* sv,
                           const oracle_instance* inst, int64_t n_inst, const int64_t* out_off, int64_t* start_tick,
                           int64_t* done_tick, double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out);

/* Closed-loop arrivals ("50 concurrent clients", 3000 requests per run): only the first n_clients
 * requests of a trace arrive at their input ticks; every completion (in completion order: tick, then request index) lets
 * the next request of the trace arrive at  completion tick + think_ticks. Same-tick ordering as everywhere: completions,
 * then same-tick arrivals (R-ORD). arrival_out [out_off[n_inst]]: the arrival tick of every simulated request (per
 * instance: arrivals now depend on the policy). Estimator and feedback as in oracle_simulate_budget.
 * batch_wait ("batch wait interval of 0.01 seconds before dispatching"; 0 = none): an IDLE server with a
 * queued request collects for at most batch_wait ticks: it dispatches when max_batch requests are queued or batch_wait
 * ticks after the collection started (the tick it went idle with a non-empty queue, else the first arrival after). */
int oracle_simulate_closed(const oracle_traces* tr, const uint8_t* category, const oracle_budget* bp, const oracle_server* sv,
                           int64_t n_clients, int64_t think_ticks, int64_t batch_wait, const oracle_instance* inst, int64_t n_inst,
                           const int64_t* out_off, int64_t* arrival_out, int64_t* start_tick, int64_t* done_tick,
                           double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out);

/* Estimation fidelity (Eq. 3-4 job classes; Tables IV, IX, X): per reporting group, exact integer sums
 * over its simulated requests: out[g*11 + ..] = { n, sum|est-P|, sum(est-P)^2, sum est, sum P, n_short, n_medium, n_long,
 * sum qdelay_short, sum qdelay_medium, sum qdelay_long } with class short: est<=128, medium: est<=512, long: else.
 * start_tick nullable (qdelay sums 0). class_seg nullable: 3*group+class per simulated request.
 * arrival_override (nullable, here and below; indexed like start_tick): per-instance arrival ticks of a closed-loop run
 * (oracle_simulate_closed's arrival_out), used instead of tr->arrival_tick. */
int oracle_estimation_error(const oracle_traces* tr, const oracle_instance* inst, int64_t n_inst, const int64_t* out_off,
                            const int64_t* arrival_override, const int64_t* est, const int64_t* start_tick, const int32_t* group, int32_t n_groups,
                            int64_t* out, int32_t* class_seg);

/* Queue depth per tenant tier over time (Fig. 8): depth[(i*n_samples + j)*3 + k] =
 * #{requests r of instance i with tier k : arrival <= t0 + j*dt < start_tick}. dt >= 1. */
int oracle_queue_depth(const oracle_traces* tr, const oracle_instance* inst, int64_t n_inst, const int64_t* out_off,
                       const int64_t* arrival_override, const int64_t* start_tick, int64_t t0, int64_t dt, int64_t n_samples, int32_t* depth);

/* PAPER.md:270 (queue wait vs end-to-end latency). seg outputs nullable. */
int oracle_latencies(const oracle_traces* tr, const oracle_instance* inst, int64_t n_inst, const int64_t* out_off,
                     const int64_t* arrival_override, const int64_t* start_tick, const int64_t* done_tick, const int32_t* group, const int64_t* t_mid,
                     int64_t* e2e, int64_t* qdelay, int32_t* seg_tier, int32_t* seg_all);

/* PAPER.md:436 (P50/P95/P99 tables), reading A13 (nearest rank). */
int oracle_tail_stats(const int64_t* values, const int32_t* seg_id, int64_t n, int32_t n_segments,
                      const int32_t* pct, int32_t n_pct, int64_t* out, int64_t* count_out);

#ifdef __cplusplus
}
#endif
#endif
