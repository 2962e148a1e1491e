// CPU ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT. See oracle.h for who may call this.
//
// Each function follows SURVEY.md §8(c) (the readings of PAPER.md this build binds itself to) in the
// order and notation given there: no blocking, fusion or reordering, single thread, int64 ticks,
// fp64 EMA with four separately rounded operations (build with -ffp-contract=off).
//
// Pin status (tests/test_oracle_*.py): characterize — pinned (Python bytes.split(), independent
// per-byte reference, closed-form token/word ratio, hand cases). simulate — pinned to the hand-worked
// traces H1-H14 (H7-H10: R-ORD, A8 blocking, A8 progress, KV release; H11/H12: A16; H13: A9 wrap; H14: R-ORD completion order), closed forms (service time, M/M/1, M/D/1, EMA geometric form), invariants I1-I9 (I2/A8 reconstructed from outputs) and
// brute force; the absolute latencies of the synthetic server model are this build's reading of
// BASELINE.json:configs[0] (DESIGN.md §4 A6-A10): "parity unpinned" beyond those pins.
// tail_stats — pinned (hand values, numpy partition).
// simulate_budget / simulate_closed (Eq. 1-2 in full, closed loop, batch wait) — pinned (tests/test_oracle_simulate_budget.py,
// tests/test_oracle_simulate_closed.py: hand traces, order-statistics identity of the releases, conservation, gate property).
// reestimate mode (reading A16) — pinned (tests/test_oracle_reestimate.py: hand traces H11/H12, reductions to the frozen run).
// estimation_error, queue_depth, latencies incl. their arrival_override form — pinned (tests/test_oracle_estimation_error.py,
// tests/test_oracle_queue_depth.py, tests/test_oracle_closed_loop_reporting.py: Eq. 4 thresholds, numpy one-liners, hand-worked
// closed-loop trace, queue-wait conservation, discrete Little's law). No function of this file is "parity unpinned".
#include "oracle.h"

#include <algorithm>
#include <cmath>
#include <vector>

namespace {

// SURVEY.md §8(c) C.1 byte classes. WS = Python bytes.split() whitespace ("split()").
inline bool is_ws(uint8_t c) { return c == 0x09 || c == 0x0A || c == 0x0B || c == 0x0C || c == 0x0D || c == 0x20; }
// PUNCT = Python string.punctuation.
inline bool is_punct(uint8_t c) {
  return (c >= 0x21 && c <= 0x2F) || (c >= 0x3A && c <= 0x40) || (c >= 0x5B && c <= 0x60) || (c >= 0x7B && c <= 0x7E);
}

}  // namespace

extern "C" int oracle_characterize(const uint8_t* bytes, int64_t n_bytes, const int64_t* offsets, int64_t n_prompts,
                                   int32_t* words_out, int32_t* tokens_out) {
  if (n_prompts < 0 || n_bytes < 0) return -1;
  for (int64_t i = 0; i < n_prompts; ++i) {
    int64_t a = offsets[i], b = offsets[i + 1];
    if (a < 0 || b < a || b > n_bytes) return -1;
    // words: number of maximal runs of non-WS bytes inside the prompt (isolated string).
    // tokens: sum over maximal LETTER runs of ceil(len/4), plus the number of PUNCT bytes.
    int32_t words = 0, tokens = 0;
    bool in_word = false;
    int64_t run = 0;  // current LETTER run length
    for (int64_t k = a; k < b; ++k) {
      uint8_t c = bytes[k];
      bool ws = is_ws(c), pu = is_punct(c);
      if (!ws) { if (!in_word) ++words; in_word = true; } else in_word = false;
      if (!ws && !pu) ++run;
      else { tokens += (int32_t)((run + 3) / 4); run = 0; if (pu) ++tokens; }
    }
    tokens += (int32_t)((run + 3) / 4);
    words_out[i] = words;
    tokens_out[i] = tokens;
  }
  return 0;
}

namespace {

enum { FIFO = 0, PRIORITY = 1, WEIGHTED = 2, SJF = 3, AGING = 4, AGING_UNCLAMPED = 5 };
enum { SPLIT = 0, EXACT = 1, BUDGET_SPLIT = 2, BUDGET_EXACT = 3 };

struct Sim {
  // inputs for one instance (local request index r in [0,n))
  const int64_t* arr; const uint8_t* tier; const int32_t* W; const int32_t* P; const int32_t* O;
  int64_t n; const oracle_server* sv; int policy, estimator; double alpha;
  const uint8_t* cat = nullptr; const oracle_budget* bp = nullptr;   // budget estimators only (Eq. 1-2 in full)
  // closed loop ("50 concurrent clients"): requests [released, n) have not been submitted yet
  std::vector<int64_t> arr_dyn; int64_t released = 0, think = 0; bool closed = false;
  int64_t collect_start = -1;        // batch-wait: tick at which the idle dispatcher started collecting (-1: not collecting)
  // state (SURVEY.md §8(c) C.2 "State per instance")
  int64_t now = 0, next = 0, kv_used = 0, done = 0;
  double B[4] = {1.0, 1.0, 1.0, 1.0};   // per tier (estimators 0/1) or per semantic category (budget estimators)
  int cur = 0;                       // Weighted slot cursor
  std::vector<int64_t> queued;       // all queued requests, arrival (= index) order
  std::vector<int64_t> R;            // running set, ascending request index
  std::vector<int64_t> est, g;

  bool budget() const { return estimator >= BUDGET_SPLIT; }
  int64_t base(int64_t r) const { return (estimator == SPLIT || estimator == BUDGET_SPLIT) ? (int64_t)W[r] : (int64_t)P[r]; }

  // Online re-estimation ("adaptive queue reordering, online workload
  // reclassification"; reading A16 in DESIGN.md §4): with sv->reestimate the estimate of a QUEUED request is not frozen at
  // arrival (A5) but recomputed from the factors current at every scheduling decision; est[r] ends as the value in force
  // when r was admitted to the batch.
  bool reest() const { return sv->reestimate != 0; }
  int64_t estimate_now(int64_t r) const {          // reduced estimator (A1) only: re-estimation is not defined for the budget estimators
    int64_t b = base(r);
    return b > 0 ? (int64_t)std::ceil(B[tier[r]] * (double)b) : 0;
  }
  int64_t queued_est(int64_t r) const { return reest() ? estimate_now(r) : est[r]; }

  // admit_to_queue(r): estimate frozen at arrival (A5), Eq. 1-2 reduced form (A1).
  void admit_to_queue(int64_t r) {
    int64_t b = base(r);
    if (budget()) {
      // Eq. 1-2; Alg. 1: T_budget = T_input + T_base * B_runtime * S_tenant * F_input,
      // factors multiplied left to right, each product rounded; F_input = min(f_max, 1 + f_slope*T_input) (B3).
      int c = cat[r];
      double F = 1.0 + bp->f_slope * (double)b;
      if (F > bp->f_max) F = bp->f_max;
      double x = bp->t_base[c] * B[c];
      x = x * bp->s_tenant[tier[r]];
      x = x * F;
      est[r] = b + (int64_t)std::ceil(x);
    } else if (b > 0) est[r] = (int64_t)std::ceil(B[tier[r]] * (double)b); else est[r] = 0;
    queued.push_back(r);
  }
  // ema_update(k,r): Eq. 5/6 with T_actual = tokens, T_base = base (A3); four separate roundings.
  void ema_update(int k, int64_t r) {
    if (budget()) {
      // Eq. 5-6, PAPER.md:278-286 as printed: B_measured = T_actual / T_base with T_actual the observed output length and
      // T_base the category baseline; one factor per workload category.
      int c = cat[r];
      if (alpha > 0.0 && bp->t_base[c] > 0.0) {
        double m = (double)O[r] / bp->t_base[c];
        double t1 = 1.0 - alpha;
        double t2 = t1 * B[c];
        double t3 = alpha * m;
        B[c] = t2 + t3;
      }
      return;
    }
    int64_t b = base(r);
    if (alpha > 0.0 && b > 0) {
      double m = (double)P[r] / (double)b;
      double t1 = 1.0 - alpha;
      double t2 = t1 * B[k];
      double t3 = alpha * m;
      B[k] = t2 + t3;
    }
  }
  // peek(policy, now): position in `queued` of the request the policy serves next. Lower key wins,
  // ties -> lower request index. `queued` is in index order, so the first minimum is the answer.
  size_t peek(int* weighted_pos) const {
    size_t best = 0;
    if (policy == WEIGHTED) {
      // slot pattern: weight[0] Premium slots, weight[1] Standard, weight[2] Batch (A9); scan from cur.
      int tot = sv->weight[0] + sv->weight[1] + sv->weight[2];
      for (int s = 0; s < tot; ++s) {
        int pos = (cur + s) % tot;
        int t = pos < sv->weight[0] ? 0 : (pos < sv->weight[0] + sv->weight[1] ? 1 : 2);
        for (size_t i = 0; i < queued.size(); ++i)
          if (tier[queued[i]] == t) { *weighted_pos = pos; return i; }   // head of that tier's FIFO
      }
      return 0;  // unreachable when queued is non-empty
    }
    int64_t bk0 = 0, bk1 = 0;
    for (size_t i = 0; i < queued.size(); ++i) {
      int64_t r = queued[i], k0, k1 = r;
      switch (policy) {
        case FIFO: k0 = 0; break;                                   // key = seq
        case PRIORITY: k0 = tier[r]; break;                         // (tier, seq)
        case SJF: k0 = queued_est(r); break;                        // (est, seq)   PAPER.md:231; A16: with the current factors
        default: {                                                  // AGING (A10)
          // PAPER.md:242 "waiting time progressively reduces the effective scheduling score". AGING clamps the score
          // at Premium's level (A10); AGING_UNCLAMPED (reading A15) lets it fall below 0, so
          // among long waiters the tier order survives instead of degenerating to arrival order.
          int64_t lv = (now - arr[r]) / sv->aging_step;
          int64_t eff = (int64_t)tier[r] - lv; if (eff < 0 && policy == AGING) eff = 0;
          k0 = eff;
        }
      }
      if (i == 0 || k0 < bk0 || (k0 == bk0 && k1 < bk1)) { best = i; bk0 = k0; bk1 = k1; }
    }
    return best;
  }
};

}  // namespace

static int simulate_impl(const oracle_traces* tr, const uint8_t* category, const oracle_budget* bp, const oracle_server* sv,
                         int64_t n_clients, int64_t think_ticks, int64_t batch_wait, int64_t* arrival_out,
                         const oracle_instance* inst, int64_t n_inst, const int64_t* out_off, int64_t* start_tick,
                         int64_t* done_tick, double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out) {
  const int nb = bp ? 4 : 3;   // factors per instance: semantic categories (budget estimators) or tenant tiers
  if (bp) {
    if (!category) return -1;
    for (int c = 0; c < 4; ++c) if (!(bp->t_base[c] >= 0.0)) return -1;
    for (int t = 0; t < 3; ++t) if (!(bp->s_tenant[t] > 0.0)) return -1;
    if (!(bp->f_slope >= 0.0) || !(bp->f_max >= 1.0)) return -1;
  }
  if (batch_wait < 0) return -1;
  if (n_clients < 0 || think_ticks < 0 || (n_clients > 0 && !arrival_out)) return -1;
  if (sv->max_batch < 1) return -1;
  if (sv->weight[0] < 1 || sv->weight[1] < 1 || sv->weight[2] < 1) return -1;
  if (sv->aging_step < 1) return -1;
  if (sv->reestimate != 0 && sv->reestimate != 1) return -1;
  if (sv->reestimate && bp) return -1;   // A16 is a reading for ds_simulate / ds_simulate_est only (the library returns DS_EINVAL)
  for (int64_t ii = 0; ii < n_inst; ++ii) {
    const oracle_instance& in = inst[ii];
    if (in.trace < 0 || in.trace >= tr->n_traces || in.policy < 0 || in.policy > AGING_UNCLAMPED || !(in.ema_alpha >= 0.0 && in.ema_alpha <= 1.0))
      return -1;
    if (bp ? (in.estimator != BUDGET_SPLIT && in.estimator != BUDGET_EXACT) : (in.estimator != SPLIT && in.estimator != EXACT)) return -1;
    int64_t lo = tr->trace_off[in.trace], n = tr->trace_off[in.trace + 1] - lo;
    Sim s;
    s.arr = tr->arrival_tick + lo; s.tier = tr->tier + lo; s.W = tr->words + lo; s.P = tr->tokens + lo;
    s.O = tr->out_len + lo; s.n = n; s.sv = sv; s.policy = in.policy; s.estimator = in.estimator; s.alpha = in.ema_alpha;
    s.est.assign(n, 0); s.g.assign(n, 0);
    // arrivals: the input array (open loop), or only its first n_clients entries (closed loop; the rest follow completions)
    s.arr_dyn.assign(s.arr, s.arr + n); s.arr = s.arr_dyn.data();
    s.closed = n_clients > 0; s.think = think_ticks; s.released = s.closed ? std::min<int64_t>(n_clients, n) : n;
    if (bp) {
      s.cat = category + lo; s.bp = bp;
      for (int64_t r = 0; r < n; ++r) if (s.cat[r] > 3) return -1;
    }
    int64_t* st = start_tick + out_off[ii];
    int64_t* dn = done_tick + out_off[ii];
    // instance ii owns samples [traj_off[ii], traj_off[ii+1]) of ema_traj, floor(n/traj_every) of them, 3 doubles each
    double* traj = (ema_traj && traj_off && sv->traj_every > 0) ? ema_traj + traj_off[ii] * nb : nullptr;

    bool skip_to_ingest_now = false;
    for (;;) {
      if (!skip_to_ingest_now) {
        // 1. INGEST-EARLY: arrivals strictly before `now` use the factors before this tick's completions (R-ORD).
        while (s.next < s.released && s.arr[s.next] < s.now) s.admit_to_queue(s.next++);
        // 2. RETIRE: completions at `now`, ascending request index.
        for (size_t i = 0; i < s.R.size();) {
          int64_t r = s.R[i];
          if (s.g[r] == s.O[r]) {
            dn[r] = s.now;
            s.kv_used -= (int64_t)s.P[r] + s.g[r];
            s.R.erase(s.R.begin() + i);
            s.ema_update(s.tier[r], r);
            ++s.done;
            // closed loop: the client whose request completed submits the next request after its think time
            if (s.closed && s.released < n) s.arr_dyn[s.released++] = s.now + s.think;
            if (traj && sv->traj_every > 0 && s.done % sv->traj_every == 0) {
              double* q = traj + (s.done / sv->traj_every - 1) * nb;
              for (int k = 0; k < nb; ++k) q[k] = s.B[k];
            }
          } else ++i;
        }
      }
      skip_to_ingest_now = false;
      // 3. INGEST-NOW: arrivals at exactly `now` see the updated factors.
      while (s.next < s.released && s.arr[s.next] <= s.now) s.admit_to_queue(s.next++);
      // 4. ADMIT
      int64_t prefill_new = 0;
      // batch-wait ("batch wait interval of 0.01 seconds before dispatching"; reading B6): when the server is
      // IDLE and a request is queued, the dispatcher collects for at most batch_wait ticks: it dispatches as soon as
      // max_batch requests are queued or batch_wait ticks after the collection started (= the first boundary at which
      // the server is idle with a non-empty queue: the tick it went idle, or the first arrival after that)
      bool gated = false;
      if (batch_wait > 0 && s.R.empty() && !s.queued.empty()) {
        if (s.collect_start < 0) s.collect_start = s.now;
        if ((int64_t)s.queued.size() < sv->max_batch && s.now < s.collect_start + batch_wait) gated = true;
        else s.collect_start = -1;
      }
      while (!gated && (int64_t)s.R.size() < sv->max_batch && !s.queued.empty()) {
        int wpos = 0;
        size_t qi = s.peek(&wpos);
        int64_t c = s.queued[qi];
        int64_t est_c = s.queued_est(c);                     // frozen at arrival (A5), or re-estimated now (A16)
        if (!s.R.empty() && sv->kv_budget > 0 && s.kv_used + est_c > sv->kv_budget) break;  // deferred (A8)
        s.est[c] = est_c;                                     // (A16: the estimate in force at admission to the batch)
        s.queued.erase(s.queued.begin() + qi);
        if (s.policy == WEIGHTED) s.cur = (wpos + 1) % (sv->weight[0] + sv->weight[1] + sv->weight[2]);
        st[c] = s.now; s.g[c] = 0;
        s.R.insert(std::lower_bound(s.R.begin(), s.R.end(), c), c);
        s.kv_used += s.P[c];
        prefill_new += s.P[c];
      }
      // 5. IDLE / END
      if (s.R.empty()) {
        if (gated) {                             // wake at the gate's deadline or at the next arrival, whichever is first
          int64_t t = s.collect_start + batch_wait;
          if (s.next < s.released && s.arr[s.next] < t) t = s.arr[s.next];
          s.now = t;
          skip_to_ingest_now = true;
          continue;
        }
        if (s.next == n) break;
        if (s.next >= s.released) return -1;   // unreachable: an empty server means every submitted request completed
        s.now = s.arr[s.next];
        skip_to_ingest_now = true;
        continue;
      }
      // 6. STEP: one server iteration (A6, A7).
      int64_t ctx = 0;
      for (int64_t r : s.R) ctx += (int64_t)s.P[r] + s.g[r];
      int64_t dt = sv->c_base + sv->c_batch * (int64_t)s.R.size() + sv->c_ctx * ctx + sv->c_prefill * prefill_new;
      for (int64_t r : s.R) s.g[r] += 1;
      s.kv_used += (int64_t)s.R.size();
      s.now += dt;
    }
    for (int k = 0; k < nb; ++k) ema_final[ii * nb + k] = s.B[k];
    if (est_out) for (int64_t r = 0; r < n; ++r) est_out[out_off[ii] + r] = s.est[r];   // frozen at arrival (A5)
    if (arrival_out) for (int64_t r = 0; r < n; ++r) arrival_out[out_off[ii] + r] = s.arr_dyn[r];
  }
  return 0;
}

extern "C" int oracle_simulate(const oracle_traces* tr, const oracle_server* sv, const oracle_instance* inst,
                               int64_t n_inst, const int64_t* out_off, int64_t* start_tick, int64_t* done_tick,
                               double* ema_final, const int64_t* traj_off, double* ema_traj, int64_t* est_out) {
  return simulate_impl(tr, nullptr, nullptr, sv, 0, 0, 0, nullptr, inst, n_inst, out_off, start_tick, done_tick, ema_final, traj_off, ema_traj, est_out);
}

extern "C" int oracle_simulate_budget(const oracle_traces* tr, const uint8_t* category, const oracle_budget* bp,
                                      const oracle_server* sv, const oracle_instance* inst, int64_t n_inst, const int64_t* out_off,
                                      int64_t* start_tick, int64_t* done_tick, double* ema_final, const int64_t* traj_off,
                                      double* ema_traj, int64_t* est_out) {
  if (!bp) return -1;
  return simulate_impl(tr, category, bp, sv, 0, 0, 0, nullptr, inst, n_inst, out_off, start_tick, done_tick, ema_final, traj_off, ema_traj, est_out);
}

extern "C" int oracle_simulate_closed(const oracle_traces* tr, const uint8_t* category, const oracle_budget* bp,
                                      const oracle_server* sv, int64_t n_clients, int64_t think_ticks, int64_t batch_wait,
                                      const oracle_instance* inst,
                                      int64_t n_inst, const int64_t* out_off, int64_t* arrival_out, int64_t* start_tick,
                                      int64_t* done_tick, double* ema_final, const int64_t* traj_off, double* ema_traj,
                                      int64_t* est_out) {
  if (!bp || n_clients < 1) return -1;
  return simulate_impl(tr, category, bp, sv, n_clients, think_ticks, batch_wait, arrival_out, inst, n_inst, out_off, start_tick, done_tick,
                       ema_final, traj_off, ema_traj, est_out);
}

// arrival_override (nullable, indexed like start_tick): the per-instance arrival ticks of a closed-loop run
// (oracle_simulate_closed's arrival_out; "50 concurrent clients"), used instead of tr->arrival_tick.
extern "C" int oracle_latencies(const oracle_traces* tr, const oracle_instance* inst, int64_t n_inst,
                                const int64_t* out_off, const int64_t* arrival_override, const int64_t* start_tick, const int64_t* done_tick,
                                const int32_t* group, const int64_t* t_mid, int64_t* e2e, int64_t* qdelay,
                                int32_t* seg_tier, int32_t* seg_all) {
  for (int64_t ii = 0; ii < n_inst; ++ii) {
    int64_t t = inst[ii].trace, lo = tr->trace_off[t], n = tr->trace_off[t + 1] - lo;
    for (int64_t r = 0; r < n; ++r) {
      int64_t o = out_off[ii] + r, a = arrival_override ? arrival_override[o] : tr->arrival_tick[lo + r];
      e2e[o] = done_tick[o] - a;        // end-to-end latency
      qdelay[o] = start_tick[o] - a;    // queue wait
      int32_t gph = group ? group[ii] : 0;
      if (t_mid) gph = gph * 2 + (a >= t_mid[t] ? 1 : 0);   // pre/post-drift phase (configs[4])
      if (seg_tier) seg_tier[o] = gph * 3 + tr->tier[lo + r];
      if (seg_all) seg_all[o] = gph;
    }
  }
  return 0;
}

extern "C" int oracle_tail_stats(const int64_t* values, const int32_t* seg_id, int64_t n, int32_t n_segments,
                                 const int32_t* pct, int32_t n_pct, int64_t* out, int64_t* count_out) {
  // collect values[i] with seg_id[i]==s (ids outside [0,n_segments) are skipped), sort ascending
  std::vector<std::vector<int64_t>> bucket((size_t)n_segments);
  for (int64_t i = 0; i < n; ++i) if (seg_id[i] >= 0 && seg_id[i] < n_segments) bucket[seg_id[i]].push_back(values[i]);
  for (int32_t s = 0; s < n_segments; ++s) {
    std::vector<int64_t>& v = bucket[s];
    std::sort(v.begin(), v.end());
    if (count_out) count_out[s] = (int64_t)v.size();
    for (int32_t q = 0; q < n_pct; ++q) {
      if (v.empty()) { out[s * n_pct + q] = -1; continue; }
      // nearest rank (A13): idx = max(1, ceil(p*n/100)) - 1
      int64_t rank = ((int64_t)pct[q] * (int64_t)v.size() + 99) / 100;
      if (rank < 1) rank = 1;
      if (rank > (int64_t)v.size()) rank = (int64_t)v.size();
      out[s * n_pct + q] = v[rank - 1];
    }
  }
  return 0;
}

extern "C" int oracle_estimation_error(const oracle_traces* tr, const oracle_instance* inst, int64_t n_inst,
                                       const int64_t* out_off, const int64_t* arrival_override, const int64_t* est, const int64_t* start_tick,
                                       const int32_t* group, int32_t n_groups, int64_t* out, int32_t* class_seg) {
  for (int64_t k = 0; k < (int64_t)n_groups * 11; ++k) out[k] = 0;
  for (int64_t ii = 0; ii < n_inst; ++ii) {
    int64_t t = inst[ii].trace, lo = tr->trace_off[t], n = tr->trace_off[t + 1] - lo;
    int32_t g = group ? group[ii] : 0;
    if (g < 0 || g >= n_groups) return -1;
    int64_t* o = out + (int64_t)g * 11;
    for (int64_t r = 0; r < n; ++r) {
      int64_t e = est[out_off[ii] + r], P = tr->tokens[lo + r];
      if (inst[ii].estimator >= 2) P += tr->out_len[lo + r];   // budget estimators predict input + output tokens (Eq. 1)
      int64_t err = e - P;                                  // estimate minus observed length (A3: T_actual = tokens)
      int cls = e <= 128 ? 0 : (e <= 512 ? 1 : 2);          // Eq. 4
      o[0] += 1; o[1] += err < 0 ? -err : err; o[2] += err * err; o[3] += e; o[4] += P;
      o[5 + cls] += 1;
      if (start_tick)                                        // queue wait; closed loop: the instance's own arrivals
        o[8 + cls] += start_tick[out_off[ii] + r] - (arrival_override ? arrival_override[out_off[ii] + r] : tr->arrival_tick[lo + r]);
      if (class_seg) class_seg[out_off[ii] + r] = 3 * g + cls;
    }
  }
  return 0;
}

// Per-tenant queue depth over time (Fig. 8): a request is queued from
// its arrival tick until the tick it is admitted to the batch. depth[i][j][k] = #{r of tier k : arrival <= t_j < start},
// t_j = t0 + j*dt. Written as the definition: every request increments the samples it covers.
extern "C" int oracle_queue_depth(const oracle_traces* tr, const oracle_instance* inst, int64_t n_inst, const int64_t* out_off,
                                  const int64_t* arrival_override, const int64_t* start_tick, int64_t t0, int64_t dt, int64_t n_samples, int32_t* depth) {
  if (dt < 1 || n_samples < 0) return -1;
  for (int64_t k = 0; k < n_inst * n_samples * 3; ++k) depth[k] = 0;
  for (int64_t ii = 0; ii < n_inst; ++ii) {
    int64_t t = inst[ii].trace, lo = tr->trace_off[t], n = tr->trace_off[t + 1] - lo;
    for (int64_t r = 0; r < n; ++r) {
      int64_t a = arrival_override ? arrival_override[out_off[ii] + r] : tr->arrival_tick[lo + r], st = start_tick[out_off[ii] + r];
      for (int64_t j = 0; j < n_samples; ++j) {
        int64_t tj = t0 + j * dt;
        if (tj >= st) break;
        if (tj >= a) depth[(ii * n_samples + j) * 3 + tr->tier[lo + r]] += 1;
      }
    }
  }
  return 0;
}
