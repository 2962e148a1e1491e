"""Pins for the closed-loop reporting path of the oracle: oracle.latencies / estimation_error / queue_depth with
`arrival_override` = the per-instance arrival ticks a closed-loop run produced (3000 requests, 50 clients; the
setup behind Tables VI-IX, and Fig. 8). What fixes the expected values:
  * a hand-worked closed-loop trace (ticks from tests/test_oracle_simulate_closed.py::test_hand_traces, latencies by hand);
  * reduction: an override that repeats the trace's own arrivals per instance changes nothing;
  * conservation identities that involve the overriding arrivals: sum of the queue-wait-by-class sums = sum(start - arrival_out);
    discrete Little's law at dt = 1: sum_j depth = sum(start - arrival_out);
  * a wrong source of arrivals is visible: with all clients starting at tick 0 the trace's arrivals are all 0, so latencies
    computed from them equal the raw done ticks, which is not what the override gives.
"""
import numpy as np

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import server


def _closed(n_req=400, n_clients=20, seed=31, policies=(wl.FIFO, wl.SJF, wl.PRIORITY)):
    sv = wl.Server(max_batch=8, kv_budget=3000, aging_step=30_000)
    combos = [(p, wl.BUDGET_SPLIT, 0.1) for p in policies]
    c = wl._trace_workload("t", seed, 2, n_req, sv, combos, oracle.characterize, rho=1.0)
    cat, out_len = wl.assign_categories(seed, c.out_len)
    c.out_len = out_len
    c.arrival = np.zeros_like(c.arrival)                      # the paper's clients all start together
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    st, dn, ema, est, arr = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances, n_clients=n_clients, want_est=True)
    return c, tr, st, dn, est, arr


def test_hand_trace_latencies():
    # 2 clients, batch 1, O = 1, S = 2150 + 6P: arrivals (0, 0, 2156, 4318), start (0, 2156, 4318, 6486), done (2156, 4318, 6486, 8660)
    req = np.asarray([[0, 1, 1, 1, 1], [0, 0, 1, 2, 1], [0, 2, 1, 3, 1], [0, 1, 1, 4, 1]], np.int64)
    inst = np.zeros(1, wl.INSTANCE_DTYPE); inst[0] = (0, wl.FIFO, wl.BUDGET_EXACT, 0, 0.0)
    tr = ([0, 4], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4])
    bp = wl.Budget(t_base=(0.0, 0.0, 0.0, 0.0))
    st, dn, ema, arr = oracle.simulate_budget(*tr, np.zeros(4, np.uint8), bp, server(), inst, n_clients=2)
    assert arr.tolist() == [0, 0, 2156, 4318]
    off = np.array([0, 4], np.int64)
    e2e, qd, seg_t, seg_a = oracle.latencies(*tr, inst, off, st, dn, arrival_override=arr)
    assert e2e.tolist() == [2156, 4318, 4330, 4342] and qd.tolist() == [0, 2156, 2162, 2168]
    assert seg_t.tolist() == [1, 0, 2, 1] and seg_a.tolist() == [0, 0, 0, 0]
    # drift/phase split uses the overriding arrival too: t_mid = 2156 puts r2, r3 (arrivals 2156, 4318) in phase 1
    _, _, seg_t, seg_a = oracle.latencies(*tr, inst, off, st, dn, t_mid=np.array([2156], np.int64), arrival_override=arr)
    assert seg_a.tolist() == [0, 0, 1, 1] and seg_t.tolist() == [1, 0, 5, 4]
    # queue depth: r1 waits [0, 2156), r2 [2156, 4318), r3 [4318, 6486); sampled every 1000 ticks from 0
    d = oracle.queue_depth(*tr, inst, off, st, 0, 1000, 8, arrival_override=arr)[0]
    assert d[:, 0].tolist() == [1, 1, 1, 0, 0, 0, 0, 0]       # Premium r1
    assert d[:, 2].tolist() == [0, 0, 0, 1, 1, 0, 0, 0]       # Batch r2: samples 3000, 4000
    assert d[:, 1].tolist() == [0, 0, 0, 0, 0, 1, 1, 0]       # Standard r3: samples 5000, 6000
    # estimation error: est = T_input = tokens (t_base 0) = 1..4 -> all "short"; queue wait sum of the class = 0+2156+2162+2168
    out = oracle.estimation_error(*tr, inst, off, np.asarray([1, 2, 3, 4], np.int64), st, None, 1, arrival_override=arr)
    assert out[0, 5:8].tolist() == [4, 0, 0] and out[0, 8:].tolist() == [6486, 0, 0]


def test_override_equal_to_the_trace_arrivals_changes_nothing():
    sv = wl.Server(max_batch=8, kv_budget=3000)
    c = wl.config1(oracle.characterize, n_traces=3, n_req=300, seed=9)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    st, dn, ema, est = oracle.simulate(*tr, c.server, c.instances, want_est=True)
    ov = c.arrival.reshape(c.n_traces, c.n_req)[c.instances["trace"]].reshape(-1)
    a = oracle.latencies(*tr, c.instances, c.out_off, st, dn, c.group)
    b = oracle.latencies(*tr, c.instances, c.out_off, st, dn, c.group, arrival_override=ov)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    a = oracle.estimation_error(*tr, c.instances, c.out_off, est, st, c.group, c.n_groups)
    b = oracle.estimation_error(*tr, c.instances, c.out_off, est, st, c.group, c.n_groups, arrival_override=ov)
    assert np.array_equal(a, b)
    a = oracle.queue_depth(*tr, c.instances, c.out_off, st, 0, 50_000, 64)
    b = oracle.queue_depth(*tr, c.instances, c.out_off, st, 0, 50_000, 64, arrival_override=ov)
    assert np.array_equal(a, b)


def test_conservation_identities_with_the_closed_loop_arrivals():
    c, tr, st, dn, est, arr = _closed()
    e2e, qd, seg_t, seg_a = oracle.latencies(*tr, c.instances, c.out_off, st, dn, c.group, arrival_override=arr)
    assert (qd >= 0).all() and (e2e > qd).all()
    assert not np.array_equal(e2e, dn)                        # the trace's arrivals (all 0) would give e2e == done
    # queue wait by job class sums to the total queue wait of the group
    out = oracle.estimation_error(*tr, c.instances, c.out_off, est, st, c.group, c.n_groups, arrival_override=arr)
    for g in range(c.n_groups):
        sel = np.repeat(c.group == g, c.n_req)
        assert out[g, 8:].sum() == (st - arr)[sel].sum()
        assert out[g, 0] == sel.sum()
    wrong = oracle.estimation_error(*tr, c.instances, c.out_off, est, st, c.group, c.n_groups)
    assert (wrong[:, 8:].sum(axis=1) > out[:, 8:].sum(axis=1)).all()    # trace arrivals (0) overstate every wait
    # discrete Little's law at dt = 1 on one instance: sum over ticks of the depth = sum of the queue waits
    i = 1
    sl = slice(i * c.n_req, (i + 1) * c.n_req)
    T = int(st[sl].max()) + 1
    one = c.instances[i:i + 1]
    d = oracle.queue_depth(*tr, one, np.array([0, c.n_req], np.int64), st[sl], 0, 1, T, arrival_override=arr[sl])
    assert int(d.sum()) == int((st[sl] - arr[sl]).sum())
    tier = c.tier.reshape(c.n_traces, c.n_req)[one["trace"][0]]
    for k in range(3):
        assert int(d[0, :, k].sum()) == int((st[sl] - arr[sl])[tier == k].sum())
    # never more than n_clients requests queued
    assert d.sum(axis=2).max() <= 20
