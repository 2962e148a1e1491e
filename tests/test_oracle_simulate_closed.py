"""Pins for oracle.simulate_budget(n_clients>0): closed-loop arrivals (50 concurrent clients; reading
B5 in DESIGN.md §4). What fixes the expected values independently of the oracle:
  * hand-worked traces (service time of a lone request 2150 + 6P for O = 1, from the cost formula);
  * the order-statistics identity: request r >= n_clients arrives at (the (r - n_clients + 1)-th smallest completion tick)
    + think, evaluated with numpy.sort on the oracle's own done ticks (a wrong release order or tick breaks it);
  * conservation: with think = 0 exactly n_clients requests are in the system until the last one has been submitted, so
    n_clients * t_last_release <= sum(e2e) <= n_clients * makespan;
  * n_clients >= n reduces to the open-loop run.
"""
import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import server


def _run(req, sv, policy, n_clients, think=0, cat=None, bp=None, est=wl.BUDGET_EXACT, alpha=0.0):
    req = np.asarray(req, np.int64).reshape(-1, 5)
    inst = np.zeros(1, wl.INSTANCE_DTYPE)
    inst[0] = (0, policy, est, 0, alpha)
    n = len(req)
    cat = np.zeros(n, np.uint8) if cat is None else cat
    bp = wl.Budget(t_base=(0.0, 0.0, 0.0, 0.0)) if bp is None else bp
    tr = ([0, n], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4])
    return oracle.simulate_budget(*tr, cat, bp, sv, inst, n_clients=n_clients, think_ticks=think)


def test_hand_traces():
    req = [[0, 1, 1, 1, 1], [0, 1, 1, 2, 1], [0, 1, 1, 3, 1], [0, 1, 1, 4, 1]]     # S = 2156, 2162, 2168, 2174
    st, dn, ema, arr = _run(req, server(), wl.FIFO, n_clients=2)
    assert arr.tolist() == [0, 0, 2156, 4318] and st.tolist() == [0, 2156, 4318, 6486] and dn.tolist() == [2156, 4318, 6486, 8660]
    st, dn, ema, arr = _run(req, server(), wl.FIFO, n_clients=2, think=100)
    assert arr.tolist() == [0, 0, 2256, 4418] and st.tolist() == [0, 2156, 4318, 6486]
    # one client: strictly sequential, each request arrives when the previous one completes (+ think); idle gap = think
    st, dn, ema, arr = _run(req, server(), wl.SJF, n_clients=1, think=1000)
    assert arr.tolist() == [0, 3156, 6318, 9486] and st.tolist() == arr.tolist() and dn.tolist() == [2156, 5318, 8486, 11660]
    # batch 2, two clients: nothing ever queues; both finish at 2000+300+3+15 = 2318, the next two at +2000+300+7+35
    st, dn, ema, arr = _run(req, server(max_batch=2), wl.FIFO, n_clients=2)
    assert arr.tolist() == [0, 0, 2318, 2318] and st.tolist() == arr.tolist() and dn.tolist() == [2318, 2318, 4660, 4660]
    # SJF reorders the queued pair: three clients, r1 (P 2) and r2 (P 3) queue behind r0; r3 arrives at r0's completion
    req2 = [[0, 1, 1, 9, 1], [0, 1, 1, 5, 1], [0, 1, 1, 3, 1], [0, 1, 1, 1, 1]]    # S = 2204, 2180, 2168, 2156
    st, dn, ema, arr = _run(req2, server(), wl.SJF, n_clients=3)
    # t=0: queue {r0,r1,r2}: SJF takes r2 (P 3): done 2168 -> r3 arrives; then r3 (P 1): 4324; r1: 6504; r0: 8708
    assert arr.tolist() == [0, 0, 0, 2168] and st.tolist() == [6504, 4324, 0, 2168] and dn.tolist() == [8708, 6504, 2168, 4324]


@pytest.mark.parametrize("policy", wl.ALL_POLICIES)
@pytest.mark.parametrize("n_clients,think", [(1, 0), (7, 0), (50, 0), (50, 25_000)])
def test_release_follows_completion_order_statistics(policy, n_clients, think):
    sv = wl.Server(max_batch=8, kv_budget=3000, aging_step=30_000)
    c = wl._trace_workload("t", 13, 1, 600, sv, [(policy, wl.BUDGET_SPLIT, 0.1)], oracle.characterize, rho=1.0)
    cat, out_len = wl.assign_categories(13, c.out_len)
    arrival0 = np.zeros_like(c.arrival)                      # all clients start at tick 0
    tr = (c.trace_off, arrival0, c.tier, c.words, c.tokens, out_len)
    st, dn, ema, arr = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances, n_clients=n_clients, think_ticks=think)
    n = c.n_req
    assert (arr[:n_clients] == 0).all()
    assert np.array_equal(arr[n_clients:], np.sort(dn)[: n - n_clients] + think)
    assert (st >= arr).all() and (dn > st).all()
    if think == 0:
        e2e = (dn - arr).sum()
        assert n_clients * arr.max() <= e2e <= n_clients * dn.max()
    # never more than n_clients requests in the system
    ev = np.concatenate([np.stack([arr, np.ones(n, np.int64)], 1), np.stack([dn, -np.ones(n, np.int64)], 1)])
    ev = ev[np.lexsort((ev[:, 1], ev[:, 0]))]               # completions before same-tick arrivals
    assert np.cumsum(ev[:, 1]).max() <= n_clients


def test_enough_clients_is_the_open_loop():
    sv = wl.Server(max_batch=8, kv_budget=3000)
    c = wl._trace_workload("t", 17, 2, 300, sv, [(p, wl.BUDGET_SPLIT, 0.1) for p in wl.ALL_POLICIES], oracle.characterize, rho=1.1)
    cat, out_len = wl.assign_categories(17, c.out_len)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, out_len)
    a = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances)
    b = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances, n_clients=300)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2].view(np.uint64), b[2].view(np.uint64))
    assert np.array_equal(b[3], np.tile(c.arrival.reshape(2, 300), (1, 1)).reshape(2, 300)[c.instances["trace"]].reshape(-1))


def test_sjf_lowers_the_median_under_the_paper_setup():
    # 50 clients, batch 32; SJF vs FIFO median end-to-end latency (-42 % in the paper's testbed)
    sv = wl.Server(max_batch=32, kv_budget=16384)
    c = wl._trace_workload("t", 23, 1, 3000, sv, [(wl.FIFO, wl.BUDGET_SPLIT, 0.1), (wl.SJF, wl.BUDGET_SPLIT, 0.1)], oracle.characterize, rho=1.0)
    cat, out_len = wl.assign_categories(23, c.out_len)
    tr = (c.trace_off, np.zeros_like(c.arrival), c.tier, c.words, c.tokens, out_len)
    st, dn, ema, arr = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances, n_clients=50)
    e2e = (dn - arr).reshape(2, 3000)
    assert np.median(e2e[1]) < 0.8 * np.median(e2e[0])


def test_contract():
    with pytest.raises(ValueError):
        _run([[0, 0, 1, 1, 1]], server(), wl.FIFO, n_clients=1, think=-1)


def test_batch_wait_hand_trace():
    # PAPER.md:302 batch wait (reading B6). max_batch 2, W = 10000, O = 1, kv off. S(alone) = 2150 + 6P; pair: 2300 + 6(P1+P2).
    # r0 @0, r1 @3000: the batch fills at 3000 (< 0 + W) -> both start at 3000, done 3000 + 2300 + 6*3 = 5318.
    # r2 @20000 alone: idle server waits until 30000, done 30000 + 2150 + 18 = 32168.
    # r3 @32168 arrives on the completion tick of r2: idle again -> waits for r4 @33000 (fills the batch) -> both at 33000.
    req = [[0, 1, 1, 1, 1], [3000, 1, 1, 2, 1], [20000, 1, 1, 3, 1], [32168, 1, 1, 4, 1], [33000, 1, 1, 5, 1]]
    req = np.asarray(req, np.int64)
    inst = np.zeros(1, wl.INSTANCE_DTYPE); inst[0] = (0, wl.FIFO, wl.BUDGET_EXACT, 0, 0.0)
    tr = ([0, 5], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4])
    bp = wl.Budget(t_base=(0.0, 0.0, 0.0, 0.0))
    st, dn, ema, arr = oracle.simulate_budget(*tr, np.zeros(5, np.uint8), bp, server(max_batch=2), inst, n_clients=5, batch_wait=10_000)
    assert arr.tolist() == req[:, 0].tolist()
    assert st.tolist() == [3000, 3000, 30000, 33000, 33000]
    assert dn.tolist() == [5318, 5318, 32168, 33000 + 2300 + 54, 33000 + 2300 + 54]
    # W = 0: no gate
    st0, dn0, _, _ = oracle.simulate_budget(*tr, np.zeros(5, np.uint8), bp, server(max_batch=2), inst, n_clients=5)
    assert st0.tolist() == [0, 3000, 20000, 32168, 34342]          # r4 joins at the boundary after r3's only iteration (2150 + 24)


@pytest.mark.parametrize("policy", wl.ALL_POLICIES)
def test_batch_wait_gate_property(policy):
    # checked from the outputs alone: whenever requests start on an idle server (nothing running across tick t), either the
    # batch was full or W ticks had passed since the collection started (the later of: the tick the server went idle, the
    # oldest queued arrival); and such a start happens exactly at that deadline or when the batch filled
    sv = wl.Server(max_batch=4, kv_budget=0, aging_step=30_000)
    c = wl._trace_workload("t", 29, 1, 500, sv, [(policy, wl.BUDGET_SPLIT, 0.1)], oracle.characterize, rho=0.3)   # often idle
    cat, out_len = wl.assign_categories(29, c.out_len)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, out_len)
    W = 10_000
    st, dn, ema, arr = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances, n_clients=500, batch_wait=W)
    assert np.array_equal(arr, c.arrival) and (st >= arr).all()
    n_idle = 0
    for t in np.unique(st):
        if ((st < t) & (dn > t)).any():
            continue                                           # server busy across t: continuous batching, no gate
        n_idle += 1
        q = np.flatnonzero((arr <= t) & (st >= t))             # queued at t (completions at t have retired)
        went_idle = dn[st < t].max() if (st < t).any() else 0  # tick at which the server last went idle
        cs = max(arr[q].min(), went_idle)                      # collection start: idle with a non-empty queue
        assert len(q) >= sv.max_batch or t >= cs + W
        fill = np.sort(arr[q])[sv.max_batch - 1] if len(q) >= sv.max_batch else -1
        assert t == cs + W or t == max(fill, went_idle)
    assert n_idle > 50
    st0 = oracle.simulate_budget(*tr, cat, wl.Budget(), sv, c.instances, n_clients=500)[0]
    assert (st != st0).any()
