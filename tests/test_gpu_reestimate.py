"""-m gpu: online re-estimation of queued requests (ds_server.reestimate = 1, reading A16) through the
C ABI vs the oracle: bit-exact ticks and dispatch-time estimates, 0-ulp factors."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2606_02982_b200 import workload as wl


@pytest.fixture(scope="module")
def G():
    import _gpuutil
    return _gpuutil


def _gpu(G, c):
    import paper_2606_02982_b200 as ds
    d = G.upload(c)
    st, dn, ema, est = ds.simulate_est(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server, d["inst"],
                                       d["out_off"], int(c.out_off[-1]))
    assert ds.device_status() == 0
    return st.cpu().numpy(), dn.cpu().numpy(), ema.cpu().numpy(), est.cpu().numpy()


def _same(g, o, c):
    for name, a, b in (("start", g[0], o[0]), ("done", g[1], o[1]), ("est", g[3], o[3])):
        bad = np.flatnonzero(a != b)
        assert bad.size == 0, (name, bad[:5], a[bad[:5]], b[bad[:5]], c.instances[bad[:5] // c.n_req])
    assert np.array_equal(g[2].view(np.uint64), o[2].view(np.uint64))


def _oracle(c):
    return oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances, want_est=True)


def test_hand_traces(G):
    # DESIGN.md §4.4 H11 / H12 (values typed from the derivation, as in tests/test_oracle_reestimate.py)
    c = G.tiny_workload(wl, [[0, 1, 4, 2, 1], [100, 1, 8, 3, 1], [200, 0, 7, 5, 1]], wl.Server(max_batch=1, kv_budget=0, reestimate=1),
                        [(wl.SJF, wl.SPLIT, 0.5)])
    st, dn, ema, est = _gpu(G, c)
    assert st.tolist() == [0, 2162, 4330] and dn.tolist() == [2162, 4330, 6510] and est.tolist() == [4, 6, 7]
    c = G.tiny_workload(wl, [[0, 1, 4, 2, 1], [0, 1, 12, 9, 3], [10, 1, 11, 5, 1]], wl.Server(max_batch=2, kv_budget=20, reestimate=1),
                        [(wl.FIFO, wl.SPLIT, 0.5)])
    st, dn, ema, est = _gpu(G, c)
    assert st.tolist() == [0, 0, 2366] and dn.tolist() == [2366, 6867, 4706] and est.tolist() == [4, 12, 9]


@pytest.mark.parametrize("max_batch,kv,rho", [(1, 0, 0.9), (4, 500, 1.2), (8, 3000, 1.1), (32, 16384, 0.85), (32, 2500, 1.4), (128, 20000, 1.0),
                                              (256, 30000, 1.3)])
def test_policy_sweep(G, max_batch, kv, rho):
    sv = wl.Server(max_batch=max_batch, kv_budget=kv, aging_step=40_000, reestimate=1)
    combos = [(p, e, a) for p in wl.ALL_POLICIES + [wl.AGING_UNCLAMPED] for e, a in ((wl.SPLIT, 0.1), (wl.SPLIT, 0.5), (wl.EXACT, 0.1), (wl.SPLIT, 0.0))]
    c = wl._trace_workload("t", 91 + max_batch, 2, 700, sv, combos, oracle.characterize, rho=rho)
    o = _oracle(c)
    _same(_gpu(G, c), o, c)
    c.server.reestimate = 0                                   # the mode does change the schedule of the split()+EMA instances
    f = _oracle(c)
    moving = (c.instances["estimator"] == wl.SPLIT) & (c.instances["ema_alpha"] > 0)
    per = lambda x: x.reshape(c.n_inst, c.n_req)
    assert (per(o[3])[moving] != per(f[3])[moving]).any()
    assert np.array_equal(per(o[0])[~moving], per(f[0])[~moving])     # alpha = 0 / exact: the frozen run


def test_drift_and_deep_queues(G):
    # configs[4] shape (tokens/word jumps mid-trace) under overload: long queues whose SJF order keeps changing
    c = wl.config4(oracle.characterize, n_traces=2, n_req=2500, materialise=True, traj_every=0)
    c.server.max_batch, c.server.kv_budget, c.server.reestimate = 16, 6000, 1
    c.arrival = (c.arrival // 2).astype(np.int64)             # twice the offered load
    _same(_gpu(G, c), _oracle(c), c)


def test_ties_zero_lengths_and_equal_ticks(G):
    rng = np.random.default_rng(6)
    n = 400
    req = np.stack([np.sort(rng.integers(0, 30, n)) * 40_000, rng.integers(0, 3, n), rng.integers(0, 3, n),
                    rng.integers(0, 4, n), rng.integers(1, 4, n)], 1)
    for mb, kv in ((1, 0), (4, 6), (32, 0)):
        sv = wl.Server(max_batch=mb, kv_budget=kv, aging_step=7000, reestimate=1)
        c = G.tiny_workload(wl, req, sv, [(p, e, 0.3) for p in wl.ALL_POLICIES + [wl.AGING_UNCLAMPED] for e in (wl.SPLIT, wl.EXACT)])
        _same(_gpu(G, c), _oracle(c), c)


def test_not_offered_with_the_budget_estimators(G):
    import torch
    import paper_2606_02982_b200 as ds
    c = G.tiny_workload(wl, [[0, 1, 4, 2, 1]], wl.Server(max_batch=1, reestimate=1), [(wl.FIFO, wl.BUDGET_SPLIT, 0.1)])
    d = G.upload(c)
    with pytest.raises(ds.DsError):
        ds.simulate_budget(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], torch.zeros(1, dtype=torch.uint8, device=G.DEV),
                           wl.Budget(), c.server, d["inst"], d["out_off"], 1)
    c.server.reestimate = 3
    with pytest.raises(ds.DsError):
        _gpu(G, G.tiny_workload(wl, [[0, 1, 4, 2, 1]], c.server, [(wl.FIFO, wl.SPLIT, 0.1)]))
