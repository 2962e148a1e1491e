"""-m gpu: ds_simulate_budget (through the C ABI) vs the oracle: bit-exact ticks and budgets, 0-ulp factors."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

import oracle
from paper_2606_02982_b200 import workload as wl


@pytest.fixture(scope="module")
def G():
    import _gpuutil
    return _gpuutil


def _both(G, c, cat, out_len, bp, want_traj=False):
    import paper_2606_02982_b200 as ds
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, out_len)
    o = oracle.simulate_budget(*tr, cat, bp, c.server, c.instances, out_off=c.out_off, want_traj=want_traj, want_est=True)
    d = G.upload(c)
    d["out_len"] = torch.from_numpy(np.ascontiguousarray(out_len)).to(G.DEV)
    dcat = torch.from_numpy(np.ascontiguousarray(cat, np.uint8)).to(G.DEV)
    n_total = int(c.out_off[-1])
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    toff = traj = None
    if want_traj:
        toff_h = oracle.traj_offsets(c.trace_off, c.instances, c.server.traj_every)
        toff = torch.from_numpy(toff_h).to(G.DEV)
        traj = torch.zeros((int(toff_h[-1]), 4), dtype=torch.float64, device=G.DEV)
    est = torch.full((n_total,), -1, dtype=torch.int64, device=G.DEV)
    st, dn, ema = ds.api.simulate_budget(*targs, dcat, bp, c.server, d["inst"], d["out_off"], n_total, traj_off=toff, ema_traj=traj,
                                         est_out=est)
    assert ds.device_status() == 0
    for name, a, b in (("start", st, o[0]), ("done", dn, o[1]), ("est", est, o[-1])):
        a = a.cpu().numpy()
        bad = np.flatnonzero(a != b)
        assert bad.size == 0, (name, bad[:5], a[bad[:5]], b[bad[:5]])
    assert np.array_equal(ema.cpu().numpy().view(np.uint64), o[2].view(np.uint64))      # 0 ulp
    if want_traj:
        assert np.array_equal(traj.cpu().numpy().view(np.uint64), o[3].view(np.uint64))
    # estimation-error sums with observed = tokens + out_len (Eq. 1)
    osum = oracle.estimation_error(*tr, c.instances, c.out_off, o[-1], o[0], c.group, c.n_groups)
    gsum = ds.api.estimation_error(*targs, d["inst"], d["out_off"], n_total, est, st, d["group"], c.n_groups)
    assert np.array_equal(gsum.cpu().numpy(), osum)
    return o


@pytest.mark.parametrize("max_batch,kv", [(1, 0), (8, 0), (32, 16384), (32, 4000), (64, 9000), (200, 30000)])
def test_policy_sweep(G, max_batch, kv):
    sv = wl.Server(max_batch=max_batch, kv_budget=kv, aging_step=40_000, traj_every=37)
    combos = [(p, e, a) for p in wl.ALL_POLICIES for e, a in ((wl.BUDGET_SPLIT, 0.1), (wl.BUDGET_EXACT, 0.5), (wl.BUDGET_SPLIT, 0.0))]
    bp = wl.Budget(t_base=(38.0, 113.0, 189.0, 265.0), s_tenant=(1.25, 1.0, 0.8), f_slope=0.0013, f_max=1.2)
    for rho in (0.85, 1.3):
        c = wl._trace_workload("t", 31 + max_batch, 3, 600, sv, combos, oracle.characterize, rho=rho)
        cat, out_len = wl.assign_categories(31 + max_batch, c.out_len)
        _both(G, c, cat, out_len, bp, want_traj=True)


def test_hand_trace(G):
    bp = wl.Budget(t_base=(8.0, 20.0, 0.0, 0.0))
    req = [[0, 1, 3, 10, 3], [0, 1, 2, 8, 1]]
    for kv, st, dn in ((40, [0, 0], [6731, 2408]), (37, [0, 6533], [6533, 8731])):
        c = G.tiny_workload(wl, req, wl.Server(max_batch=2, kv_budget=kv), [(wl.FIFO, wl.BUDGET_EXACT, 0.0)])
        o = _both(G, c, np.array([0, 1], np.uint8), c.out_len, bp)
        assert o[0].tolist() == st and o[1].tolist() == dn and o[-1].tolist() == [18, 28]


def test_zero_baseline_and_default_budget_on_config_shape(G):
    sv = wl.Server(max_batch=32, kv_budget=16384, aging_step=500_000)
    combos = [(p, wl.BUDGET_SPLIT, 0.1) for p in wl.ALL_POLICIES]
    c = wl._trace_workload("t", 77, 4, 2000, sv, combos, oracle.characterize, rho=0.85)
    cat, out_len = wl.assign_categories(77, c.out_len)
    o = _both(G, c, cat, out_len, wl.Budget())
    assert 0.6 < o[2].mean() < 1.0                       # factors settle below 1 (Fig. 5)
    _both(G, c, cat, out_len, wl.Budget(t_base=(0.0, 0.0, 0.0, 0.0)))


def test_contracts(G):
    import paper_2606_02982_b200 as ds
    c = G.tiny_workload(wl, [[0, 0, 1, 1, 1], [5, 1, 2, 2, 1]], wl.Server(max_batch=1, kv_budget=0), [(wl.FIFO, wl.EXACT, 0.0)])
    d = G.upload(c)
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    cat = torch.tensor([0, 7], dtype=torch.uint8, device=G.DEV)
    ds.api.simulate_budget(*targs, cat, wl.Budget(), c.server, d["inst"], d["out_off"], 2)     # reduced estimator: bad instance
    assert ds.device_status() & 8
    c2 = G.tiny_workload(wl, [[0, 0, 1, 1, 1], [5, 1, 2, 2, 1]], wl.Server(max_batch=1, kv_budget=0), [(wl.SJF, wl.BUDGET_EXACT, 0.0)])
    d2 = G.upload(c2)
    ds.api.simulate_budget(*targs, cat, wl.Budget(), c2.server, d2["inst"], d2["out_off"], 2)   # category 7
    assert ds.device_status() & 2
    with pytest.raises(ds.DsError):
        ds.api.simulate_budget(*targs, cat, wl.Budget(f_max=0.5), c2.server, d2["inst"], d2["out_off"], 2)
    st, dn, ema = ds.simulate(*targs, c2.server, d2["inst"], d2["out_off"], 2)                  # budget estimator in ds_simulate
    assert ds.device_status() & 8
