"""-m gpu: ds_simulate_est / ds_estimation_error (through the C ABI) vs the oracle, bit-exact (all outputs are integers)."""
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


def _both(G, c, with_start=True, with_group=True):
    import paper_2606_02982_b200 as ds
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    ost, odn, oema, oest = oracle.simulate(*tr, c.server, c.instances, out_off=c.out_off, want_est=True)
    n_groups = c.n_groups if with_group else 1
    osum, oseg = oracle.estimation_error(*tr, c.instances, c.out_off, oest, ost if with_start else None,
                                         c.group if with_group else None, n_groups, want_class_seg=True)
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    st, dn, ema, est = ds.api.simulate_est(*targs, c.server, d["inst"], d["out_off"], n_total)
    gsum, gseg = ds.api.estimation_error(*targs, d["inst"], d["out_off"], n_total, est, st if with_start else None,
                                         d["group"] if with_group else None, n_groups, want_class_seg=True)
    assert ds.device_status() == 0
    assert np.array_equal(st.cpu().numpy(), ost) and np.array_equal(dn.cpu().numpy(), odn)
    assert np.array_equal(ema.cpu().numpy().view(np.uint64), oema.view(np.uint64))
    assert np.array_equal(est.cpu().numpy(), oest)
    assert np.array_equal(gsum.cpu().numpy(), osum)
    assert np.array_equal(gseg.cpu().numpy(), oseg)
    return osum


@pytest.mark.parametrize("max_batch,kv", [(1, 0), (8, 0), (32, 16384), (32, 3000), (200, 20000)])
def test_estimates_and_error_sums(G, max_batch, kv):
    sv = wl.Server(max_batch=max_batch, kv_budget=kv, aging_step=40_000)
    combos = [(p, e, a) for p in wl.ALL_POLICIES for e, a in ((wl.SPLIT, 0.1), (wl.EXACT, 0.1), (wl.SPLIT, 0.0))]
    c = wl._trace_workload("t", 91 + max_batch, 3, 700, sv, combos, oracle.characterize, rho=1.1)
    s = _both(G, c)
    assert (s[:, 0] == 3 * 700).all()


def test_null_start_and_null_group(G):
    sv = wl.Server(max_batch=16, kv_budget=0)
    c = wl._trace_workload("t", 7, 2, 333, sv, [(wl.SJF, wl.SPLIT, 0.2), (wl.FIFO, wl.SPLIT, 0.05)], oracle.characterize, rho=0.9)
    s = _both(G, c, with_start=False, with_group=False)
    assert s.shape == (1, 11) and (s[0, 8:] == 0).all()


def test_drift_workload(G):
    # configs[4] shape scaled down: the tokens/word ratio jumps mid-trace, estimates follow the factor
    c = wl.config4(n_traces=2, n_req=3000)
    _both(G, c)


def test_bad_group_sets_status(G):
    import paper_2606_02982_b200 as ds
    sv = wl.Server(max_batch=4, kv_budget=0)
    c = wl._trace_workload("t", 1, 1, 50, sv, [(wl.FIFO, wl.EXACT, 0.0)], oracle.characterize, rho=0.5)
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    st, dn, ema, est = ds.api.simulate_est(*targs, c.server, d["inst"], d["out_off"], n_total)
    bad = torch.full_like(d["group"], 5)
    ds.api.estimation_error(*targs, d["inst"], d["out_off"], n_total, est, st, bad, 2)
    assert ds.device_status() != 0
    assert ds.device_status() == 0        # reading clears it
