"""-m gpu: ds_queue_depth (through the C ABI) vs the oracle, bit-exact (integer counts)."""
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


def _both(G, c, grids):
    import paper_2606_02982_b200 as ds
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    ost, odn, oema = oracle.simulate(*tr, c.server, c.instances, out_off=c.out_off)
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    st, dn, ema = ds.simulate(*targs, c.server, d["inst"], d["out_off"], n_total)
    assert np.array_equal(st.cpu().numpy(), ost)
    for t0, dt, ns in grids:
        want = oracle.queue_depth(*tr, c.instances, c.out_off, ost, t0, dt, ns)
        got = ds.api.queue_depth(*targs, d["inst"], d["out_off"], st, t0, dt, ns)
        assert ds.device_status() == 0
        assert got.dtype == torch.int32 and tuple(got.shape) == want.shape
        assert np.array_equal(got.cpu().numpy(), want), (t0, dt, ns)
    return ost


@pytest.mark.parametrize("max_batch,kv,rho", [(1, 0, 0.9), (8, 0, 1.3), (32, 3000, 1.1), (200, 20000, 0.95)])
def test_depth_series(G, max_batch, kv, rho):
    sv = wl.Server(max_batch=max_batch, kv_budget=kv, aging_step=40_000)
    combos = [(p, e, 0.1) for p in wl.ALL_POLICIES for e in (wl.SPLIT, wl.EXACT)]
    c = wl._trace_workload("t", 23 + max_batch, 3, 700, sv, combos, oracle.characterize, rho=rho)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    t_end = int(c.arrival.max()) * 2
    # ragged sample counts (not multiples of 32), a grid starting before 0, a 1-tick grid, a single sample, none
    _both(G, c, [(0, max(1, t_end // 1000), 1003), (-54321, 99_991, 77), (int(c.arrival[5]), 1, 333), (t_end // 3, 7, 1), (0, 5, 0)])


def test_h1_by_hand(G):
    c = G.tiny_workload(wl, [[0, 1, 3, 4, 2], [1000, 0, 8, 10, 1], [1500, 2, 2, 3, 2]], wl.Server(max_batch=2, kv_budget=0),
                        [(wl.FIFO, wl.EXACT, 0.0)])
    import paper_2606_02982_b200 as ds
    d = G.upload(c)
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    st, dn, ema = ds.simulate(*targs, c.server, d["inst"], d["out_off"], 3)
    got = ds.api.queue_depth(*targs, d["inst"], d["out_off"], st, 0, 500, 12).cpu().numpy()
    assert got[0, :, 0].tolist() == [0, 0, 1, 1, 1, 0, 0, 0, 0, 0, 0, 0]
    assert got[0, :, 1].tolist() == [0] * 12
    assert got[0, :, 2].tolist() == [0, 0, 0, 1, 1, 1, 1, 1, 1, 1, 0, 0]


def test_configs1_scale_littles_law(G):
    # configs[1] shape at 64 traces: property that holds at any size (sum over a 1-tick... too long) -> coarse grid identity:
    # depth(t_j) = #{arrival <= t_j} - #{start <= t_j}, checked on sampled instances with numpy.searchsorted
    import paper_2606_02982_b200 as ds
    c = wl.config1(oracle.characterize, n_traces=64)
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    st, dn, ema = ds.simulate(*targs, c.server, d["inst"], d["out_off"], n_total)
    ns, dt = 2048, 100_000
    got = ds.api.queue_depth(*targs, d["inst"], d["out_off"], st, 0, dt, ns).cpu().numpy()
    sth = st.cpu().numpy()
    t = dt * np.arange(ns)
    rng = np.random.default_rng(0)
    for i in rng.choice(c.n_inst, 24, replace=False):
        tri = c.instances["trace"][i]
        lo, hi = c.trace_off[tri], c.trace_off[tri + 1]
        for k in range(3):
            m = c.tier[lo:hi] == k
            a = np.sort(c.arrival[lo:hi][m]); s = np.sort(sth[c.out_off[i]:c.out_off[i + 1]][m])
            assert np.array_equal(got[i, :, k], np.searchsorted(a, t, side="right") - np.searchsorted(s, t, side="right"))
    assert (got >= 0).all()


def test_bad_arguments(G):
    import paper_2606_02982_b200 as ds
    c = G.tiny_workload(wl, [[0, 0, 1, 1, 1]], wl.Server(max_batch=1, kv_budget=0), [(wl.FIFO, wl.EXACT, 0.0)])
    d = G.upload(c)
    targs = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"])
    st, dn, ema = ds.simulate(*targs, c.server, d["inst"], d["out_off"], 1)
    with pytest.raises(ds.DsError):
        ds.api.queue_depth(*targs, d["inst"], d["out_off"], st, 0, 0, 4)
