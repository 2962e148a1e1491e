"""-m gpu: ds_latencies + ds_tail_stats vs the oracle (bit-exact int64)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2606_02982_b200 import workload as wl


@pytest.fixture(scope="module")
def G():
    import _gpuutil
    return _gpuutil


def _gpu_tail(G, v, seg, nseg, pct):
    import torch
    import paper_2606_02982_b200 as ds
    out, cnt = ds.tail_stats(torch.from_numpy(np.ascontiguousarray(v, np.int64)).to(G.DEV),
                             torch.from_numpy(np.ascontiguousarray(seg, np.int32)).to(G.DEV), nseg, pct)
    return out.cpu().numpy(), cnt.cpu().numpy()


@pytest.mark.parametrize("nseg,n", [(1, 1), (4, 1000), (7, 300_000), (60, 2_000_000), (5000, 400_000)])
def test_random(G, nseg, n):
    rng = np.random.default_rng(nseg)
    v = rng.integers(0, 1 << 40, n)
    v[::3] = rng.integers(0, 100, len(v[::3]))
    if nseg == 7:
        v = v - (1 << 39)                       # negative values: signed order
    seg = rng.integers(-1, nseg + 1, n).astype(np.int32)      # -1 and nseg are skipped
    pct = (1, 50, 95, 99, 100)
    g, gc = _gpu_tail(G, v, seg, nseg, pct)
    o, oc = oracle.tail_stats(v, seg, nseg, pct)
    assert np.array_equal(gc, oc) and np.array_equal(g, o)


def test_extremes(G):
    v = np.array([np.iinfo(np.int64).min, -1, 0, 1, np.iinfo(np.int64).max, 5, 5, 5])
    seg = np.array([0, 0, 0, 0, 0, 1, 1, 1], np.int32)
    g, gc = _gpu_tail(G, v, seg, 3, (0, 50, 100))
    o, oc = oracle.tail_stats(v, seg, 3, (0, 50, 100))
    assert np.array_equal(g, o) and np.array_equal(gc, oc) and g[2].tolist() == [-1, -1, -1]


def test_pipeline_cfg1_small(G):
    import paper_2606_02982_b200 as ds
    c = wl.config1(oracle.characterize, n_traces=8, n_req=500, seed=3)
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    st, dn, _ = ds.simulate(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server,
                            d["inst"], d["out_off"], n_total)
    e2e, qd, seg_t, seg_a = ds.latencies(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"],
                                         d["inst"], d["out_off"], n_total, st, dn, d["group"])
    ost, odn, _ = oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances)
    oe, oq, os_t, os_a = oracle.latencies(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.instances,
                                          c.out_off, ost, odn, c.group)
    for a, b in ((e2e, oe), (qd, oq), (seg_t, os_t), (seg_a, os_a)):
        assert np.array_equal(a.cpu().numpy(), b)
    for vals, ovals in ((e2e, oe), (qd, oq)):
        for seg, oseg, ns in ((seg_t, os_t, 3 * c.n_groups), (seg_a, os_a, c.n_groups)):
            g, gc = ds.tail_stats(vals, seg, ns)
            o, oc = oracle.tail_stats(ovals, oseg, ns)
            assert np.array_equal(g.cpu().numpy(), o) and np.array_equal(gc.cpu().numpy(), oc)
