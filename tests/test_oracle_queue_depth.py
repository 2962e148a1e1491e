"""Pins for oracle.queue_depth (Fig. 8).

What fixes the expected values, independently of the oracle's loop:
  * hand trace H1: start ticks (0, 2174, 4539) for arrivals (0, 1000, 1500) -> queued intervals by hand;
  * the counting identity depth(t) = #{arrival <= t} - #{start <= t}, evaluated with numpy.searchsorted (library routine);
  * discrete Little's law: with dt = 1 over the whole run, the sum over samples of depth equals the sum of queue waits;
  * the paper's qualitative picture: under PRIORITY the Premium queue stays shortest and the Batch
    queue longest in overload; depth is 0 once the last request has been admitted.
"""
import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import server


def _sim(req, sv, combos):
    req = np.asarray(req, np.int64).reshape(-1, 5)
    inst = np.zeros(len(combos), wl.INSTANCE_DTYPE)
    for i, (p, e, a) in enumerate(combos):
        inst[i] = (0, p, e, 0, a)
    n = len(req)
    out_off = np.arange(len(combos) + 1, dtype=np.int64) * n
    tr = ([0, n], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4])
    st, dn, ema = oracle.simulate(*tr, sv, inst, out_off=out_off)
    return req, tr, inst, out_off, st


def test_h1_by_hand():
    # H1: r0=(0,Std) r1=(1000,Prem) r2=(1500,Batch), max_batch 2, FIFO -> start = (0, 2174, 4539)
    req, tr, inst, out_off, st = _sim([[0, 1, 3, 4, 2], [1000, 0, 8, 10, 1], [1500, 2, 2, 3, 2]], server(max_batch=2),
                                      [(wl.FIFO, wl.EXACT, 0.0)])
    assert st.tolist() == [0, 2174, 4539]
    d = oracle.queue_depth(*tr, inst, out_off, st, 0, 500, 12)           # t = 0, 500, ..., 5500
    prem = [0, 0, 1, 1, 1, 0, 0, 0, 0, 0, 0, 0]                           # queued on [1000, 2174): t = 1000, 1500, 2000
    batch = [0, 0, 0, 1, 1, 1, 1, 1, 1, 1, 0, 0]                          # queued on [1500, 4539): t = 1500 .. 4500
    assert d[0, :, 0].tolist() == prem and d[0, :, 1].tolist() == [0] * 12 and d[0, :, 2].tolist() == batch
    # a grid that starts before the trace and one sample exactly on the admission tick (admitted => no longer queued)
    d = oracle.queue_depth(*tr, inst, out_off, st, -1000, 2174, 4)        # t = -1000, 1174, 3348, 5522
    assert d[0, :, 0].tolist() == [0, 1, 0, 0] and d[0, :, 2].tolist() == [0, 0, 1, 0]
    d = oracle.queue_depth(*tr, inst, out_off, st, 2174, 1, 1)
    assert d[0, 0].tolist() == [0, 0, 1]


@pytest.mark.parametrize("policy", wl.ALL_POLICIES)
def test_counting_identity_and_littles_law(policy):
    sv = wl.Server(max_batch=4, kv_budget=2000, aging_step=30_000)
    c = wl._trace_workload("t", 11, 2, 300, sv, [(policy, wl.SPLIT, 0.1)], oracle.characterize, rho=1.2)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    st, dn, ema = oracle.simulate(*tr, sv, c.instances, out_off=c.out_off)
    t_end = int(st.max()) + 3
    for t0, dt, ns in ((0, 7919, t_end // 7919 + 2), (-12345, 100_003, t_end // 100_003 + 3), (5, 1, 0)):
        d = oracle.queue_depth(*tr, c.instances, c.out_off, st, t0, dt, ns)
        t = t0 + dt * np.arange(ns)
        for i in range(c.n_inst):
            lo, hi = c.trace_off[c.instances["trace"][i]], c.trace_off[c.instances["trace"][i] + 1]
            for k in range(3):
                m = c.tier[lo:hi] == k
                a = np.sort(c.arrival[lo:hi][m])
                s = np.sort(st[c.out_off[i]:c.out_off[i + 1]][m])
                want = np.searchsorted(a, t, side="right") - np.searchsorted(s, t, side="right")
                assert np.array_equal(d[i, :, k], want)
        assert (d >= 0).all()
    # Little's law on a window of the first 400 000 ticks: requests clipped to the window
    T = 400_000
    d = oracle.queue_depth(*tr, c.instances, c.out_off, st, 0, 1, T)
    for i in range(c.n_inst):
        lo, hi = c.trace_off[c.instances["trace"][i]], c.trace_off[c.instances["trace"][i] + 1]
        a = np.minimum(c.arrival[lo:hi], T)
        s = np.minimum(st[c.out_off[i]:c.out_off[i + 1]], T)
        for k in range(3):
            assert int(d[i, :, k].sum()) == int((s - a)[c.tier[lo:hi] == k].sum())


def test_priority_keeps_premium_queue_short():
    sv = wl.Server(max_batch=8, kv_budget=0)
    c = wl._trace_workload("t", 5, 1, 2000, sv, [(wl.PRIORITY, wl.EXACT, 0.0), (wl.FIFO, wl.EXACT, 0.0)], oracle.characterize, rho=1.3)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    st, dn, ema = oracle.simulate(*tr, sv, c.instances, out_off=c.out_off)
    t_end = int(st.max())
    d = oracle.queue_depth(*tr, c.instances, c.out_off, st, 0, t_end // 400, 402).astype(np.float64)
    mean = d.mean(axis=1)                                    # [instance, tier]
    assert mean[0, 0] < 0.2 * mean[0, 1] < mean[0, 2]        # PRIORITY: Premium drains first, Batch piles up
    share = np.array([0.2, 0.5, 0.3])
    assert np.allclose(mean[1] / mean[1].sum(), share, atol=0.08)   # FIFO: depth follows the tenant mix
    assert (d[:, -1, :] == 0).all()                          # after the last admission nothing is queued


def test_bad_arguments():
    req, tr, inst, out_off, st = _sim([[0, 0, 1, 1, 1]], server(), [(wl.FIFO, wl.EXACT, 0.0)])
    with pytest.raises(ValueError):
        oracle.queue_depth(*tr, inst, out_off, st, 0, 0, 4)
