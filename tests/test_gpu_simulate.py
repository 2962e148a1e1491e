"""-m gpu: ds_simulate (through the C ABI) vs the oracle: bit-exact ticks, 0-ulp EMA factors."""
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2606_02982_b200 import workload as wl


@pytest.fixture(scope="module")
def G():
    import _gpuutil
    return _gpuutil


def _oracle(c, want_traj=False):
    return oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances,
                           want_traj=want_traj)


def _assert_same(g, o, c):
    for name, a, b in (("start", g[0], o[0]), ("done", g[1], o[1])):
        bad = np.flatnonzero(a != b)
        assert bad.size == 0, (name, bad[:5], a[bad[:5]], b[bad[:5]], c.instances[bad[:5] // c.n_req])
    assert np.array_equal(g[2].view(np.uint64), o[2].view(np.uint64))    # 0 ulp


def test_hand_traces(G, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "hand_traces.json")))
    for case in g["cases"]:
        sv = wl.Server(**{k: v for k, v in case["server"].items() if k != "weight"})
        if "weight" in case["server"]:
            sv.weight = tuple(case["server"]["weight"])
        c = G.tiny_workload(wl, case["req"], sv, [(case["policy"], case["estimator"], case["alpha"])])
        st, dn, ema = G.gpu_simulate(c)
        assert st.tolist() == case["start"] and dn.tolist() == case["done"], case["name"]
        if "ema" in case:                                   # H14: completions at one tick applied in ascending request index
            assert ema[0].tolist() == case["ema"], case["name"]
        if "est" in case:                                   # frozen admission-time estimates (H7: R-ORD) through ds_simulate_est
            import paper_2606_02982_b200 as ds
            d = G.upload(c)
            st2, dn2, _, est = ds.simulate_est(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"],
                                               c.server, d["inst"], d["out_off"], int(c.out_off[-1]))
            assert ds.device_status() == 0
            assert est.cpu().tolist() == case["est"] and st2.cpu().tolist() == case["start"], case["name"]


def test_cfg0_full(G):
    c = wl.config0(oracle.characterize)
    _assert_same(G.gpu_simulate(c), _oracle(c), c)


@pytest.mark.parametrize("max_batch,kv", [(1, 0), (3, 700), (8, 0), (32, 16384), (32, 3000), (64, 9000), (128, 65536),
                                          (200, 20000), (256, 131072)])
def test_policy_sweep_small(G, max_batch, kv):
    sv = wl.Server(max_batch=max_batch, kv_budget=kv, aging_step=40_000)
    combos = [(p, e, a) for p in wl.ALL_POLICIES for e, a in ((wl.SPLIT, 0.1), (wl.EXACT, 0.1), (wl.SPLIT, 0.5), (wl.SPLIT, 0.0))]
    for rho in (0.85, 1.4):
        c = wl._trace_workload("t", 17 + max_batch, 3, 600, sv, combos, oracle.characterize, rho=rho)
        _assert_same(G.gpu_simulate(c), _oracle(c), c)


def test_pareto_outputs_deep_queues(G):
    # configs[3] shape scaled down: heavy tail, overload -> SJF heap beyond its shared-memory part
    sv = wl.Server(max_batch=16, kv_budget=6000, aging_step=250_000)
    combos = [(p, wl.SPLIT, a) for p in wl.ALL_POLICIES for a in (0.05, 0.5)]
    c = wl._trace_workload("t", 33, 2, 3000, sv, combos, None, rho=1.6, out_dist=1, materialise=False)
    _assert_same(G.gpu_simulate(c), _oracle(c), c)


def test_drift_trajectories(G):
    c = wl.config4(oracle.characterize, n_traces=2, n_req=3000, materialise=True, traj_every=100)
    c.server.max_batch = 64
    c.server.kv_budget = 20000
    toff = oracle.traj_offsets(c.trace_off, c.instances, 100)
    g = G.gpu_simulate(c, traj_off=toff)
    o = _oracle(c, want_traj=True)
    _assert_same(g, o, c)
    assert np.array_equal(g[3].view(np.uint64), o[3].view(np.uint64))
    # split()+EMA follows the drift 1.40 -> 2.14; exact estimator stays at 1.0 (Fig. 5/7)
    split = c.instances["estimator"] == wl.SPLIT
    assert (g[2][~split] == 1.0).all() and (g[2][split] > 1.9).all()


def test_equal_ticks_zero_lengths_and_ties(G):
    # equal arrival ticks, W=0 / P=0 prompts (A14), identical estimates (tie -> lower index), O=1
    rng = np.random.default_rng(5)
    n = 500
    req = np.stack([np.sort(rng.integers(0, 40, n)) * 50_000, rng.integers(0, 3, n), rng.integers(0, 3, n),
                    rng.integers(0, 4, n), rng.integers(1, 4, n)], 1)
    for mb, kv in ((1, 0), (4, 6), (32, 0)):
        sv = wl.Server(max_batch=mb, kv_budget=kv, aging_step=7000)
        c = G.tiny_workload(wl, req, sv, [(p, e, 0.3) for p in wl.ALL_POLICIES for e in (wl.SPLIT, wl.EXACT)])
        _assert_same(G.gpu_simulate(c), _oracle(c), c)


def test_estimates_above_the_kv_budget(G):
    # A8 progress guarantee + head-of-line blocking at scale: a budget so small that many estimates alone exceed it (they are
    # admitted only into an empty server) and nearly every admission is a KV decision
    for mb, kv, seed in ((4, 150, 3), (32, 120, 4), (128, 180, 5)):
        sv = wl.Server(max_batch=mb, kv_budget=kv, aging_step=60_000)
        combos = [(p, e, 0.2) for p in wl.ALL_POLICIES + [wl.AGING_UNCLAMPED] for e in (wl.SPLIT, wl.EXACT)]
        c = wl._trace_workload("t", seed, 2, 500, sv, combos, oracle.characterize, rho=0.4)
        assert (c.tokens > kv).mean() > 0.05 and (c.words > kv).any()
        _assert_same(G.gpu_simulate(c), _oracle(c), c)


def test_same_tick_arrivals_and_completions_random(G):
    # R-ORD at scale (H7 repeated with random sizes): triplets far apart on an idle batch-1 server; a arrives at T, its
    # completion tick T+S(a) is known in closed form; c arrives one tick before it (old factor), b exactly on it (new factor)
    from _simutil import service_time
    rng = np.random.default_rng(12)
    sv = wl.Server(max_batch=1, kv_budget=0, aging_step=50_000)
    rows = []
    for k in range(130):
        T, tier = k * 100_000, int(rng.integers(0, 3))
        W, P, O = rng.integers(1, 200, 3), rng.integers(1, 300, 3), rng.integers(1, 8, 3)
        S = service_time(int(P[0]), int(O[0]), sv)
        rows += [[T, tier, W[0], P[0], O[0]], [T + S - 1, tier, W[1], P[1], O[1]], [T + S, tier, W[2], P[2], O[2]]]
    combos = [(p, wl.SPLIT, a) for p in wl.ALL_POLICIES for a in (0.5, 0.9)]
    c = G.tiny_workload(wl, rows, sv, combos)
    o = _oracle(c)
    assert all(np.isin(c.arrival, o[1][i * c.n_req:(i + 1) * c.n_req]).sum() >= 130 for i in range(c.n_inst))
    _assert_same(G.gpu_simulate(c), o, c)


def test_many_completions_at_one_boundary(G):
    # more than 32 requests finishing at the same iteration boundary (equal out_len, admitted together): the retire list's
    # overflow path, with EMA on so that the ascending-index order of the completions is visible in the factors
    rng = np.random.default_rng(8)
    n = 600
    arr = np.repeat(np.arange(n // 200) * 3_000_000, 200)                     # bursts of 200 simultaneous arrivals
    req = np.stack([arr, rng.integers(0, 3, n), rng.integers(1, 9, n), rng.integers(1, 12, n), np.where(rng.random(n) < 0.8, 2, 3)], 1)
    for mb in (48, 64, 128, 256):
        sv = wl.Server(max_batch=mb, kv_budget=0, aging_step=9000, traj_every=7)
        c = G.tiny_workload(wl, req, sv, [(p, wl.SPLIT, 0.4) for p in wl.ALL_POLICIES])
        toff = oracle.traj_offsets(c.trace_off, c.instances, 7)
        g = G.gpu_simulate(c, traj_off=toff)
        o = _oracle(c, want_traj=True)
        _assert_same(g, o, c)
        assert np.array_equal(g[3].view(np.uint64), o[3].view(np.uint64))
        per = o[1].reshape(c.n_inst, n)
        assert max(np.unique(per[0], return_counts=True)[1]) > 32           # the case does put > 32 completions on one tick


def test_bad_arguments(G):
    import paper_2606_02982_b200 as ds
    c = wl.config0(oracle.characterize)
    c.server.max_batch = 0
    with pytest.raises(ds.DsError):
        G.gpu_simulate(c)
    c.server.max_batch = 8
    c.instances["policy"][0] = 9
    d = G.upload(c)
    ds.simulate(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server, d["inst"],
                d["out_off"], int(c.out_off[-1]))
    assert ds.device_status() & 8


def test_workspace_and_output_ranges_are_validated(G):
    # the whole documented workspace is required (header + permutation + SJF heap slots): one byte short => DS_ENOMEM, no launch
    import torch
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import _lib
    sv = wl.Server(max_batch=4, kv_budget=0)
    c = wl._trace_workload("t", 41, 1, 2000, sv, [(wl.SJF, wl.SPLIT, 0.1)], None, rho=3.0, materialise=False)   # overload: queue > 256
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    need = ds.simulate_workspace_bytes(n_total, c.n_inst, c.n_traces * c.n_req)      # both mandatory parts
    args = (d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server, d["inst"], d["out_off"], n_total)
    with pytest.raises(ds.DsError) as e:
        ds.simulate(*args, workspace=torch.empty(need - 1, dtype=torch.uint8, device=G.DEV))
    assert e.value.code == _lib.DS_ENOMEM
    st, dn, ema = ds.simulate(*args, workspace=torch.empty(need, dtype=torch.uint8, device=G.DEV))
    assert ds.device_status() == 0
    o = _oracle(c)
    assert np.array_equal(st.cpu().numpy(), o[0]) and np.array_equal(dn.cpu().numpy(), o[1])
    # an instance whose output range leaves [0, n_total) is skipped and reported, nothing is written outside the arrays
    canary = torch.full((n_total + 64,), -7, dtype=torch.int64, device=G.DEV)
    st2, dn2, _ = ds.simulate(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server, d["inst"],
                              d["out_off"], n_total - 1, start=canary[:n_total - 1], done=torch.empty(n_total, dtype=torch.int64, device=G.DEV)[:n_total - 1])
    assert ds.device_status() & 16
    assert bool((canary == -7).all())


def test_decreasing_arrivals_are_reported(G):
    # the monotone-arrival contract is checked on every pair of neighbouring requests, also across the 32-request windows
    import paper_2606_02982_b200 as ds
    sv = wl.Server(max_batch=4, kv_budget=0)
    for bad_at in (5, 32, 64, 96):            # inside a window, and on lane 0 of a window (pair (31, 32) etc.)
        c = wl._trace_workload("t", 43, 1, 200, sv, [(p, wl.EXACT, 0.0) for p in wl.ALL_POLICIES], None, rho=0.8, materialise=False)
        c.arrival[bad_at] = c.arrival[bad_at - 1] - 1
        d = G.upload(c)
        ds.simulate(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server, d["inst"], d["out_off"],
                    int(c.out_off[-1]))
        assert ds.device_status() & 2, bad_at


def test_large_costs_take_the_64bit_path(G):
    # cost constants near 2^31 and one huge out_len: the per-trace bound fails, so the kernel must use its 64-bit state
    sv = wl.Server(max_batch=6, kv_budget=9000, aging_step=3_000_000_000, c_base=2_000_000_000, c_batch=150_000_000,
                   c_ctx=1_000_003, c_prefill=5_000_000)
    combos = [(p, e, 0.2) for p in wl.ALL_POLICIES for e in (wl.SPLIT, wl.EXACT)]
    c = wl._trace_workload("t", 77, 2, 400, sv, combos, oracle.characterize, mean_ticks=3.0e10)
    c.out_len[5] = 70_000                                                  # > 65535
    _assert_same(G.gpu_simulate(c), _oracle(c), c)
    import paper_2606_02982_b200 as ds
    sv.c_base = 1 << 31                                                    # not representable: rejected on the host
    with pytest.raises(ds.DsError):
        G.gpu_simulate(c)
