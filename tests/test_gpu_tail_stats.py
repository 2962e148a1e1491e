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


def _fused_vs_oracle(G, c, pct=(50, 99)):
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import workload as wl
    st, dn, _ = oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances)
    e2e, qd, seg_t, seg_a = oracle.latencies(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.instances, c.out_off,
                                             st, dn, c.group, c.t_mid)
    Gn = c.n_groups * (2 if c.t_mid is not None else 1)
    d = G.upload(c)
    import torch
    for stage in (True, False):      # with and without the staging area (32-bit keys + segment codes) behind the histograms
        ge, gq, gc = ds.latency_stats(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], d["inst"],
                                      d["out_off"], torch.from_numpy(st).to(G.DEV), torch.from_numpy(dn).to(G.DEV), d["group"],
                                      c.n_groups, d["t_mid"], pct, stage=stage)
        ge, gq, gc = ge.cpu().numpy(), gq.cpu().numpy(), gc.cpu().numpy()
        for vals, got in ((e2e, ge), (qd, gq)):
            ot, ct = oracle.tail_stats(vals, seg_t, 3 * Gn, pct)
            oa, ca = oracle.tail_stats(vals, seg_a, Gn, pct)
            assert np.array_equal(got[:3 * Gn], ot) and np.array_equal(got[3 * Gn:], oa)
            assert np.array_equal(gc[:3 * Gn], ct) and np.array_equal(gc[3 * Gn:], ca)


def test_fused_latency_stats(G):
    from paper_2606_02982_b200 import workload as wl
    sv = wl.Server(max_batch=8, kv_budget=3000)
    combos = [(p, e, 0.1) for p in wl.ALL_POLICIES for e in (wl.SPLIT, wl.EXACT)]
    c = wl._trace_workload("t", 5, 7, 1500, sv, combos, oracle.characterize, rho=1.1)          # ragged block tails
    _fused_vs_oracle(G, c)
    c2 = wl._trace_workload("t", 8, 3, 700, sv, combos[:3], oracle.characterize, rho=0.9)
    _fused_vs_oracle(G, c2, pct=(0, 1, 50, 95, 99, 100))
    c4 = wl.config4(oracle.characterize, n_traces=3, n_req=2500, materialise=True, traj_every=0)   # pre/post-drift phases
    c4.server.max_batch = 32
    _fused_vs_oracle(G, c4)
    c1 = wl._trace_workload("t", 6, 1, 40, sv, [(wl.FIFO, wl.EXACT, 0.0)], oracle.characterize, rho=0.5)
    c1.tier[:] = 1                                                                               # tiers 0 and 2 empty -> -1
    _fused_vs_oracle(G, c1)


def test_fused_latency_stats_runs_of_equal_keys(G):
    """Queue delay 0 for nearly every request (an idle server), plus one burst trace whose delays are large: after the first
    digit every lane of a warp holds the SAME key, the case in which the digit passes must aggregate their adds instead of
    using plain atomics (tail_stats.cu: concentrated()). Also p50 = 0 and p99 among the outliers: both ends of the range."""
    from paper_2606_02982_b200 import workload as wl
    sv = wl.Server(max_batch=64, kv_budget=0)
    combos = [(p, wl.EXACT, 0.0) for p in (wl.FIFO, wl.SJF, wl.PRIORITY)]
    c = wl._trace_workload("t", 12, 6, 2000, sv, combos, oracle.characterize, mean_ticks=40_000_000.0)   # one request at a time
    a = c.arrival.reshape(6, 2000)
    a[5] = np.sort(a[5] // 4000)                                   # the burst: 2000 requests within 1/4000 of the time
    c.arrival = a.reshape(-1)
    st, dn, _ = oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances)
    qd = (st.reshape(c.n_inst, 2000) - a[c.instances["trace"]])
    assert (qd[c.instances["trace"] < 5] == 0).mean() > 0.99 and qd[c.instances["trace"] == 5].max() > 1_000_000
    _fused_vs_oracle(G, c)
    _fused_vs_oracle(G, c, pct=(1, 50, 90, 99, 100))


def test_fused_staging_edge_cases(G):
    """The staging area of ds_latency_stats: keys that need more than 32 bits, padded and out-of-order out_off, a staging
    area that is too small - every case must give the oracle's percentiles (the unstaged passes take over)."""
    import torch
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import workload as wl
    from paper_2606_02982_b200 import _lib
    sv = wl.Server(max_batch=8, kv_budget=3000)
    combos = [(p, wl.SPLIT, 0.1) for p in (wl.FIFO, wl.SJF, wl.AGING)]
    c = wl._trace_workload("t", 15, 4, 900, sv, combos, oracle.characterize, rho=1.2)
    st, dn, _ = oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances)
    n_inst, n_req, Gn, pct = len(c.instances), 900, c.n_groups, (50, 95, 99)

    def check(st_h, dn_h, out_off_h, ws_extra, tier_h=None):
        tier_h = c.tier if tier_h is None else tier_h
        n_tot = int(max(out_off_h[:-1]) + n_req) if len(out_off_h) > 1 else 0
        n_tot = max(n_tot, int(out_off_h[-1]))
        S = np.full(n_tot, -7, np.int64); D = np.full(n_tot, -7, np.int64)
        for i in range(n_inst):
            S[out_off_h[i]:out_off_h[i] + n_req] = st_h[i * n_req:(i + 1) * n_req]
            D[out_off_h[i]:out_off_h[i] + n_req] = dn_h[i * n_req:(i + 1) * n_req]
        e2e, qd, seg_t, seg_a = oracle.latencies(c.trace_off, c.arrival, tier_h, c.words, c.tokens, c.out_len, c.instances,
                                                 out_off_h, S, D, c.group, c.t_mid)
        d = G.upload(c)
        d["tier"] = torch.from_numpy(tier_h).to(G.DEV)
        nb = ds.api.workspace_bytes(_lib.WS_TAIL_STATS, 4 * Gn, len(pct)) + ws_extra
        ws = torch.empty(nb, dtype=torch.uint8, device=G.DEV)
        ge, gq, gc = ds.latency_stats(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], d["inst"],
                                      torch.from_numpy(out_off_h).to(G.DEV), torch.from_numpy(S).to(G.DEV), torch.from_numpy(D).to(G.DEV),
                                      d["group"], c.n_groups, d["t_mid"], pct, workspace=ws)
        sel = np.zeros(n_tot, bool)
        for i in range(n_inst):
            sel[out_off_h[i]:out_off_h[i] + n_req] = True
        for vals, got in ((e2e, ge.cpu().numpy()), (qd, gq.cpu().numpy())):
            v, a, b = vals[sel], seg_t[sel], seg_a[sel]
            ot, ct = oracle.tail_stats(v, a, 3 * Gn, pct)
            oa, ca = oracle.tail_stats(v, b, Gn, pct)
            assert np.array_equal(got[:3 * Gn], ot) and np.array_equal(got[3 * Gn:], oa)
            assert np.array_equal(gc.cpu().numpy()[:3 * Gn], ct) and np.array_equal(gc.cpu().numpy()[3 * Gn:], ca)

    full = ds.api.workspace_bytes(_lib.WS_LATENCY_STAGE, 2 * n_inst * n_req + 64, 0)
    off = c.out_off.copy()
    check(st, dn, off, full)                                             # staged
    check(st, dn, off, 5 * 100)                                          # staging area too small -> unstaged passes
    pad = (np.arange(n_inst + 1, dtype=np.int64) * (n_req + 37)) + 11    # gap before the first range and between ranges
    check(st, dn, pad, full)
    perm = c.out_off[:-1][::-1].copy()                                   # ranges not in instance order -> unstaged passes
    check(st, dn, np.concatenate([perm, c.out_off[-1:]]), full)
    big = dn.copy(); big[5::7] += 1 << 33                                # keys differ above bit 31 -> unstaged passes
    check(st, big, off, full)
    shifted_st, shifted_dn = st + (1 << 40), dn + (1 << 40)              # common high bits, low 32 vary: still staged
    check(shifted_st, shifted_dn, off, full)
