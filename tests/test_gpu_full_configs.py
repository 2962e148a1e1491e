"""-m gpu: BASELINE.json configs at FULL size through the C ABI, in the launch configuration bench.py uses.

The oracle cannot run 10^9 simulated requests in minutes, so (as the tier rules allow) the full-size runs are
checked (a) on sampled instances / prompt ranges that the oracle computes one by one, bit for bit, and (b) through
properties that hold at any size (conservation, FIFO order, EXACT => B == 1.0). Each test skips itself when the
box lacks the memory for that configuration.
"""
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


def _need(gpu_gb, host_gb):
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < gpu_gb * 2**30:
        pytest.skip(f"needs {gpu_gb} GiB of free GPU memory")
    try:
        avail = os.sysconf("SC_AVPHYS_PAGES") * os.sysconf("SC_PAGE_SIZE")
        if avail < host_gb * 2**30:
            pytest.skip(f"needs {host_gb} GiB of host memory")
    except (ValueError, OSError):
        pass


def _sim_full(G, c, want_traj=False):
    """Run ds_simulate on the whole workload; outputs stay on the device."""
    import torch
    import paper_2606_02982_b200 as ds
    d = G.upload(c)
    n_total = int(c.out_off[-1])
    toff = traj = None
    if want_traj:
        toff_h = oracle.traj_offsets(c.trace_off, c.instances, c.server.traj_every)
        toff = torch.from_numpy(toff_h).to(G.DEV)
        traj = torch.zeros((int(toff_h[-1]), 3), dtype=torch.float64, device=G.DEV)
    st, dn, ema = ds.simulate(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server,
                              d["inst"], d["out_off"], n_total, traj_off=toff, ema_traj=traj)
    assert ds.device_status() == 0
    return d, st, dn, ema, traj


def _check_sample(c, st, dn, ema, sample, traj=None):
    """Oracle, instance by instance, on the sampled instance ids; element-by-element comparison."""
    nr = c.n_req
    for i in sample:
        inst = c.instances[i:i + 1].copy()
        t = int(inst["trace"][0])
        rs = slice(t * nr, (t + 1) * nr)
        inst["trace"] = 0
        o = oracle.simulate(np.array([0, nr], np.int64), c.arrival[rs], c.tier[rs], c.words[rs], c.tokens[rs], c.out_len[rs],
                            c.server, inst, want_traj=traj is not None)
        a = slice(i * nr, (i + 1) * nr)
        gs, gd = st[a].cpu().numpy(), dn[a].cpu().numpy()
        assert np.array_equal(gs, o[0]), (i, c.instances[i], np.flatnonzero(gs != o[0])[:5])
        assert np.array_equal(gd, o[1]), (i, c.instances[i], np.flatnonzero(gd != o[1])[:5])
        assert np.array_equal(ema[i].cpu().numpy().view(np.uint64), o[2][0].view(np.uint64)), (i, c.instances[i])   # 0 ulp
        if traj is not None:
            k = nr // c.server.traj_every
            g = traj[i * k:(i + 1) * k].cpu().numpy()
            assert np.array_equal(g.view(np.uint64), o[3].view(np.uint64)), (i, c.instances[i])


def _check_properties(c, d, st, dn, ema):
    """Invariants I1, I3 and A4 over every simulated request of the full run (device-side reductions)."""
    import torch
    nr, ni = c.n_req, c.n_inst
    tr = torch.from_numpy(c.instances["trace"].astype(np.int64)).to(st.device)
    arr = d["arrival"].view(c.n_traces, nr)
    chunk = max(1, (1 << 27) // nr)
    pol = torch.from_numpy(c.instances["policy"].astype(np.int64)).to(st.device)
    for a in range(0, ni, chunk):
        b = min(ni, a + chunk)
        s = st[a * nr:b * nr].view(b - a, nr)
        e = dn[a * nr:b * nr].view(b - a, nr)
        ar = arr[tr[a:b]]
        assert bool((ar <= s).all()) and bool((s < e).all())                       # I1: arrival <= start < done
        fifo = pol[a:b] == wl.FIFO
        if bool(fifo.any()):
            sf = s[fifo]
            assert bool((sf[:, 1:] >= sf[:, :-1]).all())                           # I3: FIFO starts in arrival order
    exact = torch.from_numpy(c.instances["estimator"] == wl.EXACT).to(st.device)
    assert bool((ema[exact] == 1.0).all())                                         # A4: exact estimator keeps B == 1.0


def test_cfg1_full_pipeline(G):
    """configs[1]: 1024 traces x 2000 requests x 10 instances, whole hot path (the bench.py step)."""
    _need(6, 6)
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200.pipeline import HotPath
    c = wl.config1(G.gpu_characterize)                      # W,P of the 1.13 GB of text come from ds_characterize
    rng = np.random.default_rng(1)
    # characterization: a sample of traces against the oracle, prompt by prompt
    for t in rng.choice(c.n_traces, 24, replace=False):
        a, b = t * c.n_req, (t + 1) * c.n_req
        lo, hi = c.offsets[a], c.offsets[b]
        ow, ot = oracle.characterize(c.text[lo:hi], c.offsets[a:b + 1] - lo)
        assert np.array_equal(ow, c.words[a:b]) and np.array_equal(ot, c.tokens[a:b])
    hp = HotPath(c, G.DEV)
    hp.step()
    assert ds.device_status() == 0
    assert np.array_equal(hp.words.cpu().numpy(), c.words) and np.array_equal(hp.tokens.cpu().numpy(), c.tokens)
    d = {"arrival": hp.arrival}
    _check_properties(c, d, hp.start, hp.done, hp.ema_final)
    sample = [int(t) * 10 + k for t in rng.choice(c.n_traces, 16, replace=False) for k in range(10)]
    _check_sample(c, hp.start, hp.done, hp.ema_final, sample)
    # percentiles of the FULL run: the oracle sorts the 20.48 M latencies the GPU produced
    st, dn = hp.start.cpu().numpy(), hp.done.cpu().numpy()
    e2e, qd, seg_t, seg_a = oracle.latencies(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.instances,
                                             c.out_off, st, dn, c.group)
    hp2 = HotPath(c, G.DEV, fused=False)                      # unfused ds_latencies + ds_tail_stats give the same numbers
    hp2.step()
    assert np.array_equal(hp2.e2e.cpu().numpy(), e2e) and np.array_equal(hp2.seg_tier.cpu().numpy(), seg_t)
    assert np.array_equal(hp2.qdelay.cpu().numpy(), qd) and np.array_equal(hp2.seg_all.cpu().numpy(), seg_a)
    for name, vals, seg, ns in (("e2e_tier", e2e, seg_t, 30), ("e2e_all", e2e, seg_a, 10), ("qdelay_tier", qd, seg_t, 30),
                                ("qdelay_all", qd, seg_a, 10)):
        o, cnt = oracle.tail_stats(vals, seg, ns)
        for h in (hp, hp2):
            assert np.array_equal(h.stats[name].cpu().numpy(), o), name
            assert np.array_equal(h.counts[name].cpu().numpy(), cnt), name


def test_cfg2_full_scan(G):
    """configs[2]: 8 GiB packed text, ~7 M prompts; every prompt compared with the oracle."""
    _need(10, 20)
    import torch
    import paper_2606_02982_b200 as ds
    buf, off = wl.config2()
    assert buf.size == 8 << 30
    t = torch.from_numpy(buf).to(G.DEV)
    o = torch.from_numpy(off).to(G.DEV)
    w, k = ds.characterize(t, o)
    assert ds.device_status() == 0
    gw, gk = w.cpu().numpy(), k.cpu().numpy()
    del t, o
    n = len(off) - 1
    step = 1 << 20                                            # oracle in slices of 2^20 prompts (it is a per-byte loop)
    for a in range(0, n, step):
        b = min(n, a + step)
        ow, ot = oracle.characterize(buf[off[a]:off[b]], off[a:b + 1] - off[a])
        assert np.array_equal(gw[a:b], ow), (a, np.flatnonzero(gw[a:b] != ow)[:5])
        assert np.array_equal(gk[a:b], ot), (a, np.flatnonzero(gk[a:b] != ot)[:5])


def test_cfg3_full_heavy_contention(G):
    """configs[3]: 16384 traces x 10^4 requests x 20 instances (3.28 G simulated requests), batch 128, Pareto outputs."""
    _need(100, 24)
    c = wl.config3()
    assert c.n_inst == 327_680 and c.sim_requests == 3_276_800_000
    d, st, dn, ema, _ = _sim_full(G, c)
    _check_properties(c, d, st, dn, ema)
    rng = np.random.default_rng(3)
    sample = [int(t) * 20 + k for t in rng.choice(c.n_traces, 2, replace=False) for k in range(20)]
    sample += [int(i) for i in rng.choice(c.n_inst, 24, replace=False)]
    _check_sample(c, st, dn, ema, sample)


def test_cfg4_full_drift(G):
    """configs[4]: 4096 traces x 50000 requests x 10 instances (2.05 G), batch 256, EMA trajectories every 1000."""
    _need(70, 24)
    c = wl.config4()
    assert c.n_inst == 40_960 and c.sim_requests == 2_048_000_000
    d, st, dn, ema, traj = _sim_full(G, c, want_traj=True)
    _check_properties(c, d, st, dn, ema)
    rng = np.random.default_rng(4)
    sample = [int(t) * 10 + k for t in rng.choice(c.n_traces, 1, replace=False) for k in range(10)]
    sample += [int(i) for i in rng.choice(c.n_inst, 6, replace=False)]
    _check_sample(c, st, dn, ema, sample, traj)
    # split()+EMA tracks the drift 1.40 -> 2.14 (north_star invariant); trajectories start near 1.40
    split = c.instances["estimator"] == wl.SPLIT
    e = ema.cpu().numpy()
    assert (e[split] > 1.9).all() and (e[split] < 2.4).all()
    k = c.n_req // c.server.traj_every
    t0 = traj.view(c.n_inst, k, 3)[:, k // 2 - 2, :].cpu().numpy()      # just before the midpoint
    assert (np.abs(t0[split] - 1.3977) < 0.25).all()
