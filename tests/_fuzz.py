"""Randomised differential cases for K2: ds_simulate_est (frozen and re-estimated), ds_simulate_budget and ds_simulate_closed through
the C ABI against the oracle, bit-exact / 0 ulp. One seed = one call: 1-4 ragged traces (lengths around the 32-request window and
the 256-entry shared part of the SJF heap), arrival laws with many equal ticks and bursts, zero words / zero tokens, output lengths
from constant 1 to a heavy tail, every policy x three estimator settings, servers from max_batch 1 to 256 with zero and extreme cost
constants, tight KV budgets (est > kv_budget included), random weights and aging steps, trajectories at a random stride.
Used by tests/test_gpu_fuzz.py; the seeds and everything derived from them are inputs only (no method arithmetic here)."""
import numpy as np
import torch

import oracle
import paper_2606_02982_b200 as ds
from paper_2606_02982_b200 import workload as wl
from paper_2606_02982_b200.api import instances_to_device

DEV = "cuda:0"
DS_DEV_BAD_TRACE = 2           # include/driftsched.h
pols = [wl.FIFO, wl.PRIORITY, wl.WEIGHTED, wl.SJF, wl.AGING, wl.AGING_UNCLAMPED]


def gen_trace(rng, n):
    mode = rng.integers(0, 5)
    if mode == 0:   gaps = rng.exponential(rng.choice([50, 800, 3000, 20000]), n)
    elif mode == 1: gaps = rng.integers(0, 3, n) * rng.choice([0, 1, 1000])           # many equal ticks
    elif mode == 2: gaps = np.where(rng.random(n) < 0.1, rng.exponential(200000, n), 0)  # bursts
    elif mode == 3: gaps = rng.integers(0, 5000, n)
    else:           gaps = rng.exponential(2500, n) * (1 + 3 * (np.arange(n) > n // 2))
    arr = np.cumsum(gaps.astype(np.int64)) + int(rng.integers(0, 3) * 1000)
    tp = rng.dirichlet(np.ones(3) * rng.choice([0.2, 1, 5]))
    tier = rng.choice(3, n, p=tp).astype(np.uint8)
    words = rng.integers(0 if rng.random() < 0.3 else 1, rng.choice([4, 40, 400]), n).astype(np.int32)
    ratio = rng.choice([1.0, 1.4, 2.1, 0.6])
    tokens = np.maximum(0 if rng.random() < 0.2 else 1, np.rint(words * ratio + rng.integers(-2, 3, n))).astype(np.int32)
    om = rng.integers(0, 4)
    if om == 0:   out = rng.integers(1, 4, n)
    elif om == 1: out = rng.integers(1, 200, n)
    elif om == 2: out = np.minimum((rng.pareto(1.5, n) * 20 + 1), 3000)
    else:         out = np.where(rng.random(n) < 0.5, 1, rng.integers(1, 60, n))
    return arr, tier, words, tokens, out.astype(np.int32)


stats = {"cases": 0, "requests": 0, "kind": [0, 0, 0, 0], "closed_loop_contract_violations": 0, "deferrals_possible": 0}


def _same(name, g, o, desc):
    g = g.cpu().numpy().reshape(-1)
    o = np.ascontiguousarray(o).reshape(-1)
    if g.dtype == np.float64:
        g, o = g.view(np.uint64), o.view(np.uint64)                       # 0 ulp
    bad = np.flatnonzero(g != o)
    assert bad.size == 0, (name, desc, bad[:5], g[bad[:5]], o[bad[:5]])


def one_case(seed, long_traces=False):
    rng = np.random.default_rng(seed)
    n_tr = int(rng.integers(1, 5))
    # long_traces: queues deeper than the 256 heap entries SJF keeps in shared memory, many 32-request windows, long clocks
    lens = [int(rng.choice([1500, 3000, 5000] if long_traces else [1, 2, 5, 31, 32, 33, 64, 100, 257, 700])) for _ in range(n_tr)]
    parts = [gen_trace(rng, n) for n in lens]
    trace_off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    arrival, tier, words, tokens, out_len = (np.concatenate([p[k] for p in parts]) for k in range(5))
    mb = int(rng.choice([1, 2, 3, 7, 8, 31, 32, 33, 64, 100, 128, 129, 200, 256]))
    kv = int(rng.choice([0, 0, 50, 300, 2000, 20000, 10 ** 6]))
    sv = wl.Server(max_batch=mb, kv_budget=kv, c_base=int(rng.choice([0, 1, 2000, 70000])), c_batch=int(rng.choice([0, 150, 3])),
                   c_ctx=int(rng.choice([0, 1, 40])), c_prefill=int(rng.choice([0, 5, 300])),
                   weight=tuple(int(x) for x in rng.integers(1, 6, 3)), aging_step=int(rng.choice([1, 1000, 40_000, 500_000, 10 ** 9])),
                   traj_every=int(rng.choice([0, 1, 3, 50])))
    if sv.c_base == 0 and sv.c_batch == 0:
        sv.c_base = 1
    kind = int(rng.integers(0, 4))      # 0 ds_simulate_est, 1 the same with reestimate = 1, 2 ds_simulate_budget, 3 ds_simulate_closed
    alphas = [float(rng.choice([0.0, 0.05, 0.1, 0.5, 1.0, rng.random()])) for _ in range(2)]
    if kind <= 1:
        combos = [(p, e, a) for p in pols for e, a in ((wl.SPLIT, alphas[0]), (wl.EXACT, alphas[1]), (wl.SPLIT, alphas[1]))]
    else:
        combos = [(p, e, a) for p in pols for e, a in ((wl.BUDGET_SPLIT, alphas[0]), (wl.BUDGET_EXACT, alphas[1]))]
    inst = np.zeros(n_tr * len(combos), wl.INSTANCE_DTYPE)
    k = 0
    for t in range(n_tr):
        for (p, e, a) in combos:
            inst[k] = (t, p, e, 0, a)
            k += 1
    sizes = np.diff(trace_off)[inst["trace"]]
    out_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    n_total = int(out_off[-1])
    T = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(DEV)
    d = [T(trace_off), T(arrival), T(tier), T(words), T(tokens), T(out_len)]
    di, doff = instances_to_device(inst, DEV), T(out_off)
    desc = (seed, kind, lens, sv)
    stats["cases"] += 1
    stats["requests"] += n_total
    stats["kind"][kind] += 1
    stats["deferrals_possible"] += int(kv > 0 and mb > 1)
    fac = 3 if kind <= 1 else 4
    toff = traj = None
    if sv.traj_every > 0:
        toff_h = oracle.traj_offsets(trace_off, inst, sv.traj_every)
        toff = T(toff_h)
        traj = torch.zeros((int(toff_h[-1]), fac), dtype=torch.float64, device=DEV)
    est = torch.full((n_total,), -1, dtype=torch.int64, device=DEV)
    if kind <= 1:
        sv.reestimate = kind
        o = oracle.simulate(trace_off, arrival, tier, words, tokens, out_len, sv, inst, want_traj=True, want_est=True)
        g = ds.simulate(*d, sv, di, doff, n_total, traj_off=toff, ema_traj=traj, est_out=est)
        assert ds.device_status() == 0, desc
        names, g = ("start", "done", "ema", "traj", "est"), g + (traj, est)
    else:
        cat = rng.integers(0, 4, arrival.size).astype(np.uint8)
        bp = wl.Budget(t_base=tuple(float(x) for x in rng.choice([0.0, 10.0, 38.0, 113.5, 265.0], 4)),
                       s_tenant=tuple(float(x) for x in rng.choice([1.0, 0.8, 1.25, 1.1], 3)),
                       f_slope=float(rng.choice([0.0, 0.001, 0.01])), f_max=float(rng.choice([1.0, 1.5, 3.0])))
        if kind == 2:
            o = oracle.simulate_budget(trace_off, arrival, tier, words, tokens, out_len, cat, bp, sv, inst, want_traj=True, want_est=True)
            g = ds.simulate_budget(*d, T(cat), bp, sv, di, doff, n_total, traj_off=toff, ema_traj=traj, est_out=est)
            assert ds.device_status() == 0, desc
            names, g = ("start", "done", "ema", "traj", "est"), g + (traj, est)
        else:
            ncl = int(rng.choice([1, 2, 7, 40, 300]))
            think = int(rng.choice([0, 100, 25000]))
            bw = int(rng.choice([0, 0, 3000, 10 ** 6]))
            arr2 = arrival.copy()                     # the first n_clients arrivals of a trace are the clients' start ticks
            for t in range(n_tr):
                a, b = trace_off[t], trace_off[t + 1]
                arr2[a:b] = np.sort(np.minimum(arr2[a:b], int(rng.choice([0, 0, 500]))))
            d[1] = T(arr2)
            desc = desc + (ncl, think, bw)
            o = oracle.simulate_budget(trace_off, arr2, tier, words, tokens, out_len, cat, bp, sv, inst, want_traj=True, want_est=True,
                                       n_clients=ncl, think_ticks=think, batch_wait=bw)
            st, dn, ema, arr_o = ds.simulate_closed(*d, T(cat), bp, sv, ncl, think, bw, di, doff, n_total, traj_off=toff, ema_traj=traj,
                                                    est_out=est)
            status = ds.device_status()
            # include/driftsched.h: a client's start tick after a release is DS_DEV_BAD_TRACE (the submission order would no
            # longer be the trace order). Seen from the oracle's output: some instance's submission ticks are not ascending.
            ascending = all(bool((np.diff(o[-1][out_off[i]:out_off[i + 1]]) >= 0).all()) for i in range(len(inst)))
            assert (status == 0) == ascending and status in (0, DS_DEV_BAD_TRACE), (status, ascending, desc)
            if status != 0:
                stats["closed_loop_contract_violations"] += 1
                return
            names, g = ("start", "done", "ema", "traj", "est", "arrival"), (st, dn, ema, traj, est, arr_o)
    for nm, a, b in zip(names, g, o):
        if a is None:                                 # no trajectory asked for
            assert nm == "traj" and (b is None or np.asarray(b).size == 0), desc
            continue
        _same(nm, a, b, desc)


def one_case_k1(seed):
    """ds_characterize on a random buffer: alphabet, size, prompt cuts (empty prompts, bytes outside every prompt) and base
    misalignment all drawn from the seed."""
    rng = np.random.default_rng([seed, 1])
    alphabets = (b" \t\n\r\x0b\x0c\x08\x0e\x1c\x1f\x7f\x80\x85\xa0\xff!/:@[`{~09AZaz_\x00,.", b"  ab", b"a", b" ", b"a,. \n",
                 bytes(range(256)), b"abcdefghijklmnopqrstuvwxyz      .,;")
    alpha = np.frombuffer(alphabets[int(rng.integers(0, len(alphabets)))], np.uint8)
    n = int(rng.choice([0, 1, 7, 4095, 4096, 4097, 8192, 12289, 50_000, 300_001, int(rng.integers(1, 400_000))]))
    mis = int(rng.choice([0, 0, 1, 5, 8, 15]))
    big = alpha[rng.integers(0, len(alpha), n + mis)] if rng.random() < 0.7 else np.repeat(
        alpha[rng.integers(0, len(alpha), (n + mis) // 37 + 1)], 37)[:n + mis]          # long runs of one byte
    buf = big[mis:mis + n]
    k = int(rng.choice([0, 1, 3, 50, max(1, n // 3), max(1, n)]))
    cuts = np.sort(rng.integers(0, n + 1, k)).astype(np.int64)
    lo, hi = (0, n) if rng.random() < 0.7 or k == 0 else (int(cuts[0]), int(cuts[-1]))
    off = np.concatenate([[lo], cuts, [hi]]).astype(np.int64)
    ow, ot = oracle.characterize(buf, off)
    t = torch.from_numpy(np.ascontiguousarray(big)).to(DEV)
    w, tk = ds.characterize(t[mis:mis + n], torch.from_numpy(off).to(DEV))
    assert ds.device_status() == 0, (seed, n, mis, k)
    assert np.array_equal(w.cpu().numpy(), ow) and np.array_equal(tk.cpu().numpy(), ot), (seed, n, mis, k)


def one_case_k3(seed):
    """ds_tail_stats (and the static entry point when the sizes fit) on random values / segments / percentiles."""
    rng = np.random.default_rng([seed, 3])
    n = int(rng.choice([0, 1, 2, 33, 1000, 70_000, int(rng.integers(1, 300_000))]))
    nseg = int(rng.choice([1, 2, 3, 16, 60, 128, 1000]))
    mode = int(rng.integers(0, 6))
    if mode == 0:   v = rng.integers(-10, 10, n)
    elif mode == 1: v = rng.integers(0, 1 << 25, n)
    elif mode == 2: v = (rng.pareto(1.2, n) * 1e4).astype(np.int64)
    elif mode == 3: v = rng.integers(np.iinfo(np.int64).min, np.iinfo(np.int64).max, n, dtype=np.int64, endpoint=True)
    elif mode == 4: v = np.full(n, int(rng.integers(-5, 5)) << int(rng.integers(0, 60)))
    else:           v = (1 << 40) + rng.integers(0, 3, n) * (1 << int(rng.integers(0, 30)))
    v = np.asarray(v, np.int64)
    seg = (rng.integers(0, nseg, n) if rng.random() < 0.6 else np.minimum(rng.geometric(0.3, n) - 1, nseg - 1)).astype(np.int32)
    if n:
        seg[rng.random(n) < rng.choice([0.0, 0.05, 0.9])] = int(rng.choice([-1, nseg, nseg + 7]))   # skipped values
    pct = tuple(int(x) for x in rng.choice([0, 1, 25, 50, 90, 95, 99, 100], int(rng.integers(1, 9)), replace=True))
    o, oc = oracle.tail_stats(v, seg, nseg, pct)
    dv, dseg = torch.from_numpy(v).to(DEV), torch.from_numpy(seg).to(DEV)
    g, gc = ds.tail_stats(dv, dseg, nseg, pct)
    assert ds.device_status() == 0
    assert np.array_equal(g.cpu().numpy(), o) and np.array_equal(gc.cpu().numpy(), oc), (seed, n, nseg, mode, pct)
    if nseg * len(pct) <= 128 and nseg <= 128:
        out = torch.full((nseg, len(pct)), -777, dtype=torch.int64, device=DEV)
        cnt = torch.full((nseg,), -777, dtype=torch.int64, device=DEV)
        ds.tail_stats_static(dv, dseg, nseg, out, cnt, pct)
        assert np.array_equal(out.cpu().numpy(), o) and np.array_equal(cnt.cpu().numpy(), oc), (seed, n, nseg, mode, pct, "static")
