"""-m gpu: policy DS_AGING_UNCLAMPED (A15) through the C ABI vs the oracle, bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2606_02982_b200 import workload as wl
from test_gpu_simulate import G, _assert_same, _oracle   # noqa: F401  (fixture + helpers)

POLS = (wl.AGING_UNCLAMPED, wl.AGING)


def test_hand_trace_where_the_clamp_decides(G):
    # same worked example as tests/test_oracle_aging_unclamped.py: expected values are the hand-computed ones
    req = [[0, 0, 1, 1, 25], [10, 2, 1, 1, 1], [20, 1, 1, 1, 1]]
    sv = wl.Server(max_batch=1, kv_budget=0, c_base=10, c_batch=0, c_ctx=0, c_prefill=0, aging_step=100)
    c = G.tiny_workload(wl, req, sv, [(wl.AGING, wl.EXACT, 0.0), (wl.AGING_UNCLAMPED, wl.EXACT, 0.0)])
    st, dn, _ = G.gpu_simulate(c)
    assert st.tolist() == [0, 250, 260, 0, 260, 250] and dn.tolist() == [250, 260, 270, 250, 270, 260]


@pytest.mark.parametrize("max_batch,kv", [(1, 0), (3, 700), (8, 0), (32, 16384), (32, 3000), (128, 65536), (256, 131072)])
@pytest.mark.parametrize("step", [1, 900, 40_000])
def test_sweep(G, max_batch, kv, step):
    # step 1: every waited tick is a level (scores far below zero); 900: dozens of levels; 40 000: a few
    sv = wl.Server(max_batch=max_batch, kv_budget=kv, aging_step=step)
    combos = [(p, e, a) for p in POLS for e, a in ((wl.SPLIT, 0.1), (wl.EXACT, 0.1), (wl.SPLIT, 0.0))]
    differs = False
    for rho in (0.85, 1.4):
        c = wl._trace_workload("t", 91 + max_batch, 3, 600, sv, combos, oracle.characterize, rho=rho)
        g, o = G.gpu_simulate(c), _oracle(c)
        _assert_same(g, o, c)
        un = c.instances["policy"] == wl.AGING_UNCLAMPED
        s = g[0].reshape(len(c.instances), -1)
        differs |= not np.array_equal(s[un], s[~un])
    if step == 900 and max_batch <= 8:
        assert differs                      # the variant really schedules differently from AGING on these inputs


def test_overload_pareto_and_ties(G):
    sv = wl.Server(max_batch=16, kv_budget=6000, aging_step=25_000)
    c = wl._trace_workload("t", 35, 2, 3000, sv, [(p, wl.SPLIT, a) for p in POLS for a in (0.05, 0.5)], None, rho=1.6,
                           out_dist=1, materialise=False)
    _assert_same(G.gpu_simulate(c), _oracle(c), c)
    # equal arrival ticks, zero-length prompts, O=1
    rng = np.random.default_rng(6)
    n = 500
    req = np.stack([np.sort(rng.integers(0, 40, n)) * 50_000, rng.integers(0, 3, n), rng.integers(0, 3, n),
                    rng.integers(0, 4, n), rng.integers(1, 4, n)], 1)
    for mb, kv in ((1, 0), (4, 6), (32, 0)):
        sv = wl.Server(max_batch=mb, kv_budget=kv, aging_step=7000)
        c = G.tiny_workload(wl, req, sv, [(wl.AGING_UNCLAMPED, e, 0.3) for e in (wl.SPLIT, wl.EXACT)])
        _assert_same(G.gpu_simulate(c), _oracle(c), c)


def test_64bit_path_and_huge_step(G):
    sv = wl.Server(max_batch=6, kv_budget=9000, aging_step=3_000_000_000, c_base=2_000_000_000, c_batch=150_000_000,
                   c_ctx=1_000_003, c_prefill=5_000_000)
    c = wl._trace_workload("t", 78, 2, 400, sv, [(wl.AGING_UNCLAMPED, e, 0.2) for e in (wl.SPLIT, wl.EXACT)],
                           oracle.characterize, mean_ticks=3.0e10)
    c.out_len[5] = 70_000
    _assert_same(G.gpu_simulate(c), _oracle(c), c)
    # a step no wait reaches: identical to PRIORITY (property at any size)
    sv = wl.Server(max_batch=32, kv_budget=16384, aging_step=1 << 60)
    c = wl._trace_workload("t", 79, 4, 2000, sv, [(wl.AGING_UNCLAMPED, wl.SPLIT, 0.1), (wl.PRIORITY, wl.SPLIT, 0.1)],
                           oracle.characterize, rho=0.95)
    st, dn, ema = G.gpu_simulate(c)
    un = c.instances["policy"] == wl.AGING_UNCLAMPED
    for a in (st.reshape(len(un), -1), dn.reshape(len(un), -1), ema.view(np.uint64)):
        assert np.array_equal(a[un], a[~un])


def test_budget_estimator_and_closed_loop(G):
    # the same policy body inside ds_simulate_budget / ds_simulate_closed (Eq. 1-2 in full, 50 clients, batch wait)
    import torch
    import paper_2606_02982_b200 as ds
    sv = wl.Server(max_batch=32, kv_budget=16384, aging_step=20_000, weight=(5, 3, 2))
    bp = wl.Budget()
    c = wl._trace_workload("t", 80, 3, 1500, sv, [(wl.AGING_UNCLAMPED, wl.BUDGET_SPLIT, 0.1), (wl.AGING_UNCLAMPED, wl.BUDGET_EXACT, 0.0)],
                           oracle.characterize, rho=1.0)
    cat, out_len = wl.assign_categories(80, c.out_len)
    arrival = np.zeros_like(c.arrival)               # closed loop: the 50 clients start together; later entries are ignored
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, out_len)
    d = G.upload(c)
    d["out_len"] = torch.from_numpy(out_len).to(G.DEV)
    dcat = torch.from_numpy(cat).to(G.DEV)
    targs = tuple(d[k] for k in ("trace_off", "arrival", "tier", "words", "tokens", "out_len"))
    n_total = int(c.out_off[-1])
    for n_clients, wait in ((0, 0), (50, 0), (50, 10_000)):
        if n_clients:
            tr = (c.trace_off, arrival, c.tier, c.words, c.tokens, out_len)
            d["arrival"] = torch.from_numpy(arrival).to(G.DEV)
            targs = tuple(d[k] for k in ("trace_off", "arrival", "tier", "words", "tokens", "out_len"))
        o = oracle.simulate_budget(*tr, cat, bp, c.server, c.instances, n_clients=n_clients, batch_wait=wait)
        arr_out = torch.zeros(n_total, dtype=torch.int64, device=G.DEV) if n_clients else None
        r = ds.api.simulate_budget(*targs, dcat, bp, c.server, d["inst"], d["out_off"], n_total, n_clients=n_clients,
                                   arrival_out=arr_out, batch_wait=wait)
        assert ds.device_status() == 0
        assert np.array_equal(r[0].cpu().numpy(), o[0]) and np.array_equal(r[1].cpu().numpy(), o[1])
        assert np.array_equal(r[2].cpu().numpy().view(np.uint64), o[2].view(np.uint64))
        if n_clients:
            assert np.array_equal(r[3].cpu().numpy(), o[-1])
