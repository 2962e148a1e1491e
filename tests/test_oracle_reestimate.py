"""Pins for the online re-estimation mode of oracle.simulate ("adaptive queue
reordering, online workload reclassification"; reading A16 in DESIGN.md §4): queued requests are re-estimated with the factors
current at every scheduling decision instead of keeping the estimate frozen at arrival (A5). What fixes the expected values:
  * two hand-worked traces (DESIGN.md §4.4 H11, H12): a refreshed estimate flips the SJF order; a refreshed estimate lets a
    KV-deferred head in (each next to the frozen run of the same trace);
  * reductions: alpha = 0 or the exact estimator (B == 1.0) => identical to the frozen run, for every policy;
  * policies that never read an estimate (no KV budget, not SJF) produce identical ticks in both modes;
  * the paper's motivation: during a token drift dispatch-time estimates are closer to the truth than arrival-time ones.
"""
import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import run_oracle, server


def test_h11_refreshed_estimate_flips_the_sjf_order():
    # r0 = (0, Std, W 4, P 2, O 1) completes at 2162 with m = 0.5, alpha = 0.5 -> B[Std] = 0.75.
    # r1 = (100, Std, W 8): frozen est 8, refreshed ceil(0.75*8) = 6.  r2 = (200, Prem, W 7): est 7 either way.
    req = [[0, 1, 4, 2, 1], [100, 1, 8, 3, 1], [200, 0, 7, 5, 1]]
    st, dn, ema, est = run_oracle(req, server(), wl.SJF, wl.SPLIT, 0.5, want_est=True)
    assert st.tolist() == [0, 4342, 2162] and dn.tolist() == [2162, 6510, 4342] and est.tolist() == [4, 8, 7]
    st, dn, ema, est = run_oracle(req, server(reestimate=1), wl.SJF, wl.SPLIT, 0.5, want_est=True)
    assert st.tolist() == [0, 2162, 4330] and dn.tolist() == [2162, 4330, 6510] and est.tolist() == [4, 6, 7]
    assert ema[0, 1] == 0.5 * 0.75 + 0.5 * (3 / 8)            # r1 completed second-to-last in tier Std


def test_h12_refreshed_estimate_passes_the_kv_check():
    # FIFO, max_batch 2, KV 20. r0 = (0, Std, W 4, P 2, O 1), r1 = (0, Std, W 12, P 9, O 3), r2 = (10, Std, W 11, P 5, O 1).
    # At 2366 r0 retires (kv 10, B[Std] 0.75): frozen est(r2) = 11 -> 21 > 20 deferred until r1 is done;
    # refreshed est(r2) = ceil(0.75*11) = 9 -> 19 <= 20 admitted at once.
    req = [[0, 1, 4, 2, 1], [0, 1, 12, 9, 3], [10, 1, 11, 5, 1]]
    sv = dict(max_batch=2, kv_budget=20)
    st, dn, ema, est = run_oracle(req, server(**sv), wl.FIFO, wl.SPLIT, 0.5, want_est=True)
    assert st.tolist() == [0, 0, 6687] and dn.tolist() == [2366, 6687, 8867] and est.tolist() == [4, 12, 11]
    st, dn, ema, est = run_oracle(req, server(reestimate=1, **sv), wl.FIFO, wl.SPLIT, 0.5, want_est=True)
    assert st.tolist() == [0, 0, 2366] and dn.tolist() == [2366, 6867, 4706] and est.tolist() == [4, 12, 9]


def _cfg(seed=11, n_req=500, kv=3000, rho=1.1, combos=None):
    sv = wl.Server(max_batch=8, kv_budget=kv, aging_step=30_000)
    combos = combos or [(p, e, a) for p in wl.ALL_POLICIES + [wl.AGING_UNCLAMPED] for e, a in ((wl.SPLIT, 0.0), (wl.EXACT, 0.3), (wl.SPLIT, 0.3))]
    return wl._trace_workload("t", seed, 2, n_req, sv, combos, oracle.characterize, rho=rho)


def _run(c, reest):
    c.server.reestimate = reest
    out = oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances, want_est=True)
    c.server.reestimate = 0
    return out


def test_reductions_to_the_frozen_run():
    c = _cfg()
    a, b = _run(c, 0), _run(c, 1)
    per = lambda x: x.reshape(c.n_inst, c.n_req)
    same = (per(a[0]) == per(b[0])).all(axis=1) & (per(a[1]) == per(b[1])).all(axis=1) & (per(a[3]) == per(b[3])).all(axis=1)
    fixed = (c.instances["ema_alpha"] == 0.0) | (c.instances["estimator"] == wl.EXACT)     # B == 1.0 throughout
    assert same[fixed].all()
    assert not same[~fixed].all()                              # and the mode does change something when the factors move
    assert np.array_equal(a[2][fixed].view(np.uint64), b[2][fixed].view(np.uint64))


def test_policies_that_read_no_estimate_are_unchanged():
    c = _cfg(kv=0, combos=[(p, wl.SPLIT, 0.3) for p in (wl.FIFO, wl.PRIORITY, wl.WEIGHTED, wl.AGING, wl.AGING_UNCLAMPED)])
    a, b = _run(c, 0), _run(c, 1)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2].view(np.uint64), b[2].view(np.uint64))
    assert (a[3] != b[3]).any()                                # est_out is the dispatch-time estimate in mode 1


def test_dispatch_time_estimates_track_a_drift_better():
    # configs[4] shape: tokens/word jumps 1.40 -> 2.14 mid-trace; a request that waits through the jump is re-estimated with
    # the newer factor, so the mean absolute error of est vs the true tokens is lower than with arrival-time estimates
    c = wl.config4(oracle.characterize, n_traces=2, n_req=3000, materialise=True, traj_every=0)
    c.server.max_batch, c.server.kv_budget = 16, 6000
    sel = (c.instances["policy"] == wl.FIFO) & (c.instances["estimator"] == wl.SPLIT)
    c.instances = c.instances[sel]
    a, b = _run(c, 0), _run(c, 1)
    P = c.tokens.reshape(c.n_traces, c.n_req)[c.instances["trace"]].reshape(-1)
    mae0, mae1 = np.abs(a[3] - P).mean(), np.abs(b[3] - P).mean()
    assert mae1 < mae0


def test_contract():
    with pytest.raises(ValueError):
        run_oracle([[0, 0, 1, 1, 1]], server(reestimate=2), wl.FIFO)


def test_not_defined_for_the_budget_estimators():
    # A16 is a reading for the reduced estimator; with the full Eq. 1-2 estimator the oracle refuses (as the library does: DS_EINVAL)
    req = np.asarray([[0, 1, 4, 2, 1]], np.int64)
    inst = np.zeros(1, wl.INSTANCE_DTYPE); inst[0] = (0, wl.FIFO, wl.BUDGET_SPLIT, 0, 0.1)
    tr = ([0, 1], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4])
    with pytest.raises(ValueError):
        oracle.simulate_budget(*tr, np.zeros(1, np.uint8), wl.Budget(), server(reestimate=1), inst)
