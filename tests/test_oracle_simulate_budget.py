"""Pins for oracle.simulate_budget: the paper's full estimator (Eq. 1-2, Alg. 1) with per-category feedback
(Eq. 5-6 as printed). SURVEY.md §8(f) NEXT-2; readings B1-B4 in DESIGN.md §4.

What fixes the expected values, independently of the oracle:
  * hand-worked KV trace (below): with T_budget = T_input + T_estimated_output the second request is deferred three times,
    while the reduced estimator (est = tokens) admits it at tick 0 - ticks worked by hand from the cost formula;
  * with alpha = 0 and power-of-two constants every factor product is exact, so est is an integer formula;
  * SJF order at max_batch = 1 with everything queued at tick 0 = a stable sort by that integer budget;
  * EMA closed form B_k = m + (1-m)(1-alpha)^k per category when every request of a category has the same output length,
    and untouched categories stay exactly 1.0;
  * stationary outputs: the factor's time average -> E[out_len | category] / T_base (the paper's Fig. 5 plateau, ~0.8);
  * T_base = 0 reduces the budget estimator to the reduced EXACT estimator: identical ticks, factors exactly 1.0.
"""
import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import server, service_time


def _run(req, cat, bp, sv, combos, want_traj=False):
    req = np.asarray(req, np.int64).reshape(-1, 5)
    inst = np.zeros(len(combos), wl.INSTANCE_DTYPE)
    for i, (p, e, a) in enumerate(combos):
        inst[i] = (0, p, e, 0, a)
    n = len(req)
    out_off = np.arange(len(combos) + 1, dtype=np.int64) * n
    tr = ([0, n], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4])
    return oracle.simulate_budget(*tr, cat, bp, sv, inst, out_off=out_off, want_est=True, want_traj=want_traj)


def test_hand_trace_kv_deferral_uses_the_output_term():
    # r0 = (arrival 0, Std, W., P 10, O 3) category 0, T_base 8 -> budget 18; r1 = (0, Std, ., P 8, O 1) category 1, T_base 20 -> 28
    req = [[0, 1, 3, 10, 3], [0, 1, 2, 8, 1]]
    bp = wl.Budget(t_base=(8.0, 20.0, 0.0, 0.0))
    # kv 40: 10 + 28 <= 40, both admitted at 0: dt = 2000+300+18+5*18 = 2408 -> r1 done; 2161 -> 4569; 2162 -> 6731 r0 done
    st, dn, ema, est = _run(req, [0, 1], bp, server(max_batch=2, kv_budget=40), [(wl.FIFO, wl.BUDGET_EXACT, 0.0)])
    assert est.tolist() == [18, 28] and st.tolist() == [0, 0] and dn.tolist() == [6731, 2408]
    # kv 37: 10+28, 11+28, 12+28 > 37: deferred at 0, 2210, 4371; r0 done at 6533 (2210 + 2161 + 2162), then r1 alone: 2198
    st, dn, ema, est = _run(req, [0, 1], bp, server(max_batch=2, kv_budget=37), [(wl.FIFO, wl.BUDGET_EXACT, 0.0)])
    assert st.tolist() == [0, 6533] and dn.tolist() == [6533, 8731]
    # the reduced estimator (est = tokens = 8) admits r1 at once under the same budget
    tr = ([0, 2], [0, 0], [1, 1], [3, 2], [10, 8], [3, 1])
    inst = np.zeros(1, wl.INSTANCE_DTYPE); inst[0] = (0, wl.FIFO, wl.EXACT, 0, 0.0)
    st2, dn2, _ = oracle.simulate(*tr, server(max_batch=2, kv_budget=37), inst)
    assert st2.tolist() == [0, 0] and dn2.tolist() == [6731, 2408]


def test_budget_is_an_integer_formula_when_products_are_exact():
    rng = np.random.default_rng(2)
    n = 300
    W = rng.integers(0, 400, n); P = rng.integers(0, 500, n); tier = rng.integers(0, 3, n); cat = rng.integers(0, 4, n)
    req = np.stack([np.cumsum(rng.integers(0, 4000, n)), tier, W, P, rng.integers(1, 9, n)], 1)
    bp = wl.Budget(t_base=(16.0, 64.0, 128.5, 256.0), s_tenant=(1.0, 2.0, 0.5), f_slope=1.0 / 256, f_max=2.0)
    st, dn, ema, est = _run(req, cat, bp, server(max_batch=4), [(wl.SJF, wl.BUDGET_SPLIT, 0.0), (wl.PRIORITY, wl.BUDGET_EXACT, 0.0)])
    tb = np.array(bp.t_base)[cat]; s = np.array(bp.s_tenant)[tier]
    for k, T in enumerate((W, P)):
        F = np.minimum(2.0, 1.0 + T / 256.0)             # exact in binary: T < 2^9, slope 2^-8
        want = T + np.ceil(tb * s * F).astype(np.int64)   # every product exact (<= 12 significant bits each)
        assert np.array_equal(est[k * n:(k + 1) * n], want)
    assert np.all(ema == 1.0)                             # alpha = 0: BIAS OFF


def test_sjf_serves_in_budget_order():
    rng = np.random.default_rng(4)
    n = 6
    for trial in range(30):
        P = rng.integers(1, 60, n); cat = rng.integers(0, 4, n)
        req = np.stack([np.zeros(n, np.int64), rng.integers(0, 3, n), P, P, np.full(n, 2)], 1)
        bp = wl.Budget(t_base=(4.0, 16.0, 32.0, 64.0))
        sv = server()
        st, dn, ema, est = _run(req, cat, bp, sv, [(wl.SJF, wl.BUDGET_EXACT, 0.0)])
        key = P + np.array(bp.t_base, np.int64)[cat]
        assert np.array_equal(est, key)
        order = np.argsort(key, kind="stable")
        t = 0
        for r in order:
            assert st[r] == t
            t += service_time(int(P[r]), 2, sv)
            assert dn[r] == t


def test_ema_closed_form_per_category():
    # category c always decodes O_c tokens -> m_c = O_c / T_base_c is constant -> B_k = m + (1-m)(1-alpha)^k
    n = 240
    rng = np.random.default_rng(6)
    cat = rng.integers(0, 3, n)                            # category 3 never occurs
    O = np.array([30, 100, 7, 1])[cat]
    req = np.stack([np.arange(n) * 100_000, rng.integers(0, 3, n), np.full(n, 5), np.full(n, 6), O], 1)
    bp = wl.Budget(t_base=(40.0, 80.0, 21.0, 50.0))
    alpha = 0.2
    sv = wl.Server(max_batch=1, kv_budget=0, traj_every=1)
    st, dn, ema, traj, est = _run(req, cat, bp, sv, [(wl.FIFO, wl.BUDGET_SPLIT, alpha)], want_traj=True)
    m = np.array([30 / 40, 100 / 80, 7 / 21])
    k = np.array([(cat == c).sum() for c in range(3)])
    want = m + (1 - m) * (1 - alpha) ** k
    assert np.allclose(ema[0, :3], want, rtol=1e-12, atol=0)
    assert ema[0, 3] == 1.0
    # light load: requests complete in index order, so sample j holds the factors after request j
    cnt = np.zeros(4, int)
    for j in range(n):
        cnt[cat[j]] += 1
        w = np.ones(4); w[:3] = m + (1 - m) * (1 - alpha) ** cnt[:3]
        assert np.allclose(traj[j], w, rtol=1e-12, atol=0)
    # the estimate of a request arriving after k completions of its category uses that factor
    c9 = cat[9]; k9 = (cat[:9] == c9).sum()
    assert est[9] == 5 + int(np.ceil(bp.t_base[c9] * (m[c9] + (1 - m[c9]) * (1 - alpha) ** k9)))


def test_factor_settles_at_mean_output_over_baseline():
    c = wl._trace_workload("t", 9, 1, 6000, wl.Server(max_batch=32, kv_budget=0), [(wl.FIFO, wl.BUDGET_SPLIT, 0.1)],
                           oracle.characterize, rho=0.8)
    cat, out_len = wl.assign_categories(9, c.out_len)
    bp = wl.Budget()
    sv = wl.Server(max_batch=32, kv_budget=16384, traj_every=50)
    st, dn, ema, traj = oracle.simulate_budget(c.trace_off, c.arrival, c.tier, c.words, c.tokens, out_len, cat, bp, sv, c.instances,
                                               want_traj=True)
    late = traj[len(traj) // 4:]                           # after the transient
    for k in range(4):
        want = out_len[cat == k].mean() / bp.t_base[k]
        assert abs(late[:, k].mean() - want) < 0.04 * want
        assert 0.70 < late[:, k].mean() < 0.90            # Fig. 5: split()+feedback settles at 0.79-0.84


def test_zero_baseline_reduces_to_the_reduced_estimator():
    sv = wl.Server(max_batch=8, kv_budget=1500, aging_step=30_000)
    combos_b = [(p, wl.BUDGET_EXACT, 0.3) for p in wl.ALL_POLICIES]
    combos_r = [(p, wl.EXACT, 0.3) for p in wl.ALL_POLICIES]
    c = wl._trace_workload("t", 3, 2, 400, sv, combos_r, oracle.characterize, rho=1.1)
    cat, _ = wl.assign_categories(3, c.out_len)
    tr = (c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len)
    st_r, dn_r, _ = oracle.simulate(*tr, sv, c.instances)
    inst_b = c.instances.copy(); inst_b["estimator"] = wl.BUDGET_EXACT
    st_b, dn_b, ema_b = oracle.simulate_budget(*tr, cat, wl.Budget(t_base=(0.0, 0.0, 0.0, 0.0)), sv, inst_b)
    assert np.array_equal(st_r, st_b) and np.array_equal(dn_r, dn_b) and np.all(ema_b == 1.0)


def test_contract_violations():
    req = [[0, 0, 1, 1, 1]]
    with pytest.raises(ValueError):
        _run(req, [4], wl.Budget(), server(), [(wl.FIFO, wl.BUDGET_EXACT, 0.0)])          # category > 3
    with pytest.raises(ValueError):
        _run(req, [0], wl.Budget(), server(), [(wl.FIFO, wl.EXACT, 0.0)])                 # reduced estimator in a budget call
    with pytest.raises(ValueError):
        _run(req, [0], wl.Budget(s_tenant=(1.0, 0.0, 1.0)), server(), [(wl.FIFO, wl.BUDGET_EXACT, 0.0)])
    with pytest.raises(ValueError):
        _run(req, [0], wl.Budget(f_max=0.5), server(), [(wl.FIFO, wl.BUDGET_EXACT, 0.0)])


def test_order_of_the_three_products_of_eq2():
    # Reading B3: T_budget = T_input + ceil(((T_base * B) * S_tenant) * F_input), each product rounded to fp64 in that
    # order. Products of doubles do not associate, so the order is part of the definition. Parameters chosen (by a search over
    # two-digit decimals) so that the prescribed order and the swapped one, ((T_base * B) * F_input) * S_tenant, land on different
    # sides of an integer. Expected values: exact rational arithmetic with a correct rounding to the nearest double after every
    # product (float(Fraction) rounds correctly), i.e. IEEE-754 applied by hand, not this formula in floating point.
    from fractions import Fraction as Fr
    import math

    def rounded_product_chain(*factors):
        x = Fr(factors[0])
        for f in factors[1:]:
            x = Fr(float(x * Fr(f)))
        return x

    for t_base, s_ten, f_in, expect, swapped in ((75.0, 1.1, 1.2, 99, 100), (200.0, 1.25, 1.1, 275, 276), (189.0, 0.8, 1.25, 190, 189)):
        assert math.ceil(rounded_product_chain(t_base, 1.0, s_ten, f_in)) == expect          # the prescribed order, by hand
        assert math.ceil(rounded_product_chain(t_base, 1.0, f_in, s_ten)) == swapped         # the other order differs: the case discriminates
        # F_input = min(f_max, 1 + f_slope * T_input) = f_max exactly once 1 + T_input >= f_max; alpha = 0 keeps B = 1.0
        bp = wl.Budget(t_base=(t_base, 1.0, 1.0, 1.0), s_tenant=(s_ten, 1.0, 1.0), f_slope=1.0, f_max=f_in)
        req = [[0, 0, 7, 9, 1]]                                           # tier 0 (-> s_ten), words 7, tokens 9
        for estimator, t_input in ((wl.BUDGET_SPLIT, 7), (wl.BUDGET_EXACT, 9)):
            out = _run(req, np.zeros(1, np.uint8), bp, server(), [(wl.FIFO, estimator, 0.0)])
            assert out[-1].tolist() == [t_input + expect], (t_base, s_ten, f_in, estimator)


def test_the_factor_of_eq2_is_the_categorys_not_the_tiers():
    # PAPER.md:276 "one factor per workload category" (reading B4). alpha = 0.5, t_base = 100 for every category.
    # r0 (Batch = tier 2, category 0, O 50) completes first: B[category 0] = 0.5 * 1 + 0.5 * (50 / 100) = 0.75, the others stay 1.
    # r1 arrives long after: tier 2, category 0 -> T_budget = 5 + ceil(100 * 0.75) = 80 (with the tier's factor B[2] = 1: 105).
    # r2: tier 0, category 2 -> 5 + ceil(100 * 1.0) = 105 (with the tier's factor B[0] = 0.75: 80).
    bp = wl.Budget(t_base=(100.0, 100.0, 100.0, 100.0), s_tenant=(1.0, 1.0, 1.0), f_slope=0.0, f_max=1.0)
    req = [[0, 2, 5, 5, 50], [50_000_000, 2, 5, 5, 1], [60_000_000, 0, 5, 5, 1]]
    out = _run(req, np.array([0, 0, 2], np.uint8), bp, server(), [(wl.FIFO, wl.BUDGET_SPLIT, 0.5)])
    assert out[-1].tolist() == [105, 80, 105]
