"""Invariants I1-I9 and brute force over orderings for oracle.simulate (SURVEY.md §8(c) 'Pins')."""
import itertools

import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import run_oracle, server, service_time


@pytest.fixture(scope="module")
def small():
    # 6 traces x 400 requests shaped like configs[1], all 5 policies x both estimators
    return wl.config1(oracle.characterize, n_traces=6, n_req=400, seed=5)


@pytest.fixture(scope="module")
def small_out(small):
    c = small
    return oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances)


def _per_inst(c, arr):
    return arr.reshape(c.n_inst, c.n_req)


def test_i1_conservation_and_ordering(small, small_out):
    c = small
    st, dn, _ = small_out
    assert (st >= 0).all() and (dn >= 0).all()          # every request started and finished exactly once
    a = c.arrival.reshape(c.n_traces, c.n_req)[c.instances["trace"]]
    S, D = _per_inst(c, st), _per_inst(c, dn)
    assert (a <= S).all() and (S < D).all()
    # a request holds a slot for exactly O iterations, each >= c_base + c_batch ticks
    O = c.out_len.reshape(c.n_traces, c.n_req)[c.instances["trace"]]
    assert (D - S >= O * (c.server.c_base + c.server.c_batch)).all()


def test_i2_batch_limit(small, small_out):
    c = small
    st, dn, _ = small_out
    S, D = _per_inst(c, st), _per_inst(c, dn)
    for i in range(c.n_inst):
        ev = np.concatenate([np.stack([S[i], np.ones_like(S[i])], 1), np.stack([D[i], -np.ones_like(D[i])], 1)])
        ev = ev[np.lexsort((ev[:, 1], ev[:, 0]))]        # completions (-1) before starts (+1) at the same tick
        assert np.cumsum(ev[:, 1]).max() <= c.server.max_batch


def test_i3_i4_fifo_and_within_tier_order(small, small_out):
    c = small
    st, _, _ = small_out
    S = _per_inst(c, st)
    tier = c.tier.reshape(c.n_traces, c.n_req)
    for i, ins in enumerate(c.instances):
        if ins["policy"] == wl.FIFO:
            assert (np.diff(S[i]) >= 0).all()            # I3 ("strictly in arrival order")
        if ins["policy"] != wl.SJF:
            for t in range(3):                           # I4 (PAPER.md:228-230 FIFO inside each tier)
                assert (np.diff(S[i][tier[ins["trace"]] == t]) >= 0).all()


def test_priority_tier_ordering_qualitative():
    # PAPER.md Table VIII (507-525): under Priority queue wait Premium << Standard << Batch; FIFO about equal;
    # Weighted in between. Needs real contention: overloaded server (rho 1.3), queue delay.
    sv = wl.Server(max_batch=32, kv_budget=16384)
    c = wl._trace_workload("x", 5, 6, 400, sv, [(p, wl.EXACT, 0.0) for p in wl.ALL_POLICIES], oracle.characterize, rho=1.3)
    st, dn, _ = oracle.simulate(c.trace_off, c.arrival, c.tier, c.words, c.tokens, c.out_len, c.server, c.instances)
    a = c.arrival.reshape(c.n_traces, c.n_req)[c.instances["trace"]]
    qd = _per_inst(c, st) - a
    tier = c.tier.reshape(c.n_traces, c.n_req)[c.instances["trace"]]
    means = {pol: [qd[c.instances["policy"] == pol][tier[c.instances["policy"] == pol] == t].mean() for t in range(3)]
             for pol in range(5)}
    p = means[wl.PRIORITY]
    assert p[0] * 3 < p[1] and p[1] * 3 < p[2]
    f = means[wl.FIFO]
    assert max(f) / min(f) < 1.15
    w = means[wl.WEIGHTED]
    assert p[0] < w[0] < f[0] and f[2] < w[2] < p[2]
    # SJF lowers the aggregate queue wait when the key is informative
    assert qd[c.instances["policy"] == wl.SJF].mean() < qd[c.instances["policy"] == wl.FIFO].mean()


def test_i6_makespan_policy_independent_single_server():
    rng = np.random.default_rng(2)
    n = 40
    req = np.stack([np.sort(rng.integers(0, 300_000, n)), rng.integers(0, 3, n), rng.integers(1, 50, n),
                    rng.integers(1, 200, n), rng.integers(1, 40, n)], 1)
    sv = server()
    ends, busy = set(), []
    for pol in range(5):
        for est in (wl.SPLIT, wl.EXACT):
            st, dn, _ = run_oracle(req, sv, pol, est, 0.1)
            ends.add(int(dn.max()))
            assert np.array_equal(dn - st, [service_time(int(p), int(o), sv) for p, o in req[:, 3:5]])
            busy.append(sorted((dn - st).tolist()))
    assert len(ends) == 1 and all(b == busy[0] for b in busy)


def test_i8_tier_relabelling():
    rng = np.random.default_rng(4)
    n = 60
    req = np.stack([np.sort(rng.integers(0, 100_000, n)), rng.integers(0, 3, n), rng.integers(1, 50, n),
                    rng.integers(1, 200, n), rng.integers(1, 40, n)], 1)
    req2 = req.copy()
    req2[:, 1] = (req[:, 1] + 1) % 3
    sv = server(max_batch=4, kv_budget=600)
    for pol, est in ((wl.FIFO, wl.EXACT), (wl.SJF, wl.EXACT), (wl.FIFO, wl.SPLIT)):
        a, b = run_oracle(req, sv, pol, est, 0.0), run_oracle(req2, sv, pol, est, 0.0)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_i9_degenerate_equivalences():
    rng = np.random.default_rng(6)
    n = 80
    req = np.stack([np.sort(rng.integers(0, 200_000, n)), rng.integers(0, 3, n), rng.integers(1, 50, n),
                    rng.integers(1, 200, n), rng.integers(1, 40, n)], 1)
    sv = server(max_batch=3, aging_step=10**15)
    a, p = run_oracle(req, sv, wl.AGING), run_oracle(req, sv, wl.PRIORITY)
    assert np.array_equal(a[0], p[0]) and np.array_equal(a[1], p[1])     # huge aging step == PRIORITY
    one = req.copy()
    one[:, 1] = 1
    f = run_oracle(one, sv, wl.FIFO)
    for pol in (wl.WEIGHTED, wl.PRIORITY, wl.AGING):
        x = run_oracle(one, sv, pol)
        assert np.array_equal(x[0], f[0]) and np.array_equal(x[1], f[1])  # single-tier trace == FIFO


def test_kv_budget_never_binds_equals_unlimited_and_tiny_budget_serialises():
    rng = np.random.default_rng(8)
    n = 50
    req = np.stack([np.sort(rng.integers(0, 50_000, n)), rng.integers(0, 3, n), rng.integers(1, 50, n),
                    rng.integers(1, 200, n), rng.integers(1, 40, n)], 1)
    big, unl, tiny = server(max_batch=8, kv_budget=10**12), server(max_batch=8, kv_budget=0), server(max_batch=8, kv_budget=1)
    for pol in range(5):
        a, b = run_oracle(req, big, pol), run_oracle(req, unl, pol)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
        st, dn, _ = run_oracle(req, tiny, pol)      # est>=1 never fits next to a running request: one at a time
        order = np.argsort(st, kind="stable")
        assert (st[order][1:] >= dn[order][:-1]).all()


def _policy_order_direct(req, pol, sv, now):
    idx = list(range(len(req)))
    if pol == wl.FIFO:
        return idx
    if pol == wl.PRIORITY:
        return sorted(idx, key=lambda r: (req[r][1], r))
    if pol == wl.SJF:
        return sorted(idx, key=lambda r: (req[r][3], r))
    raise AssertionError


@pytest.mark.parametrize("n", [2, 3, 4, 5, 6])
def test_brute_force_orderings(n):
    # all n requests queued behind a running head request; max_batch=1 (SURVEY.md 'Brute force (<=6 queued)')
    rng = np.random.default_rng(100 + n)
    sv = server(aging_step=10**12)
    for trial in range(6):
        q = np.stack([np.zeros(n, np.int64), rng.integers(0, 3, n), rng.integers(1, 9, n), rng.integers(1, 30, n),
                      np.full(n, 3)], 1)
        for pol in (wl.FIFO, wl.PRIORITY, wl.SJF):
            st, dn, _ = run_oracle(q, sv, pol, wl.EXACT)
            # request 0 is admitted first at tick 0 whatever the policy says about the others? No: all arrive at
            # tick 0, so the policy orders all n.
            assert np.argsort(st, kind="stable").tolist() == _policy_order_direct(q.tolist(), pol, sv, 0)
        # WEIGHTED: direct simulation of the slot pattern PPPPSSB
        st, _, _ = run_oracle(q, sv, wl.WEIGHTED, wl.EXACT)
        pattern, cur, left, order = [0, 0, 0, 0, 1, 1, 2], 0, list(range(n)), []
        while left:
            for s in range(7):
                pos = (cur + s) % 7
                cand = [r for r in left if q[r][1] == pattern[pos]]
                if cand:
                    order.append(cand[0]); left.remove(cand[0]); cur = (pos + 1) % 7
                    break
        assert np.argsort(st, kind="stable").tolist() == order
        # SJF + EXACT with equal O minimises sum(done) over all n! orders (closed form (i))
        st, dn, _ = run_oracle(q, sv, wl.SJF, wl.EXACT)
        S = [service_time(int(p), 3, sv) for p in q[:, 3]]
        best = min(sum(itertools.accumulate(S[i] for i in perm)) for perm in itertools.permutations(range(n)))
        assert int(dn.sum()) == best


def test_aging_brute_force_against_direct_key():
    # queued requests with different waits: AGING order = repeated argmin of (max(0,tier-floor(wait/step)), seq)
    rng = np.random.default_rng(77)
    sv = server(aging_step=3000)
    for trial in range(20):
        n = 6
        head = [[0, 0, 1, int(rng.integers(500, 3000)), 1]]
        arr = np.sort(rng.integers(1, 9000, n))
        q = [[int(arr[i]), int(rng.integers(0, 3)), 1, int(rng.integers(1, 400)), 1] for i in range(n)]
        req = head + q
        st, dn, _ = run_oracle(req, sv, wl.AGING)
        now, left, order = service_time(head[0][3], 1, sv), list(range(1, n + 1)), []
        while left:
            avail = [r for r in left if req[r][0] <= now]
            if not avail:
                now = min(req[r][0] for r in left)
                continue
            r = min(avail, key=lambda r: (max(0, req[r][1] - (now - req[r][0]) // 3000), r))
            order.append(r); left.remove(r)
            assert st[r] == now
            now += service_time(req[r][3], 1, sv)
        assert len(order) == n


def check_kv_admission_from_outputs(arrival, P, O, start, done, max_batch, kv_budget, step):
    """I2 + A8 verified from the outputs alone (FIFO, EXACT estimator, iteration cost == `step` ticks whatever the batch):
    with a constant iteration cost a running request has decoded g = (t - start)/step tokens at boundary t, so the context
    held, kv_used(t) = sum over running r of P[r] + g[r], is reconstructed without the simulator. Every admission and every
    boundary at which the FIFO head stayed queued although a slot was free must agree with SURVEY.md §8(c) C.2 step 4:
    admit iff server empty or kv_used + est <= kv_budget (est = P); a deferred head blocks everything behind it."""
    n = len(P)
    assert (done - start == O * step).all()                       # exactly O iterations in the batch
    assert (np.diff(start) >= 0).all()                            # FIFO admits in index order
    def running_before(c, t):                                     # requests holding a slot at boundary t when c is considered:
        r = np.arange(c)                                          # FIFO: only lower indices can have been admitted before c
        return r[(start[:c] <= t) & (done[:c] > t)]               # done == t retired in step 2, before step 4
    def kv_used(rs, t):
        assert ((t - start[rs]) % step == 0).all()                # boundaries of a busy period lie on its grid
        return int((P[rs] + (t - start[rs]) // step).sum())
    n_deferred = n_over = 0
    for c in range(n):
        t = int(start[c])
        rs = running_before(c, t)
        assert len(rs) < max_batch                                # I2: |R| <= max_batch
        if len(rs) > 0:
            assert kv_used(rs, t) + P[c] <= kv_budget, (c, t)     # admitted into a busy server => it fitted
        elif P[c] > kv_budget:
            n_over += 1                                           # progress guarantee: admitted although est > budget
        # boundaries at which c was already the queue head (c-1 admitted) and had arrived, but was not admitted
        t_head = max(int(arrival[c]), int(start[c - 1]) if c else 0)
        if t_head < t:
            busy = running_before(c, t - 1)                       # the busy period c waits in
            assert len(busy) > 0                                  # I5: an idle server never leaves a queued request waiting
            g0 = int(start[busy].max())                           # a grid point of that busy period
            k0 = -(-(t_head - g0) // step)                        # first boundary at or after t_head
            for tb in range(g0 + k0 * step, t, step):
                rb = running_before(c, tb)
                assert len(rb) > 0
                if len(rb) < max_batch:                           # a slot was free: only the KV budget can have deferred c
                    assert kv_used(rb, tb) + P[c] > kv_budget, (c, tb)
                    n_deferred += 1
    return n_deferred, n_over


def test_i2_kv_accounting_and_a8_reconstructed_from_outputs():
    # direct check of I2 (kv_used = sum(P+g)) and of the three parts of A8 (check on the estimate, head-of-line blocking,
    # unconditional admission into an empty server), independent of the oracle's own bookkeeping
    rng = np.random.default_rng(11)
    n, step = 3000, 1000
    P = rng.integers(1, 60, n).astype(np.int64)
    P[rng.integers(0, n, 40)] = rng.integers(130, 200, 40)        # some estimates alone exceed the budget
    O = rng.integers(1, 30, n).astype(np.int64)
    arr = np.cumsum(rng.integers(0, 2 * 1900, n)).astype(np.int64)     # utilisation high enough for regular deferrals
    req = np.stack([arr, rng.integers(0, 3, n), P, P, O], 1)
    sv = server(max_batch=6, kv_budget=120, c_base=step, c_batch=0, c_ctx=0, c_prefill=0)
    st, dn, _ = run_oracle(req, sv, wl.FIFO, wl.EXACT)
    n_deferred, n_over = check_kv_admission_from_outputs(arr, P, O, st, dn, 6, 120, step)
    assert n_deferred > 200 and n_over > 10                       # the case does exercise deferral and the progress rule
