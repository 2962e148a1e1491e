"""Pins for the oracle's AGING_UNCLAMPED policy (reading A15).

PAPER.md:242: "Waiting time progressively reduces the effective scheduling score, allowing long-waiting requests to
eventually execute even under continuous high-priority traffic." AGING (A10) clamps the score at Premium's level 0;
the variant does not: key = (tier - floor(waited/aging_step), seq).
"""
import numpy as np
import pytest

from paper_2606_02982_b200 import workload as wl
from _simutil import run_oracle, server, service_time


def test_hand_trace_where_the_clamp_decides():
    # Worked by hand. Server: batch 1, c_base 10, everything else 0 => a request of O tokens holds the server 10*O ticks.
    # r0 Premium arrives 0, O=25 -> runs [0, 250). r1 Batch arrives 10, r2 Standard arrives 20, aging_step 100.
    # At tick 250: waited(r1) = 240 -> 2 levels, waited(r2) = 230 -> 2 levels.
    #   AGING:           score(r1) = max(0, 2-2) = 0, score(r2) = max(0, 1-2) = 0 -> tie -> lower seq r1 first.
    #   AGING_UNCLAMPED: score(r1) = 0,               score(r2) = -1            -> r2 first.
    # r1, r2 have O=1 (10 ticks each).
    req = [[0, 0, 1, 1, 25], [10, 2, 1, 1, 1], [20, 1, 1, 1, 1]]
    sv = server(c_base=10, c_batch=0, c_ctx=0, c_prefill=0, aging_step=100)
    st, dn, _ = run_oracle(req, sv, wl.AGING)
    assert st.tolist() == [0, 250, 260] and dn.tolist() == [250, 260, 270]
    st, dn, _ = run_oracle(req, sv, wl.AGING_UNCLAMPED)
    assert st.tolist() == [0, 260, 250] and dn.tolist() == [250, 270, 260]


def test_hand_trace_aged_batch_overtakes_fresh_premium():
    # the promotion itself (common to both variants): r1 Batch has waited 3 levels when r0 completes, r2 Premium 0 levels
    # server as above; r0 runs [0, 400); r1 Batch arrives 50 (waited 350 -> 3 levels -> score -1 / clamped 0),
    # r2 Premium arrives 390 (score 0). Unclamped: r1 (-1) first. Clamped: tie at 0 -> r1 (lower seq) first as well.
    req = [[0, 0, 1, 1, 40], [50, 2, 1, 1, 1], [390, 0, 1, 1, 1]]
    sv = server(c_base=10, c_batch=0, c_ctx=0, c_prefill=0, aging_step=100)
    for pol in (wl.AGING, wl.AGING_UNCLAMPED):
        st, _, _ = run_oracle(req, sv, pol)
        assert st.tolist() == [0, 400, 410]
    # with only 1 level waited (aging_step 300) the fresh Premium request wins under both
    sv = server(c_base=10, c_batch=0, c_ctx=0, c_prefill=0, aging_step=300)
    for pol in (wl.AGING, wl.AGING_UNCLAMPED):
        st, _, _ = run_oracle(req, sv, pol)
        assert st.tolist() == [0, 410, 400]


def test_brute_force_against_direct_key():
    # batch 1: the admission order is the repeated argmin of (tier - floor(waited/step), seq) over the arrived requests,
    # restated here with Python integers; also counts how often the clamp would have decided differently
    rng = np.random.default_rng(78)
    sv = server(aging_step=1500)
    differs = 0
    for trial in range(30):
        n = 6
        head = [[0, 0, 1, int(rng.integers(500, 3000)), 1]]
        arr = np.sort(rng.integers(1, 9000, n))
        q = [[int(arr[i]), int(rng.integers(0, 3)), 1, int(rng.integers(1, 400)), 1] for i in range(n)]
        req = head + q
        st, dn, _ = run_oracle(req, sv, wl.AGING_UNCLAMPED)
        st_c, _, _ = run_oracle(req, sv, wl.AGING)
        differs += int(not np.array_equal(st, st_c))
        now, left = service_time(head[0][3], 1, sv), list(range(1, n + 1))
        while left:
            avail = [r for r in left if req[r][0] <= now]
            if not avail:
                now = min(req[r][0] for r in left)
                continue
            r = min(avail, key=lambda r: (req[r][1] - (now - req[r][0]) // 1500, r))
            left.remove(r)
            assert st[r] == now
            now += service_time(req[r][3], 1, sv)
    assert differs >= 3          # the variant is not a relabelling of AGING on these inputs


def test_reductions():
    rng = np.random.default_rng(16)
    n = 120
    req = np.stack([np.sort(rng.integers(0, 300_000, n)), rng.integers(0, 3, n), rng.integers(1, 50, n),
                    rng.integers(1, 200, n), rng.integers(1, 40, n)], 1)
    # (i) a step no wait can reach: no promotion at all == PRIORITY
    sv = server(max_batch=3, aging_step=10**15)
    a, p = run_oracle(req, sv, wl.AGING_UNCLAMPED), run_oracle(req, sv, wl.PRIORITY)
    assert np.array_equal(a[0], p[0]) and np.array_equal(a[1], p[1])
    # (ii) a single tier: score is monotone in the wait, the oldest request always wins == FIFO
    one = req.copy()
    one[:, 1] = 2
    for step in (1, 777, 50_000):
        sv = server(max_batch=3, aging_step=step)
        a, f = run_oracle(one, sv, wl.AGING_UNCLAMPED), run_oracle(one, sv, wl.FIFO)
        assert np.array_equal(a[0], f[0]) and np.array_equal(a[1], f[1])
    # (iii) while no request has waited more than one level past its tier, the clamp never acts: identical to AGING.
    # Light load (arrivals 20x the mean service apart) and a step far above any wait that occurs.
    light = req.copy()
    light[:, 0] = np.arange(n) * 400_000
    sv = server(max_batch=3, aging_step=10_000_000)
    a, c = run_oracle(light, sv, wl.AGING_UNCLAMPED), run_oracle(light, sv, wl.AGING)
    assert np.array_equal(a[0], c[0]) and np.array_equal(a[1], c[1])


@pytest.mark.parametrize("max_batch,kv", [(1, 0), (4, 0), (4, 900)])
def test_conservation_and_head_of_tier_order(max_batch, kv):
    rng = np.random.default_rng(33)
    n = 300
    req = np.stack([np.sort(rng.integers(0, 400_000, n)), rng.integers(0, 3, n), rng.integers(1, 50, n),
                    rng.integers(1, 200, n), rng.integers(1, 40, n)], 1)
    sv = server(max_batch=max_batch, kv_budget=kv, aging_step=20_000)
    st, dn, _ = run_oracle(req, sv, wl.AGING_UNCLAMPED)
    assert (st >= req[:, 0]).all() and (dn > st).all()          # every request served once, after it arrived
    for t in range(3):                                           # inside a tier the score is monotone in the wait: FIFO
        s = st[req[:, 1] == t]
        assert (np.diff(s) >= 0).all()
