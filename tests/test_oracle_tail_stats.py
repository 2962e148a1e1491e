"""Pins for oracle.tail_stats / latencies (reading A13 nearest rank)."""
import numpy as np

import oracle


def test_hand_values():
    out, cnt = oracle.tail_stats([5, 1, 9, 3], [0, 0, 0, 0], 1)
    assert out.tolist() == [[3, 9]] and cnt.tolist() == [4]
    out, _ = oracle.tail_stats([42], [0], 1, pct=(1, 50, 99, 100))
    assert out.tolist() == [[42, 42, 42, 42]]
    out, _ = oracle.tail_stats(np.arange(1, 101)[::-1], np.zeros(100, np.int32), 1)
    assert out.tolist() == [[50, 99]]
    out, _ = oracle.tail_stats(np.arange(1, 201), np.zeros(200, np.int32), 1)
    assert out.tolist() == [[100, 198]]
    out, cnt = oracle.tail_stats([7, 8], [1, -1], 3)
    assert out.tolist() == [[-1, -1], [7, 7], [-1, -1]] and cnt.tolist() == [0, 1, 0]


def test_against_numpy_partition():
    rng = np.random.default_rng(1)
    n, nseg = 200_000, 7
    v = rng.integers(-10**12, 10**12, n)
    v[::5] = rng.integers(0, 50, len(v[::5]))        # many duplicates
    seg = rng.integers(-1, nseg, n).astype(np.int32)
    pct = (1, 50, 95, 99, 100)
    out, cnt = oracle.tail_stats(v, seg, nseg, pct)
    for s in range(nseg):
        x = v[seg == s]
        assert cnt[s] == x.size
        for j, p in enumerate(pct):
            k = max(1, -(-p * x.size // 100)) - 1
            assert out[s, j] == np.partition(x, k)[k]   # independent selection routine


def test_latencies_definition():
    from paper_2606_02982_b200 import workload as wl
    cfg = wl.config0(oracle.characterize)
    st, dn, _ = oracle.simulate(cfg.trace_off, cfg.arrival, cfg.tier, cfg.words, cfg.tokens, cfg.out_len, cfg.server,
                                cfg.instances)
    e2e, qd, seg_t, seg_a = oracle.latencies(cfg.trace_off, cfg.arrival, cfg.tier, cfg.words, cfg.tokens, cfg.out_len,
                                             cfg.instances, cfg.out_off, st, dn, cfg.group)
    a = np.tile(cfg.arrival, 2)
    assert np.array_equal(e2e, dn - a) and np.array_equal(qd, st - a)
    assert np.array_equal(seg_a, np.repeat([0, 1], 200)) and np.array_equal(seg_t, seg_a * 3 + np.tile(cfg.tier, 2))


def test_segment_ids_outside_the_range_are_skipped():
    # SURVEY.md §8(c) C.3 / driftsched.h: seg_id outside [0, n_segments) is skipped, negative or too large alike (by hand)
    vals = np.array([5, 1, 9, 3, 100, 200, 7], np.int64)
    seg = np.array([0, 0, 0, 0, -1, 2, 1], np.int32)          # 200 has id 2 = n_segments: not segment 0 (2 % 2), not counted at all
    out, cnt = oracle.tail_stats(vals, seg, 2, (50, 99))
    assert out.tolist() == [[3, 9], [7, 7]] and cnt.tolist() == [4, 1]
    out, cnt = oracle.tail_stats(vals, np.full(7, 9, np.int32), 2, (50,))
    assert out.tolist() == [[-1], [-1]] and cnt.tolist() == [0, 0]


def test_percentile_0_and_100_are_the_extremes():
    # nearest rank (A13): rank = max(1, ceil(p n / 100)): p = 0 -> the smallest element, p = 100 -> the largest (by hand)
    out, cnt = oracle.tail_stats(np.array([5, 1, 9, 3], np.int64), np.zeros(4, np.int32), 1, (0, 100))
    assert out.tolist() == [[1, 9]] and cnt.tolist() == [4]
