"""Pins for oracle.simulate: hand-worked traces H1-H10, EMA bit pattern H3, closed forms.
H7-H10 (derivations: DESIGN.md §4.4) pin the readings R-ORD (same-tick order), A8 (KV deferral is head-of-line blocking; an
empty server admits unconditionally) and the KV release kv_used -= P+g on retirement."""
import json
import math
import os
import struct

import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl
from _simutil import run_oracle, server, service_time


def _golden(golden_dir):
    return json.load(open(os.path.join(golden_dir, "hand_traces.json")))


def test_hand_traces(golden_dir):
    g = _golden(golden_dir)
    assert len(g["cases"]) == 21
    for c in g["cases"]:
        sv = server(**c["server"])
        if "weight" in c["server"]:
            sv.weight = tuple(c["server"]["weight"])
        st, dn, ema, est = run_oracle(c["req"], sv, c["policy"], c["estimator"], c["alpha"], want_est=True)
        assert st.tolist() == c["start"], c["name"]
        assert dn.tolist() == c["done"], c["name"]
        if "est" in c:
            assert est.tolist() == c["est"], c["name"]
        if "ema" in c:
            assert ema[0].tolist() == c["ema"], c["name"]


def test_h7_factor_after_same_tick_completion():
    # H7 (R-ORD, SURVEY.md:486): r0 completes at 2162 with m = 2/4 and alpha = 0.5 -> B[Std] = 0.5*1 + 0.5*0.5 = 0.75 exactly;
    # r1 (arrival 2161 < 2162) was estimated with the old factor 1.0, r2 (arrival 2162) with 0.75: ceil(0.75*8) = 6, not 8
    req = [[0, 1, 4, 2, 1], [2161, 1, 7, 3, 1], [2162, 1, 8, 5, 1]]
    sv = server(traj_every=1)
    st, dn, ema, traj, est = run_oracle(req, sv, wl.SJF, wl.SPLIT, 0.5, want_traj=True, want_est=True)
    assert traj[0].tolist() == [1.0, 0.75, 1.0]
    assert est.tolist() == [4, 7, 6]
    assert st[2] < st[1]                       # SJF serves r2 (est 6) before r1 (est 7)
    # moving r2 one tick earlier makes it an INGEST-EARLY arrival: old factor, est 8, served after r1
    req[2][0] = 2161
    st, dn, ema, est = run_oracle(req, sv, wl.SJF, wl.SPLIT, 0.5, want_est=True)
    assert est.tolist() == [4, 7, 8] and st[1] < st[2]


def test_h3_ema_bit_pattern(golden_dir):
    g = _golden(golden_dir)
    # the bit pattern is fixed by IEEE-754 arithmetic, independent of the oracle:
    m = 4.0 / 3.0
    b = (1.0 - 0.1) * 1.0 + 0.1 * m
    assert hex(struct.unpack("<Q", struct.pack("<d", b))[0]).upper() == g["H3_ema"]["B_std_bits"].upper()
    # one Standard request completes -> B[Std] is exactly that, others untouched
    st, dn, ema = run_oracle([[0, 1, 3, 4, 2]], server(), wl.SJF, wl.SPLIT, 0.1)
    bits = struct.unpack("<Q", struct.pack("<d", ema[0, 1]))[0]
    assert bits == int(g["H3_ema"]["B_std_bits"], 16)
    assert ema[0, 0] == 1.0 and ema[0, 2] == 1.0
    # H2 with SPLIT: r1/r2 arrive before r0 completes -> est frozen at 8 and 2 (B=1.0), SJF picks r2 first
    c = [x for x in g["cases"] if x["name"].startswith("H2/H3")][0]
    st, dn, ema = run_oracle(c["req"], server(), wl.SJF, wl.SPLIT, 0.1)
    assert st.tolist() == c["start"]
    # after all three: Std saw m=4/3, Prem m=10/8, Batch m=3/2, one update each
    assert ema[0].tolist() == [(1.0 - 0.1) * 1.0 + 0.1 * (10 / 8), b, (1.0 - 0.1) * 1.0 + 0.1 * (3 / 2)]


def test_h4_round_robin_variant():
    # weights {1,1,1}: r0 Prem running, then queued r1 Prem, r2 Std, r3 Batch -> WEIGHTED serves r2, r3, r1
    req = [[0, 0, 1, 1, 1], [10, 0, 1, 1, 1], [20, 1, 1, 1, 1], [30, 2, 1, 1, 1]]
    sv = server(weight=(1, 1, 1))
    st, _, _ = run_oracle(req, sv, wl.WEIGHTED)
    assert np.argsort(st).tolist() == [0, 2, 3, 1]
    for pol in (wl.FIFO, wl.PRIORITY):
        st, _, _ = run_oracle(req, sv, pol)
        assert np.argsort(st).tolist() == [0, 1, 2, 3]


def test_closed_form_service_time_single_request():
    sv = server()
    rng = np.random.default_rng(3)
    for _ in range(50):
        P, O = int(rng.integers(0, 500)), int(rng.integers(1, 300))
        st, dn, _ = run_oracle([[17, 1, 5, P, O]], sv, wl.FIFO)
        assert st[0] == 17 and dn[0] - st[0] == service_time(P, O, sv)
    assert service_time(3, 2, sv) == 4322  # SURVEY.md check: 2168 + 2154


def _queue_trace(n, mean_service, rho, seed, exponential):
    rng = np.random.default_rng(seed)
    P = np.maximum(0, np.rint(rng.exponential(mean_service, n))).astype(np.int64) if exponential \
        else np.full(n, int(mean_service), np.int64)
    ia = np.maximum(0, np.rint(rng.exponential(mean_service / rho, n))).astype(np.int64)
    arr = np.cumsum(ia)
    req = np.stack([arr, np.ones(n, np.int64), P, P, np.ones(n, np.int64)], axis=1)
    return req


@pytest.mark.parametrize("rho", [0.5, 0.8])
def test_mm1_mean_wait(rho):
    # M/M/1 FIFO: Wq = rho/(mu-lambda); degenerate server c_prefill=1, everything else 0, O=1 (closed form (ii))
    n, mean_s = 1_000_000, 100_000.0
    sv = server(c_base=0, c_batch=0, c_ctx=0, c_prefill=1)
    req = _queue_trace(n, mean_s, rho, 5, True)
    st, dn, _ = run_oracle(req, sv, wl.FIFO)
    assert np.array_equal(dn - st, req[:, 3])           # service time = P ticks exactly
    wq = (st - req[:, 0]).mean()
    mu, lam = 1.0 / mean_s, rho / mean_s
    assert abs(wq / (rho / (mu - lam)) - 1.0) < 0.02


def test_md1_mean_wait():
    # Pollaczek-Khinchine, constant service: Wq = rho/(2 mu (1-rho)) (closed form (iii))
    n, mean_s, rho = 400_000, 50_000.0, 0.7
    sv = server(c_base=0, c_batch=0, c_ctx=0, c_prefill=1)
    req = _queue_trace(n, mean_s, rho, 9, False)
    st, dn, _ = run_oracle(req, sv, wl.FIFO)
    wq = (st - req[:, 0]).mean()
    assert abs(wq / (rho * mean_s / (2 * (1 - rho))) - 1.0) < 0.02


def test_sjf_beats_fifo_statistically_mg1():
    # C-SJF (ii): O=1, S = c_prefill*P, Poisson arrivals, 1e5 requests, rho 0.8: mean wait SJF < FIFO
    n, mean_s, rho = 100_000, 20_000.0, 0.8
    sv = server(c_base=0, c_batch=0, c_ctx=0, c_prefill=1)
    req = _queue_trace(n, mean_s, rho, 13, True)
    w = {}
    for pol in (wl.FIFO, wl.SJF):
        st, dn, _ = run_oracle(req, sv, pol)
        w[pol] = (st - req[:, 0]).mean()
    assert w[wl.SJF] < 0.8 * w[wl.FIFO]


@pytest.mark.parametrize("alpha", [0.05, 0.1, 0.5, 1.0])
def test_ema_geometric_closed_form(alpha):
    # constant ratio m=P/W: B_k = m + (1-m)(1-alpha)^k (closed form (iv)); trajectory sampled every completion
    k = 60
    req = [[i * 10_000_000, 1, 4, 6, 1] for i in range(k)]   # far apart: one completion at a time, m = 1.5
    sv = server(traj_every=1)
    st, dn, ema, traj = run_oracle(req, sv, wl.FIFO, wl.SPLIT, alpha, want_traj=True)
    assert traj.shape == (k, 3)
    for i in range(k):
        expect = 1.5 + (1 - 1.5) * (1 - alpha) ** (i + 1)
        assert abs(traj[i, 1] / expect - 1) < 1e-14
        assert traj[i, 0] == 1.0 and traj[i, 2] == 1.0
    assert ema[0, 1] == traj[-1, 1]


def test_ema_exact_estimator_stays_one_and_alpha_zero():
    cfg = wl.config0(oracle.characterize)
    for alpha in (0.0, 0.05, 0.1, 0.3, 0.7, 1.0):
        inst = np.zeros(1, wl.INSTANCE_DTYPE)
        inst[0] = (0, wl.SJF, wl.EXACT, 0, alpha)
        _, _, ema = oracle.simulate(cfg.trace_off, cfg.arrival, cfg.tier, cfg.words, cfg.tokens, cfg.out_len,
                                    cfg.server, inst)
        assert (ema == 1.0).all()          # (v) EXACT => B == 1.0 bit-exactly (A4)
    inst[0] = (0, wl.SJF, wl.SPLIT, 0, 0.0)   # I7: alpha=0 => BIAS OFF
    _, _, ema = oracle.simulate(cfg.trace_off, cfg.arrival, cfg.tier, cfg.words, cfg.tokens, cfg.out_len, cfg.server, inst)
    assert (ema == 1.0).all()


def test_ema_converges_to_token_word_ratio():
    # stationary drift: time-average of B -> E[P/W] = 1.3977 (north_star invariant; Fig. 5 shows the
    # same convergence of the bias factor on the real testbed)
    cfg = wl.config1(oracle.characterize, n_traces=1, n_req=4000, seed=21)
    cfg.server.traj_every = 1
    inst = np.zeros(1, wl.INSTANCE_DTYPE)
    inst[0] = (0, wl.FIFO, wl.SPLIT, 0, 0.05)
    _, _, ema, traj = oracle.simulate(cfg.trace_off, cfg.arrival, cfg.tier, cfg.words, cfg.tokens, cfg.out_len,
                                      cfg.server, inst, want_traj=True)
    assert traj.shape == (4000, 3)
    assert np.abs(traj[1000:].mean(axis=0) - 1.3977).max() < 0.02
    assert np.abs(ema[0] - 1.3977).max() < 0.08


def test_h13_weighted_cursor_wraps_after_the_last_slot():
    # H13 (A9; derivation in DESIGN.md §4.4). Weights 4:2:1 = slots PPPPSSB, max_batch 1, all O = 1, P = 1: S = 2150 + 6 = 2156.
    # t=0: only r0 (Batch) is queued, cur = 0: slots 0-5 (P, S) are empty, slot 6 serves r0 and the cursor wraps to 0.
    # r1..r4 Premium, r5 Standard, r6 Premium arrive while r0 runs. From cur = 0: four Premium slots -> r1, r2, r3, r4; slot 4 is
    # a Standard slot -> r5; slot 5: Standard and Batch empty, wrap to slot 0 -> r6. A scan that never reaches the last slot
    # serves r0 by accident but leaves cur = 1: then only three Premium slots remain and r5 overtakes r4.
    req = [[0, 2, 1, 1, 1], [10, 0, 1, 1, 1], [20, 0, 1, 1, 1], [30, 0, 1, 1, 1], [40, 0, 1, 1, 1], [50, 1, 1, 1, 1], [60, 0, 1, 1, 1]]
    st, dn, _ = run_oracle(req, server(weight=(4, 2, 1)), wl.WEIGHTED)
    assert st.tolist() == [0, 2156, 4312, 6468, 8624, 10780, 12936]
    assert dn.tolist() == [2156, 4312, 6468, 8624, 10780, 12936, 15092]


def test_h14_completions_at_one_tick_update_the_factor_in_ascending_index():
    # H14 (R-ORD: "multiple completions at one tick: ascending request index"; derivation in DESIGN.md §4.4). max_batch 2, FIFO, SPLIT,
    # alpha = 0.5. r0 = (0, Std, W 4, P 2, O 1) and r1 = (0, Std, W 2, P 3, O 1) are admitted together and both complete at
    # 2000 + 300 + 5 + 25 = 2330. r0 first: m = 0.5 -> B = 0.5 + 0.25 = 0.75; then r1: m = 1.5 -> B = 0.375 + 0.75 = 1.125.
    # (The other order gives 1.25, then 0.875.) All values are exact in binary.
    req = [[0, 1, 4, 2, 1], [0, 1, 2, 3, 1]]
    st, dn, ema, traj = run_oracle(req, server(max_batch=2, traj_every=1), wl.FIFO, wl.SPLIT, 0.5, want_traj=True)
    assert st.tolist() == [0, 0] and dn.tolist() == [2330, 2330]
    assert traj.tolist() == [[1.0, 0.75, 1.0], [1.0, 1.125, 1.0]] and ema[0].tolist() == [1.0, 1.125, 1.0]


def test_trajectory_stride():
    # traj_every = 3: sample j holds the factors after 3 (j + 1) completions; constant ratio m = 1.5 -> closed form (iv)
    k = 10
    req = [[i * 10_000_000, 1, 4, 6, 1] for i in range(k)]
    st, dn, ema, traj = run_oracle(req, server(traj_every=3), wl.FIFO, wl.SPLIT, 0.1, want_traj=True)
    assert traj.shape == (3, 3)                                    # floor(10 / 3) samples
    for j in range(3):
        expect = 1.5 + (1 - 1.5) * 0.9 ** (3 * (j + 1))
        assert abs(traj[j, 1] / expect - 1) < 1e-14 and traj[j, 0] == 1.0 and traj[j, 2] == 1.0
