"""Seeded synthetic workloads shaped like BASELINE.json:configs[0..4] (recipe: DESIGN.md §5).

Inputs only.  This module (and gen.cpp beside it) holds none of the method's arithmetic: word/token
counts of generated text are obtained by calling a ``characterize`` function supplied by the caller
(the CUDA binding in bench/GPU tests, the oracle in CPU tests).  It is the one module that both the
oracle's tests and the CUDA path's tests import.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libdsgen.so")
_SRC = os.path.join(_HERE, "gen.cpp")

FIFO, PRIORITY, WEIGHTED, SJF, AGING = 0, 1, 2, 3, 4
AGING_UNCLAMPED = 5   # NEXT-4 variant (A15): the aging score is not clamped at Premium's level
SPLIT, EXACT = 0, 1
BUDGET_SPLIT, BUDGET_EXACT = 2, 3
POLICY_NAMES = ["FIFO", "PRIORITY", "WEIGHTED", "SJF", "AGING", "AGING_UNCLAMPED"]

# layout of ds_instance in include/driftsched.h (24 bytes)
INSTANCE_DTYPE = np.dtype(
    [("trace", "<i4"), ("policy", "<i4"), ("estimator", "<i4"), ("_pad", "<i4"), ("ema_alpha", "<f8")]
)


def build_generator(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", "-o", _SO, _SRC])
    return _SO


_lib = None


def _gen():
    global _lib
    if _lib is None:
        lib = C.CDLL(build_generator())
        p = C.c_void_p
        lib.dsgen_text.restype = C.c_int64
        lib.dsgen_text.argtypes = [C.c_uint64, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double,
                                   p, p, C.c_int64, p, C.c_int]
        lib.dsgen_requests.restype = None
        lib.dsgen_requests.argtypes = [C.c_uint64, C.c_int64, C.c_int64, C.c_int, p, p, p, C.c_int]
        lib.dsgen_counts.restype = None
        lib.dsgen_counts.argtypes = [C.c_uint64, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double,
                                     p, p, p, C.c_int]
        lib.dsgen_scan_layout.restype = C.c_int64
        lib.dsgen_scan_layout.argtypes = [C.c_uint64, C.c_int64, C.c_int64, p, p]
        lib.dsgen_scan_fill.restype = None
        lib.dsgen_scan_fill.argtypes = [C.c_uint64, C.c_int64, p, p, C.c_int64, C.c_int64, p, C.c_int]
        _lib = lib
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _threads():
    return max(1, min(32, os.cpu_count() or 1))


LAW0 = (0.3, 0.1)    # word-length geometric p, punctuation p (configs[0])
LAW1 = (0.15, 0.35)  # post-drift law (configs[4])


def make_text(seed, n_traces, n_req, post_drift=None, law0=LAW0, law1=LAW1):
    """Packed prompt text (uint8) + int64 offsets[n+1] for n_traces*n_req prompts, trace-major."""
    g = _gen()
    n = n_traces * n_req
    off = np.empty(n + 1, np.int64)
    pd = None if post_drift is None else np.ascontiguousarray(post_drift, np.uint8)
    total = g.dsgen_text(seed, n_traces, n_req, law0[0], law0[1], law1[0], law1[1], _ptr(pd), None, 0, _ptr(off), _threads())
    buf = np.empty(total, np.uint8)
    r = g.dsgen_text(seed, n_traces, n_req, law0[0], law0[1], law1[0], law1[1], _ptr(pd), _ptr(buf), total, _ptr(off), _threads())
    assert r == total
    return buf, off


def make_requests(seed, n_traces, n_req, out_dist=0):
    """tier u8 (20/50/30), out_len i32, unit-mean exponential inter-arrival draws f64."""
    n = n_traces * n_req
    tier = np.empty(n, np.uint8)
    out_len = np.empty(n, np.int32)
    expo = np.empty(n, np.float64)
    _gen().dsgen_requests(seed, n_traces, n_req, out_dist, _ptr(tier), _ptr(out_len), _ptr(expo), _threads())
    return tier, out_len, expo


def make_counts(seed, n_traces, n_req, post_drift=None, law0=LAW0, law1=LAW1):
    """Text-free (words, tokens) per request for configs 3/4 (see gen.cpp: dsgen_counts)."""
    n = n_traces * n_req
    w = np.empty(n, np.int32)
    t = np.empty(n, np.int32)
    pd = None if post_drift is None else np.ascontiguousarray(post_drift, np.uint8)
    _gen().dsgen_counts(seed, n_traces, n_req, law0[0], law0[1], law1[0], law1[1], _ptr(pd), _ptr(w), _ptr(t), _threads())
    return w, t


def make_scan_layout(seed, total_bytes):
    """configs[2] prompt layout: offsets[n+1], kind[n] for exactly total_bytes of text."""
    cap = max(1024, total_bytes // 64 + 1024)
    off = np.empty(cap + 1, np.int64)
    kind = np.empty(cap, np.uint8)
    n = _gen().dsgen_scan_layout(seed, total_bytes, cap, _ptr(off), _ptr(kind))
    assert n >= 0
    return off[: n + 1].copy(), kind[:n].copy()


def fill_scan_text(seed, off, kind, first, end, out):
    """Fill prompts [first,end) of a configs[2] layout into `out` (uint8, len off[end]-off[first])."""
    assert out.dtype == np.uint8 and out.size == off[end] - off[first] and out.flags.c_contiguous
    _gen().dsgen_scan_fill(seed, len(kind), _ptr(off), _ptr(kind), first, end, _ptr(out), _threads())


def make_scan_text(seed, total_bytes):
    off, kind = make_scan_layout(seed, total_bytes)
    buf = np.empty(total_bytes, np.uint8)
    fill_scan_text(seed, off, kind, 0, len(kind), buf)
    return buf, off


@dataclass
class Server:
    """Mirror of ds_server (include/driftsched.h); cost constants from BASELINE.json:configs[0]."""
    max_batch: int = 8
    kv_budget: int = 0
    c_base: int = 2000
    c_batch: int = 150
    c_ctx: int = 1
    c_prefill: int = 5
    weight: tuple = (4, 2, 1)
    aging_step: int = 500_000
    traj_every: int = 0
    reestimate: int = 0      # 1: online re-estimation of queued requests (NEXT-4; A16)


@dataclass
class Budget:
    """Mirror of ds_budget (include/driftsched.h): parameters of the paper's full estimator, Eq. 1-2.
    The paper prints none of these constants; the defaults put T_base 25 % above each category's mean synthetic output
    so that the feedback factor settles near 0.8, the range of Fig. 5."""
    t_base: tuple = (38.0, 113.0, 189.0, 265.0)     # short_qa, summary, technical, report
    s_tenant: tuple = (1.0, 1.0, 1.0)
    f_slope: float = 0.0
    f_max: float = 1.0


CATEGORY_OUT_SCALE = (0.25, 0.75, 1.25, 1.75)       # mean output of a category relative to the trace's output law


def assign_categories(seed, out_len, cap=512):
    """Synthetic semantic categories (the paper's corpus, ~295 prompts per category, is not available):
    each request gets one of four categories uniformly (seeded), and its decode length is rescaled by the category's
    factor so that categories differ in output length as in Table I. Returns (category u8, out_len i32)."""
    rng = np.random.default_rng([int(seed), 0xC47])
    cat = rng.integers(0, 4, size=out_len.shape[0]).astype(np.uint8)
    scale = np.asarray(CATEGORY_OUT_SCALE)[cat]
    o = np.clip(np.rint(out_len.astype(np.float64) * scale), 1, cap).astype(np.int32)
    return cat, o


def mean_interarrival_ticks(rho, tokens, out_len, sv: Server):
    """Offered load rho -> mean inter-arrival (ticks) for ONE trace: S_bar/rho with S_bar the
    per-request server time at a full batch (SURVEY.md §8(d) 'Arrivals')."""
    O = out_len.astype(np.float64)
    P = tokens.astype(np.float64)
    s_bar = (O.mean() * (sv.c_base / sv.max_batch + sv.c_batch)
             + sv.c_ctx * ((O * P).mean() + (O * (O - 1.0)).mean() / 2.0) + sv.c_prefill * P.mean())
    return s_bar / rho


def make_arrivals(expo, n_traces, n_req, mean_ticks):
    """arrival_tick[i] = cumsum(max(0, round(expo*mean))) per trace; mean_ticks scalar or [n_traces]."""
    e = expo.reshape(n_traces, n_req)
    m = np.broadcast_to(np.asarray(mean_ticks, np.float64).reshape(-1, 1), (n_traces, 1))
    ia = np.maximum(0, np.rint(e * m)).astype(np.int64)
    return np.cumsum(ia, axis=1).reshape(-1)


@dataclass
class Workload:
    name: str
    n_traces: int
    n_req: int
    server: Server
    trace_off: np.ndarray
    arrival: np.ndarray
    tier: np.ndarray
    words: np.ndarray
    tokens: np.ndarray
    out_len: np.ndarray
    instances: np.ndarray            # INSTANCE_DTYPE
    group: np.ndarray                # int32 [n_inst] reporting group (policy x estimator x alpha index)
    n_groups: int
    text: np.ndarray | None = None
    offsets: np.ndarray | None = None
    t_mid: np.ndarray | None = None  # int64 [n_traces] drift split tick (configs[4])
    extra: dict = field(default_factory=dict)

    @property
    def n_inst(self):
        return len(self.instances)

    @property
    def out_off(self):
        return (np.arange(self.n_inst + 1, dtype=np.int64) * self.n_req)

    @property
    def sim_requests(self):
        return self.n_inst * self.n_req


def make_instances(n_traces, combos):
    """combos: list of (policy, estimator, alpha). Trace-major so the instances of one trace run together."""
    inst = np.zeros(n_traces * len(combos), INSTANCE_DTYPE)
    grp = np.zeros(n_traces * len(combos), np.int32)
    k = 0
    for t in range(n_traces):
        for gidx, (pol, est, a) in enumerate(combos):
            inst[k] = (t, pol, est, 0, a)
            grp[k] = gidx
            k += 1
    return inst, grp


def _trace_workload(name, seed, n_traces, n_req, sv, combos, characterize, *, rho=None, mean_ticks=None,
                    out_dist=0, drift=False, materialise=True, text_traces=0):
    tier, out_len, expo = make_requests(seed, n_traces, n_req, out_dist)
    post = None
    if drift:
        ce = np.cumsum(expo.reshape(n_traces, n_req), axis=1)
        post = (ce >= ce[:, -1:] / 2.0).reshape(-1).astype(np.uint8)
    text = offsets = None
    if materialise:
        text, offsets = make_text(seed, n_traces, n_req, post)
        words, tokens = characterize(text, offsets)
        words = np.asarray(words, np.int32)
        tokens = np.asarray(tokens, np.int32)
    else:
        words, tokens = make_counts(seed, n_traces, n_req, post)
        if text_traces > 0:
            # text-free configuration with a materialised sample: the prompts of the first text_traces traces exist as text
            # and their (W, P) come from `characterize`; the remaining traces keep the numeric draw of the same word law
            nt = min(text_traces, n_traces)
            text, offsets = make_text(seed, nt, n_req, None if post is None else post[:nt * n_req])
            w, t = characterize(text, offsets)
            words[:nt * n_req] = np.asarray(w, np.int32)
            tokens[:nt * n_req] = np.asarray(t, np.int32)
    if mean_ticks is None:
        mean_ticks = np.array([
            mean_interarrival_ticks(rho, tokens[t * n_req:(t + 1) * n_req], out_len[t * n_req:(t + 1) * n_req], sv)
            for t in range(n_traces)])
    arrival = make_arrivals(expo, n_traces, n_req, mean_ticks)
    inst, grp = make_instances(n_traces, combos)
    t_mid = None
    if drift:
        a2 = arrival.reshape(n_traces, n_req)
        first_post = post.reshape(n_traces, n_req).argmax(axis=1)
        t_mid = a2[np.arange(n_traces), first_post].astype(np.int64)
    return Workload(name, n_traces, n_req, sv, np.arange(n_traces + 1, dtype=np.int64) * n_req, arrival, tier,
                    words, tokens, out_len, inst, grp, len(combos), text, offsets, t_mid,
                    {"post_drift": post, "combos": combos})


def paper_phases(characterize, n_runs=3, seed=7, n_cal=1000, n_stress=2000, rho_cal=0.5, rho_stress=1.3):
    """The paper's experiment shape: per run 1000 calibration requests followed by 2000 stress
    requests, batch 32, feedback on throughout, three runs; Weighted 50/30/20 = weight {5,3,2}; the three
    estimator modes of Table IX (split() OFF, split() ON, tokenizer-aware ON) for all five policies, with the full
    estimator of Eq. 1-2 over four synthetic semantic categories. The paper's arrivals are closed-loop (50 clients);
    here they stay an open-loop input (reading A12): the calibration phase arrives at offered load rho_cal, the stress
    phase at rho_stress. t_mid[run] = arrival of the first stress request, so ds_latencies' phases = calibration/stress.
    Returns (Workload, category u8, Budget); Workload.out_len already carries the per-category output scaling."""
    n_req = n_cal + n_stress
    sv = Server(max_batch=32, kv_budget=16384, weight=(5, 3, 2), aging_step=500_000, traj_every=100)
    combos = [(p, e, a) for p in ALL_POLICIES for e, a in ((BUDGET_SPLIT, 0.0), (BUDGET_SPLIT, 0.1), (BUDGET_EXACT, 0.1))]
    c = _trace_workload("paper_phases", seed, n_runs, n_req, sv, combos, characterize, rho=1.0)
    cat, out_len = assign_categories(seed, c.out_len)
    _, _, expo = make_requests(seed, n_runs, n_req, 0)
    arrival = np.empty(n_runs * n_req, np.int64)
    t_mid = np.empty(n_runs, np.int64)
    for t in range(n_runs):
        sl = slice(t * n_req, (t + 1) * n_req)
        s_bar = mean_interarrival_ticks(1.0, c.tokens[sl], out_len[sl], sv)
        mean = np.concatenate([np.full(n_cal, s_bar / rho_cal), np.full(n_stress, s_bar / rho_stress)])
        ia = np.maximum(0, np.rint(expo[sl] * mean)).astype(np.int64)
        arrival[sl] = np.cumsum(ia)
        t_mid[t] = arrival[t * n_req + n_cal]
    c.arrival, c.out_len, c.t_mid = arrival, out_len, t_mid
    return c, cat, Budget()


def config0(characterize):
    """configs[0]: 1 trace, 200 requests, seed 0, 2 req/s, batch 8, KV unlimited, FIFO+SJF, split()+EMA 0.1."""
    sv = Server(max_batch=8, kv_budget=0)
    return _trace_workload("cfg0", 0, 1, 200, sv, [(FIFO, SPLIT, 0.1), (SJF, SPLIT, 0.1)], characterize,
                           mean_ticks=500_000.0)


ALL_POLICIES = [FIFO, PRIORITY, WEIGHTED, SJF, AGING]


def config1(characterize, n_traces=1024, n_req=2000, seed=1):
    """configs[1]: policy sweep, 5 policies x {split()+EMA 0.1, exact}, rho 0.85, batch 32, KV 16384."""
    sv = Server(max_batch=32, kv_budget=16384, aging_step=500_000)
    combos = [(p, e, 0.1) for p in ALL_POLICIES for e in (SPLIT, EXACT)]
    return _trace_workload("cfg1", seed, n_traces, n_req, sv, combos, characterize, rho=0.85)


def config3(characterize=None, n_traces=16384, n_req=10000, seed=3, materialise=False, text_traces=0):
    """configs[3]: heavy contention, Pareto outputs, batch 128, KV 65536, aging 250 ms, 4 alphas. text_traces > 0: the
    prompts of the first text_traces traces are materialised as text (Workload.text / .offsets cover those prompts only)
    and characterised by `characterize`; SURVEY.md §8(d) draws the other traces' (W, P) numerically."""
    sv = Server(max_batch=128, kv_budget=65536, aging_step=250_000)
    combos = [(p, SPLIT, a) for p in ALL_POLICIES for a in (0.05, 0.1, 0.2, 0.5)]
    return _trace_workload("cfg3", seed, n_traces, n_req, sv, combos, characterize, rho=0.95, out_dist=1,
                           materialise=materialise, text_traces=text_traces)


def config4(characterize=None, n_traces=4096, n_req=50000, seed=4, materialise=False, traj_every=1000):
    """configs[4]: token drift at the trace's midpoint tick, batch 256, KV 131072, both estimators."""
    sv = Server(max_batch=256, kv_budget=131072, traj_every=traj_every)
    combos = [(p, e, 0.1) for p in ALL_POLICIES for e in (SPLIT, EXACT)]
    return _trace_workload("cfg4", seed, n_traces, n_req, sv, combos, characterize, rho=0.9, drift=True,
                           materialise=materialise)


def config2(total_bytes=8 << 30, seed=2):
    """configs[2]: characterization-only scan buffer (bytes, offsets)."""
    return make_scan_text(seed, total_bytes)
