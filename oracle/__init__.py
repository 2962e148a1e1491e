"""CPU ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT (see oracle.h).

ctypes wrapper around liboracle.so (plain single-threaded C++, built with -ffp-contract=off). Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package. It
imports nothing from the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, "oracle.cpp"), os.path.join(_HERE, "oracle.h")]

INSTANCE_DTYPE = np.dtype(
    [("trace", "<i4"), ("policy", "<i4"), ("estimator", "<i4"), ("_pad", "<i4"), ("ema_alpha", "<f8")]
)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or any(os.path.getmtime(_SO) < os.path.getmtime(s) for s in _SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-o", _SO, _SRC[0]])
    return _SO


class _Traces(C.Structure):
    _fields_ = [("n_traces", C.c_int64), ("trace_off", C.c_void_p), ("arrival_tick", C.c_void_p), ("tier", C.c_void_p),
                ("words", C.c_void_p), ("tokens", C.c_void_p), ("out_len", C.c_void_p)]


class _Server(C.Structure):
    _fields_ = [("max_batch", C.c_int32), ("kv_budget", C.c_int64), ("c_base", C.c_int64), ("c_batch", C.c_int64),
                ("c_ctx", C.c_int64), ("c_prefill", C.c_int64), ("weight", C.c_int32 * 3), ("aging_step", C.c_int64),
                ("traj_every", C.c_int32), ("reestimate", C.c_int32)]


class _Budget(C.Structure):
    _fields_ = [("t_base", C.c_double * 4), ("s_tenant", C.c_double * 3), ("f_slope", C.c_double), ("f_max", C.c_double)]


_lib = None


def _o():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        p = C.c_void_p
        lib.oracle_characterize.argtypes = [p, C.c_int64, p, C.c_int64, p, p]
        lib.oracle_simulate.argtypes = [p, p, p, C.c_int64, p, p, p, p, p, p, p]
        lib.oracle_estimation_error.argtypes = [p, p, C.c_int64, p, p, p, p, p, C.c_int32, p, p]
        lib.oracle_estimation_error.restype = C.c_int
        lib.oracle_queue_depth.argtypes = [p, p, C.c_int64, p, p, p, C.c_int64, C.c_int64, C.c_int64, p]
        lib.oracle_queue_depth.restype = C.c_int
        lib.oracle_simulate_budget.argtypes = [p, p, p, p, p, C.c_int64, p, p, p, p, p, p, p]
        lib.oracle_simulate_budget.restype = C.c_int
        lib.oracle_simulate_closed.argtypes = [p, p, p, p, C.c_int64, C.c_int64, C.c_int64, p, C.c_int64, p, p, p, p, p, p, p, p]
        lib.oracle_simulate_closed.restype = C.c_int
        lib.oracle_latencies.argtypes = [p, p, C.c_int64, p, p, p, p, p, p, p, p, p, p]
        lib.oracle_tail_stats.argtypes = [p, p, C.c_int64, C.c_int32, p, C.c_int32, p, p]
        for f in (lib.oracle_characterize, lib.oracle_simulate, lib.oracle_latencies, lib.oracle_tail_stats):
            f.restype = C.c_int
        _lib = lib
    return _lib


def _c(a, dt):
    a = np.ascontiguousarray(a, dt)
    return a


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def characterize(text, offsets):
    text = _c(text, np.uint8)
    offsets = _c(offsets, np.int64)
    n = len(offsets) - 1
    w = np.zeros(n, np.int32)
    t = np.zeros(n, np.int32)
    rc = _o().oracle_characterize(_p(text), text.size, _p(offsets), n, _p(w), _p(t))
    if rc:
        raise ValueError("oracle_characterize: contract violation")
    return w, t


def _traces(trace_off, arrival, tier, words, tokens, out_len):
    keep = [_c(trace_off, np.int64), _c(arrival, np.int64), _c(tier, np.uint8), _c(words, np.int32),
            _c(tokens, np.int32), _c(out_len, np.int32)]
    tr = _Traces(len(keep[0]) - 1, *[_p(a).value if a.size else 0 for a in keep])
    return tr, keep


def _server(sv):
    return _Server(sv.max_batch, sv.kv_budget, sv.c_base, sv.c_batch, sv.c_ctx, sv.c_prefill,
                   (C.c_int32 * 3)(*sv.weight), sv.aging_step, sv.traj_every, int(getattr(sv, "reestimate", 0)))


def traj_offsets(trace_off, instances, traj_every):
    n_per = np.diff(np.asarray(trace_off, np.int64))[instances["trace"]]
    k = n_per // traj_every if traj_every > 0 else np.zeros_like(n_per)
    return np.concatenate([[0], np.cumsum(k)]).astype(np.int64)


def simulate(trace_off, arrival, tier, words, tokens, out_len, server, instances, out_off=None, want_traj=False,
             want_est=False):
    """Returns start_tick, done_tick, ema_final[n_inst,3] (then ema_traj[samples,3] if want_traj, then est if want_est)."""
    tr, keep = _traces(trace_off, arrival, tier, words, tokens, out_len)
    sv = _server(server)
    inst = _c(instances, INSTANCE_DTYPE)
    n_inst = len(inst)
    n_per = np.diff(keep[0])[inst["trace"]] if n_inst else np.zeros(0, np.int64)
    if out_off is None:
        out_off = np.concatenate([[0], np.cumsum(n_per)]).astype(np.int64)
    out_off = _c(out_off, np.int64)
    total = int(out_off[-1]) if n_inst else 0
    start = np.full(total, -1, np.int64)
    done = np.full(total, -1, np.int64)
    ema = np.zeros((n_inst, 3), np.float64)
    toff = traj = None
    if want_traj and server.traj_every > 0:
        toff = traj_offsets(keep[0], inst, server.traj_every)
        traj = np.zeros((int(toff[-1]), 3), np.float64)
    est = np.full(total, -1, np.int64) if want_est else None
    rc = _o().oracle_simulate(C.byref(tr), C.byref(sv), _p(inst), n_inst, _p(out_off), _p(start), _p(done), _p(ema),
                              _p(toff), _p(traj), _p(est))
    if rc:
        raise ValueError("oracle_simulate: contract violation")
    out = (start, done, ema) + ((traj,) if want_traj else ()) + ((est,) if want_est else ())
    return out


def latencies(trace_off, arrival, tier, words, tokens, out_len, instances, out_off, start, done, group=None, t_mid=None,
              arrival_override=None):
    tr, keep = _traces(trace_off, arrival, tier, words, tokens, out_len)
    inst = _c(instances, INSTANCE_DTYPE)
    out_off = _c(out_off, np.int64)
    start = _c(start, np.int64)
    done = _c(done, np.int64)
    n = start.size
    e2e = np.zeros(n, np.int64)
    qd = np.zeros(n, np.int64)
    st = np.zeros(n, np.int32)
    sa = np.zeros(n, np.int32)
    g = None if group is None else _c(group, np.int32)
    tm = None if t_mid is None else _c(t_mid, np.int64)
    ao = None if arrival_override is None else _c(arrival_override, np.int64)
    rc = _o().oracle_latencies(C.byref(tr), _p(inst), len(inst), _p(out_off), _p(ao), _p(start), _p(done), _p(g), _p(tm),
                               _p(e2e), _p(qd), _p(st), _p(sa))
    assert rc == 0
    return e2e, qd, st, sa


def tail_stats(values, seg_id, n_segments, pct=(50, 99)):
    values = _c(values, np.int64)
    seg_id = _c(seg_id, np.int32)
    pct = _c(pct, np.int32)
    out = np.zeros((n_segments, len(pct)), np.int64)
    cnt = np.zeros(n_segments, np.int64)
    rc = _o().oracle_tail_stats(_p(values), _p(seg_id), values.size, n_segments, _p(pct), len(pct), _p(out), _p(cnt))
    assert rc == 0
    return out, cnt


ERR_FIELDS = ("n", "sum_abs_err", "sum_sq_err", "sum_est", "sum_tokens", "n_short", "n_medium", "n_long",
              "sum_qdelay_short", "sum_qdelay_medium", "sum_qdelay_long")


def estimation_error(trace_off, arrival, tier, words, tokens, out_len, instances, out_off, est, start, group, n_groups,
                     want_class_seg=False, arrival_override=None):
    """-> sums int64[n_groups, 11] (ERR_FIELDS) and, if asked, class_seg int32 per simulated request."""
    tr, keep = _traces(trace_off, arrival, tier, words, tokens, out_len)
    inst = _c(instances, INSTANCE_DTYPE)
    out_off = _c(out_off, np.int64)
    est = _c(est, np.int64)
    start = None if start is None else _c(start, np.int64)
    g = None if group is None else _c(group, np.int32)
    out = np.zeros((n_groups, 11), np.int64)
    seg = np.zeros(est.size, np.int32) if want_class_seg else None
    ao = None if arrival_override is None else _c(arrival_override, np.int64)
    rc = _o().oracle_estimation_error(C.byref(tr), _p(inst), len(inst), _p(out_off), _p(ao), _p(est), _p(start), _p(g), n_groups,
                                      _p(out), _p(seg))
    if rc:
        raise ValueError("oracle_estimation_error: contract violation")
    return (out, seg) if want_class_seg else out


def queue_depth(trace_off, arrival, tier, words, tokens, out_len, instances, out_off, start, t0, dt, n_samples,
                arrival_override=None):
    """-> depth int32[n_inst, n_samples, 3]: requests of each tier queued (arrival <= t < start) at t = t0 + j*dt."""
    tr, keep = _traces(trace_off, arrival, tier, words, tokens, out_len)
    inst = _c(instances, INSTANCE_DTYPE)
    out_off = _c(out_off, np.int64)
    start = _c(start, np.int64)
    depth = np.zeros((len(inst), int(n_samples), 3), np.int32)
    ao = None if arrival_override is None else _c(arrival_override, np.int64)
    rc = _o().oracle_queue_depth(C.byref(tr), _p(inst), len(inst), _p(out_off), _p(ao), _p(start), int(t0), int(dt), int(n_samples),
                                 _p(depth))
    if rc:
        raise ValueError("oracle_queue_depth: contract violation")
    return depth


def simulate_budget(trace_off, arrival, tier, words, tokens, out_len, category, budget, server, instances, out_off=None,
                    want_traj=False, want_est=False, n_clients=0, think_ticks=0, batch_wait=0):
    """Full Eq. 1-2 estimator with per-category feedback. budget: object with t_base[4], s_tenant[3], f_slope, f_max.
    Returns start_tick, done_tick, ema_final[n_inst,4] (then ema_traj[samples,4] if want_traj, then est if want_est)."""
    tr, keep = _traces(trace_off, arrival, tier, words, tokens, out_len)
    cat = _c(category, np.uint8)
    assert cat.size == keep[1].size
    bp = _Budget((C.c_double * 4)(*budget.t_base), (C.c_double * 3)(*budget.s_tenant), budget.f_slope, budget.f_max)
    sv = _server(server)
    inst = _c(instances, INSTANCE_DTYPE)
    n_inst = len(inst)
    if out_off is None:
        sizes = np.array([keep[0][i["trace"] + 1] - keep[0][i["trace"]] for i in inst], np.int64)
        out_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    out_off = _c(out_off, np.int64)
    total = int(out_off[-1])
    start = np.full(total, -1, np.int64)
    done = np.full(total, -1, np.int64)
    ema = np.zeros((n_inst, 4), np.float64)
    toff = traj = None
    if want_traj and server.traj_every > 0:
        toff = traj_offsets(keep[0], inst, server.traj_every)
        traj = np.zeros((int(toff[-1]), 4), np.float64)
    est = np.full(total, -1, np.int64) if want_est else None
    if n_clients > 0:   # closed loop: also returns the arrival tick of every simulated request (last element)
        arr_out = np.full(total, -1, np.int64)
        rc = _o().oracle_simulate_closed(C.byref(tr), _p(cat), C.byref(bp), C.byref(sv), int(n_clients), int(think_ticks), int(batch_wait),
                                         _p(inst),
                                         n_inst, _p(out_off), _p(arr_out), _p(start), _p(done), _p(ema), _p(toff), _p(traj), _p(est))
        if rc:
            raise ValueError("oracle_simulate_closed: contract violation")
        return (start, done, ema) + ((traj,) if want_traj else ()) + ((est,) if want_est else ()) + (arr_out,)
    rc = _o().oracle_simulate_budget(C.byref(tr), _p(cat), C.byref(bp), C.byref(sv), _p(inst), n_inst, _p(out_off), _p(start),
                                     _p(done), _p(ema), _p(toff), _p(traj), _p(est))
    if rc:
        raise ValueError("oracle_simulate_budget: contract violation")
    return (start, done, ema) + ((traj,) if want_traj else ()) + ((est,) if want_est else ())
