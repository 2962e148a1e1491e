"""Same-name Python wrappers of the C ABI (include/driftsched.h): argument marshalling only."""
from __future__ import annotations

import ctypes as C

import numpy as np
import torch

from . import _lib
from ._lib import DsBudget, DsServer, DsTraces, check, lib

INSTANCE_BYTES = 24


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _need_cuda(*ts):
    for t in ts:
        if t is not None and (not t.is_cuda or not t.is_contiguous()):
            raise ValueError("driftsched: tensors must be contiguous CUDA tensors (no CPU fallback)")


def workspace_bytes(which, n, m):
    return int(lib().ds_workspace_bytes(which, int(n), int(m)))


def _workspace(which, n, m, device):
    return torch.empty(workspace_bytes(which, n, m), dtype=torch.uint8, device=device)


def simulate_workspace_bytes(n_total, n_inst, n_requests):
    """Both mandatory parts of the ds_simulate* workspace: per simulated request / instance, and per trace request."""
    return workspace_bytes(_lib.WS_SIMULATE, n_total, n_inst) + workspace_bytes(_lib.WS_SIMULATE_TRACES, n_requests, 0)


def launch_count():
    return int(lib().ds_launch_count())


def device_status():
    rc = lib().ds_device_status(_stream())
    if rc < 0:
        check("ds_device_status", rc)
    return rc


def characterize(text, offsets, words_out=None, tokens_out=None, workspace=None):
    """ds_characterize: text uint8[N], offsets int64[n+1] (CUDA) -> (words int32[n], tokens int32[n])."""
    _need_cuda(text, offsets, words_out, tokens_out)
    assert text.dtype == torch.uint8 and offsets.dtype == torch.int64
    n = offsets.numel() - 1
    if words_out is None:
        words_out = torch.empty(n, dtype=torch.int32, device=text.device)
    if tokens_out is None:
        tokens_out = torch.empty(n, dtype=torch.int32, device=text.device)
    if workspace is None:
        workspace = _workspace(_lib.WS_CHARACTERIZE, text.numel(), n, text.device)
    check("ds_characterize", lib().ds_characterize(_ptr(text), text.numel(), _ptr(offsets), n, _ptr(words_out), _ptr(tokens_out),
                                                   _ptr(workspace), workspace.numel(), _stream()))
    return words_out, tokens_out


def _traces(trace_off, arrival, tier, words, tokens, out_len):
    _need_cuda(trace_off, arrival, tier, words, tokens, out_len)
    assert trace_off.dtype == torch.int64 and arrival.dtype == torch.int64 and tier.dtype == torch.uint8
    assert words.dtype == torch.int32 and tokens.dtype == torch.int32 and out_len.dtype == torch.int32
    return DsTraces(trace_off.numel() - 1, trace_off.data_ptr(), arrival.data_ptr(), tier.data_ptr(), words.data_ptr(),
                    tokens.data_ptr(), out_len.data_ptr(), arrival.numel())


def _server(sv):
    return DsServer(sv.max_batch, sv.kv_budget, sv.c_base, sv.c_batch, sv.c_ctx, sv.c_prefill, (C.c_int32 * 3)(*sv.weight),
                    sv.aging_step, sv.traj_every, int(getattr(sv, "reestimate", 0)))


def instances_to_device(instances: np.ndarray, device):
    """numpy structured ds_instance array -> uint8 CUDA tensor with the same bytes."""
    assert instances.dtype.itemsize == INSTANCE_BYTES
    return torch.from_numpy(np.ascontiguousarray(instances).view(np.uint8).copy()).to(device)


def simulate(trace_off, arrival, tier, words, tokens, out_len, server, inst, out_off, n_total, start=None, done=None,
             ema_final=None, traj_off=None, ema_traj=None, workspace=None, est_out=None):
    """ds_simulate. inst: uint8 CUDA tensor holding ds_instance[n_inst]; out_off int64[n_inst+1] (CUDA);
    n_total = out_off[-1] (host int). Returns (start_tick, done_tick, ema_final[n_inst,3])."""
    tr = _traces(trace_off, arrival, tier, words, tokens, out_len)
    sv = _server(server)
    _need_cuda(inst, out_off, start, done, ema_final, traj_off, ema_traj)
    n_inst = inst.numel() // INSTANCE_BYTES
    dev = arrival.device
    if start is None:
        start = torch.empty(n_total, dtype=torch.int64, device=dev)
    if done is None:
        done = torch.empty(n_total, dtype=torch.int64, device=dev)
    if ema_final is None:
        ema_final = torch.empty((n_inst, 3), dtype=torch.float64, device=dev)
    if workspace is None:
        workspace = torch.empty(simulate_workspace_bytes(n_total, n_inst, arrival.numel()), dtype=torch.uint8, device=dev)
    if est_out is not None:                     # ds_simulate_est: same call, also writes the frozen estimates
        _need_cuda(est_out)
        assert est_out.dtype == torch.int64 and est_out.numel() >= n_total
        check("ds_simulate_est", lib().ds_simulate_est(C.byref(tr), C.byref(sv), _ptr(inst), n_inst, _ptr(out_off), int(n_total), _ptr(start),
                                                       _ptr(done), _ptr(ema_final), _ptr(traj_off), _ptr(ema_traj), _ptr(est_out),
                                                       _ptr(workspace), workspace.numel(), _stream()))
        return start, done, ema_final
    check("ds_simulate", lib().ds_simulate(C.byref(tr), C.byref(sv), _ptr(inst), n_inst, _ptr(out_off), int(n_total), _ptr(start), _ptr(done),
                                           _ptr(ema_final), _ptr(traj_off), _ptr(ema_traj), _ptr(workspace), workspace.numel(),
                                           _stream()))
    return start, done, ema_final


def simulate_est(trace_off, arrival, tier, words, tokens, out_len, server, inst, out_off, n_total, **kw):
    """ds_simulate_est -> (start_tick, done_tick, ema_final, est int64[n_total])."""
    est = kw.pop("est_out", None)
    if est is None:
        est = torch.empty(n_total, dtype=torch.int64, device=arrival.device)
    s, d, e = simulate(trace_off, arrival, tier, words, tokens, out_len, server, inst, out_off, n_total, est_out=est, **kw)
    return s, d, e, est


ERR_FIELDS = 11


def estimation_error(trace_off, arrival, tier, words, tokens, out_len, inst, out_off, n_total, est, start=None, group=None,
                     n_groups=1, want_class_seg=False, out=None, arrival_override=None):
    """ds_estimation_error -> sums int64[n_groups, 11] (and class_seg int32[n_total] if asked)."""
    tr = _traces(trace_off, arrival, tier, words, tokens, out_len)
    _need_cuda(inst, out_off, est, start, group, out, arrival_override)
    n_inst = inst.numel() // INSTANCE_BYTES
    dev = est.device
    if out is None:
        out = torch.empty((n_groups, ERR_FIELDS), dtype=torch.int64, device=dev)
    seg = torch.empty(n_total, dtype=torch.int32, device=dev) if want_class_seg else None
    check("ds_estimation_error", lib().ds_estimation_error(C.byref(tr), _ptr(inst), n_inst, _ptr(out_off), _ptr(arrival_override), _ptr(est), _ptr(start),
                                                           _ptr(group), n_groups, _ptr(out), _ptr(seg), _stream()))
    return (out, seg) if want_class_seg else out


def latencies(trace_off, arrival, tier, words, tokens, out_len, inst, out_off, n_total, start, done, group=None, t_mid=None,
              want_seg_tier=True, want_seg_all=True, out=None, arrival_override=None):
    """ds_latencies -> (e2e, qdelay, seg_tier, seg_all)."""
    tr = _traces(trace_off, arrival, tier, words, tokens, out_len)
    _need_cuda(inst, out_off, start, done, group, t_mid, arrival_override)
    n_inst = inst.numel() // INSTANCE_BYTES
    dev = start.device
    if out is not None:
        e2e, qd, st, sa = out
        _need_cuda(e2e, qd, st, sa)
    else:
        e2e = torch.empty(n_total, dtype=torch.int64, device=dev)
        qd = torch.empty(n_total, dtype=torch.int64, device=dev)
        st = torch.empty(n_total, dtype=torch.int32, device=dev) if want_seg_tier else None
        sa = torch.empty(n_total, dtype=torch.int32, device=dev) if want_seg_all else None
    check("ds_latencies", lib().ds_latencies(C.byref(tr), _ptr(inst), n_inst, _ptr(out_off), n_total, _ptr(arrival_override), _ptr(start), _ptr(done),
                                             _ptr(group), _ptr(t_mid), _ptr(e2e), _ptr(qd), _ptr(st), _ptr(sa), _stream()))
    return e2e, qd, st, sa


def tail_stats(values, seg_id, n_segments, pct=(50, 99), out=None, count_out=None, workspace=None):
    """ds_tail_stats -> (out int64[n_segments, n_pct], count int64[n_segments])."""
    _need_cuda(values, seg_id, out, count_out)
    assert values.dtype == torch.int64 and seg_id.dtype == torch.int32
    dev = values.device
    n_pct = len(pct)
    if out is None:
        out = torch.empty((n_segments, n_pct), dtype=torch.int64, device=dev)
    if count_out is None:
        count_out = torch.empty(n_segments, dtype=torch.int64, device=dev)
    if workspace is None:
        workspace = _workspace(_lib.WS_TAIL_STATS, n_segments, n_pct, dev)
    arr = (C.c_int32 * n_pct)(*[int(x) for x in pct])
    check("ds_tail_stats", lib().ds_tail_stats(_ptr(values), _ptr(seg_id), values.numel(), n_segments, arr, n_pct, _ptr(out),
                                               _ptr(count_out), _ptr(workspace), workspace.numel(), _stream()))
    return out, count_out


def tail_stats_static(values, seg_id, n_segments, out, count_out, pct=(50, 99)):
    """ds_tail_stats_static: ds_tail_stats on the library's built-in scratch array; the binding allocates nothing either, so
    `out` int64[n_segments, n_pct] and `count_out` int64[n_segments] (CUDA) must be passed in. Limit: n_segments * n_pct <= 128."""
    _need_cuda(values, seg_id, out, count_out)
    assert values.dtype == torch.int64 and seg_id.dtype == torch.int32 and out.dtype == torch.int64 and count_out.dtype == torch.int64
    n_pct = len(pct)
    arr = (C.c_int32 * n_pct)(*[int(x) for x in pct])
    check("ds_tail_stats_static", lib().ds_tail_stats_static(_ptr(values), _ptr(seg_id), values.numel(), n_segments, arr, n_pct,
                                                             _ptr(out), _ptr(count_out), _stream()))
    return out, count_out


def latency_stats(trace_off, arrival, tier, words, tokens, out_len, inst, out_off, start, done, group, n_groups, t_mid=None,
                  pct=(50, 99), e2e_out=None, qdelay_out=None, count_out=None, workspace=None, stage=True, arrival_override=None):
    """ds_latency_stats -> (e2e_out, qdelay_out, count_out), each laid out [4*G, n_pct] / [4*G] with G = n_groups * phases:
    rows [0, 3G) are the (group, tier) segments 3*g+tier, rows [3G, 4G) the per-group overall segments."""
    tr = _traces(trace_off, arrival, tier, words, tokens, out_len)
    _need_cuda(inst, out_off, start, done, group, t_mid, e2e_out, qdelay_out, count_out, arrival_override)
    n_inst = inst.numel() // INSTANCE_BYTES
    dev = start.device
    G = n_groups * (2 if t_mid is not None else 1)
    n_pct = len(pct)
    if e2e_out is None:
        e2e_out = torch.empty((4 * G, n_pct), dtype=torch.int64, device=dev)
    if qdelay_out is None:
        qdelay_out = torch.empty((4 * G, n_pct), dtype=torch.int64, device=dev)
    if count_out is None:
        count_out = torch.empty(4 * G, dtype=torch.int64, device=dev)
    if workspace is None:     # histograms + the optional staging area (5 bytes per simulated request)
        nbytes = workspace_bytes(_lib.WS_TAIL_STATS, 4 * G, n_pct)
        if stage:
            nbytes += workspace_bytes(_lib.WS_LATENCY_STAGE, int((start if start is not None else done).numel()), 0)
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    arr = (C.c_int32 * n_pct)(*[int(x) for x in pct])
    check("ds_latency_stats", lib().ds_latency_stats(C.byref(tr), _ptr(inst), n_inst, _ptr(out_off), _ptr(arrival_override), _ptr(start), _ptr(done),
                                                     _ptr(group), n_groups, _ptr(t_mid), arr, n_pct, _ptr(e2e_out), _ptr(qdelay_out),
                                                     _ptr(count_out), _ptr(workspace), workspace.numel(), _stream()))
    return e2e_out, qdelay_out, count_out


def queue_depth(trace_off, arrival, tier, words, tokens, out_len, inst, out_off, start, t0, dt, n_samples, out=None,
                arrival_override=None):
    """ds_queue_depth -> depth int32[n_inst, n_samples, 3]."""
    tr = _traces(trace_off, arrival, tier, words, tokens, out_len)
    _need_cuda(inst, out_off, start, out, arrival_override)
    n_inst = inst.numel() // INSTANCE_BYTES
    if out is None:
        out = torch.empty((n_inst, int(n_samples), 3), dtype=torch.int32, device=start.device)
    check("ds_queue_depth", lib().ds_queue_depth(C.byref(tr), _ptr(inst), n_inst, _ptr(out_off), _ptr(arrival_override), _ptr(start), int(t0), int(dt),
                                                 int(n_samples), _ptr(out), _stream()))
    return out


def simulate_budget(trace_off, arrival, tier, words, tokens, out_len, category, budget, server, inst, out_off, n_total,
                    start=None, done=None, ema_final=None, traj_off=None, ema_traj=None, est_out=None, workspace=None,
                    n_clients=0, think_ticks=0, arrival_out=None, batch_wait=0):
    """ds_simulate_budget. category uint8 CUDA tensor (per request); budget: object with t_base[4], s_tenant[3], f_slope,
    f_max. Returns (start_tick, done_tick, ema_final[n_inst,4])."""
    tr = _traces(trace_off, arrival, tier, words, tokens, out_len)
    sv = _server(server)
    bp = DsBudget((C.c_double * 4)(*budget.t_base), (C.c_double * 3)(*budget.s_tenant), budget.f_slope, budget.f_max)
    _need_cuda(category, inst, out_off, start, done, ema_final, traj_off, ema_traj, est_out)
    assert category.dtype == torch.uint8 and category.numel() == tier.numel()
    n_inst = inst.numel() // INSTANCE_BYTES
    dev = arrival.device
    if start is None:
        start = torch.empty(n_total, dtype=torch.int64, device=dev)
    if done is None:
        done = torch.empty(n_total, dtype=torch.int64, device=dev)
    if ema_final is None:
        ema_final = torch.empty((n_inst, 4), dtype=torch.float64, device=dev)
    if workspace is None:
        workspace = torch.empty(simulate_workspace_bytes(n_total, n_inst, arrival.numel()), dtype=torch.uint8, device=dev)
    if n_clients > 0:   # ds_simulate_closed: closed-loop arrivals, returns arrival_out as a 4th element
        if arrival_out is None:
            arrival_out = torch.empty(n_total, dtype=torch.int64, device=dev)
        _need_cuda(arrival_out)
        check("ds_simulate_closed", lib().ds_simulate_closed(C.byref(tr), _ptr(category), C.byref(bp), C.byref(sv), int(n_clients),
                                                             int(think_ticks), int(batch_wait), _ptr(inst), n_inst, _ptr(out_off), int(n_total), _ptr(arrival_out),
                                                             _ptr(start), _ptr(done), _ptr(ema_final), _ptr(traj_off), _ptr(ema_traj),
                                                             _ptr(est_out), _ptr(workspace), workspace.numel(), _stream()))
        return start, done, ema_final, arrival_out
    check("ds_simulate_budget", lib().ds_simulate_budget(C.byref(tr), _ptr(category), C.byref(bp), C.byref(sv), _ptr(inst), n_inst,
                                                         _ptr(out_off), int(n_total), _ptr(start), _ptr(done), _ptr(ema_final), _ptr(traj_off),
                                                         _ptr(ema_traj), _ptr(est_out), _ptr(workspace), workspace.numel(), _stream()))
    return start, done, ema_final


def simulate_closed(trace_off, arrival, tier, words, tokens, out_len, category, budget, server, n_clients, think_ticks, batch_wait,
                    inst, out_off, n_total, **kw):
    """ds_simulate_closed -> (start_tick, done_tick, ema_final[n_inst,4], arrival_out)."""
    if n_clients < 1:
        raise ValueError("ds_simulate_closed: n_clients >= 1")
    return simulate_budget(trace_off, arrival, tier, words, tokens, out_len, category, budget, server, inst, out_off, n_total,
                           n_clients=n_clients, think_ticks=think_ticks, batch_wait=batch_wait, **kw)
