"""ctypes loader for libdriftsched.so. Argument marshalling only; fails loudly when the library is missing."""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdriftsched.so")

DS_OK, DS_EINVAL, DS_ECUDA, DS_ENOMEM, DS_ELIMIT = 0, -1, -2, -3, -4
TAIL_STATS_STATIC_MAX_SEGPCT = 128
WS_CHARACTERIZE, WS_SIMULATE, WS_TAIL_STATS = 0, 1, 2
WS_LATENCY_STAGE = 3
WS_SIMULATE_TRACES = 4

EXPORTS = ["ds_characterize", "ds_simulate", "ds_simulate_est", "ds_simulate_budget", "ds_simulate_closed", "ds_estimation_error", "ds_queue_depth", "ds_latencies", "ds_tail_stats",
           "ds_tail_stats_static", "ds_latency_stats", "ds_workspace_bytes", "ds_device_status",
           "ds_strerror", "ds_last_cuda_error", "ds_launch_count"]


class DsTraces(C.Structure):
    _fields_ = [("n_traces", C.c_int64), ("trace_off", C.c_void_p), ("arrival_tick", C.c_void_p), ("tier", C.c_void_p),
                ("words", C.c_void_p), ("tokens", C.c_void_p), ("out_len", C.c_void_p), ("n_requests", C.c_int64)]


class DsServer(C.Structure):
    _fields_ = [("max_batch", C.c_int32), ("kv_budget", C.c_int64), ("c_base", C.c_int64), ("c_batch", C.c_int64),
                ("c_ctx", C.c_int64), ("c_prefill", C.c_int64), ("weight", C.c_int32 * 3), ("aging_step", C.c_int64),
                ("traj_every", C.c_int32), ("reestimate", C.c_int32)]


class DsBudget(C.Structure):
    _fields_ = [("t_base", C.c_double * 4), ("s_tenant", C.c_double * 3), ("f_slope", C.c_double), ("f_max", C.c_double)]


class DsError(RuntimeError):
    def __init__(self, fn, code, detail=""):
        super().__init__(f"{fn} failed: {code} ({detail})")
        self.code = code


_lib = None


def lib():
    """The loaded library. Raises if it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_02982_b200.build` "
                              "(there is no CPU or PyTorch fallback)")
        L = C.CDLL(LIB_PATH)
        p, i64, i32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_size_t
        L.ds_characterize.argtypes = [p, i64, p, i64, p, p, p, sz, p]
        L.ds_simulate.argtypes = [C.POINTER(DsTraces), C.POINTER(DsServer), p, i64, p, i64, p, p, p, p, p, p, sz, p]
        L.ds_simulate_est.argtypes = [C.POINTER(DsTraces), C.POINTER(DsServer), p, i64, p, i64, p, p, p, p, p, p, p, sz, p]
        L.ds_simulate_budget.argtypes = [C.POINTER(DsTraces), p, C.POINTER(DsBudget), C.POINTER(DsServer), p, i64, p, i64, p, p, p, p, p, p, p, sz, p]
        L.ds_simulate_closed.argtypes = [C.POINTER(DsTraces), p, C.POINTER(DsBudget), C.POINTER(DsServer), i32, i64, i64, p, i64, p, i64, p, p, p, p, p, p, p, p, sz, p]
        L.ds_estimation_error.argtypes = [C.POINTER(DsTraces), p, i64, p, p, p, p, p, i32, p, p, p]
        L.ds_queue_depth.argtypes = [C.POINTER(DsTraces), p, i64, p, p, p, i64, i64, i64, p, p]
        L.ds_latencies.argtypes = [C.POINTER(DsTraces), p, i64, p, i64, p, p, p, p, p, p, p, p, p, p]
        L.ds_tail_stats.argtypes = [p, p, i64, i32, C.POINTER(i32), i32, p, p, p, sz, p]
        L.ds_tail_stats_static.argtypes = [p, p, i64, i32, C.POINTER(i32), i32, p, p, p]
        L.ds_tail_stats_static.restype = C.c_int
        L.ds_latency_stats.argtypes = [C.POINTER(DsTraces), p, i64, p, p, p, p, p, i32, p, C.POINTER(i32), i32, p, p, p, p, sz, p]
        L.ds_workspace_bytes.argtypes = [C.c_int, i64, i64]
        L.ds_workspace_bytes.restype = sz
        L.ds_device_status.argtypes = [p]
        L.ds_strerror.argtypes = [C.c_int]
        L.ds_strerror.restype = C.c_char_p
        L.ds_last_cuda_error.restype = C.c_char_p
        L.ds_launch_count.restype = i64
        for f in ("ds_characterize", "ds_simulate", "ds_simulate_est", "ds_simulate_budget", "ds_simulate_closed", "ds_estimation_error", "ds_queue_depth", "ds_latencies", "ds_tail_stats", "ds_latency_stats", "ds_device_status"):
            getattr(L, f).restype = C.c_int
        _lib = L
    return _lib


def check(fn, rc):
    if rc != DS_OK:
        L = lib()
        raise DsError(fn, rc, L.ds_strerror(rc).decode() + " " + L.ds_last_cuda_error().decode())
