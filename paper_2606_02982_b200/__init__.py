"""B200-native DriftSched evaluation hot path (arxiv/paper_2606_02982): thin Python binding over the C ABI in
include/driftsched.h. Every step of the path runs in the CUDA kernels of libdriftsched.so; torch only provides
device memory and streams. See DESIGN.md."""
from .api import (characterize, device_status, estimation_error, latencies, latency_stats, launch_count, queue_depth,
                  simulate, simulate_budget, simulate_closed, simulate_est, simulate_workspace_bytes, tail_stats, tail_stats_static,
                  workspace_bytes)  # noqa: F401
from ._lib import DsError, LIB_PATH  # noqa: F401
