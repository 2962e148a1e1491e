"""Test helpers: build tiny traces and run them through the oracle (tests only)."""
import numpy as np

import oracle
from paper_2606_02982_b200 import workload as wl


def server(**kw):
    return wl.Server(**{**dict(max_batch=1, kv_budget=0), **kw})


def run_oracle(req, sv, policy, estimator=wl.EXACT, alpha=0.0, want_traj=False, want_est=False):
    """req: rows [arrival, tier, words, tokens, out_len]. One trace, one instance."""
    req = np.asarray(req, np.int64).reshape(-1, 5)
    inst = np.zeros(1, wl.INSTANCE_DTYPE)
    inst[0] = (0, policy, estimator, 0, alpha)
    return oracle.simulate([0, len(req)], req[:, 0], req[:, 1], req[:, 2], req[:, 3], req[:, 4], sv, inst,
                           want_traj=want_traj, want_est=want_est)


def service_time(P, O, sv):
    """closed form (i): max_batch=1 service time of one request."""
    return O * (sv.c_base + sv.c_batch) + sv.c_ctx * (O * P + O * (O - 1) // 2) + sv.c_prefill * P
