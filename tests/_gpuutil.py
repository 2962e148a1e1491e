"""Test helpers for the CUDA path: upload a workload, run ds_* through the binding, bring results back."""
import numpy as np
import torch

import paper_2606_02982_b200 as ds
from paper_2606_02982_b200.api import instances_to_device

DEV = "cuda:0"


def gpu_characterize(text, offsets):
    t = torch.from_numpy(np.ascontiguousarray(text, np.uint8)).to(DEV)
    o = torch.from_numpy(np.ascontiguousarray(offsets, np.int64)).to(DEV)
    w, k = ds.characterize(t, o)
    assert ds.device_status() == 0
    return w.cpu().numpy(), k.cpu().numpy()


def upload(wl_obj):
    c = wl_obj
    d = {k: torch.from_numpy(np.ascontiguousarray(getattr(c, k))).to(DEV)
         for k in ("trace_off", "arrival", "tier", "words", "tokens", "out_len")}
    d["inst"] = instances_to_device(c.instances, DEV)
    d["out_off"] = torch.from_numpy(c.out_off).to(DEV)
    d["group"] = torch.from_numpy(c.group).to(DEV)
    d["t_mid"] = None if c.t_mid is None else torch.from_numpy(c.t_mid).to(DEV)
    return d


def gpu_simulate(c, d=None, traj_off=None):
    d = d or upload(c)
    n_total = int(c.out_off[-1])
    toff = traj = None
    if traj_off is not None:
        toff = torch.from_numpy(traj_off).to(DEV)
        traj = torch.zeros((int(traj_off[-1]), 3), dtype=torch.float64, device=DEV)
    st, dn, ema = ds.simulate(d["trace_off"], d["arrival"], d["tier"], d["words"], d["tokens"], d["out_len"], c.server,
                              d["inst"], d["out_off"], n_total, traj_off=toff, ema_traj=traj)
    status = ds.device_status()
    assert status == 0, status
    out = (st.cpu().numpy(), dn.cpu().numpy(), ema.cpu().numpy())
    return out + ((traj.cpu().numpy(),) if traj is not None else ())


def tiny_workload(wl, req, sv, combos):
    """One trace from rows [arrival, tier, words, tokens, out_len]; combos = [(policy, estimator, alpha)]."""
    req = np.asarray(req, np.int64).reshape(-1, 5)
    inst, grp = wl.make_instances(1, combos)
    return wl.Workload("tiny", 1, len(req), sv, np.array([0, len(req)], np.int64), req[:, 0].copy(),
                       req[:, 1].astype(np.uint8), req[:, 2].astype(np.int32), req[:, 3].astype(np.int32),
                       req[:, 4].astype(np.int32), inst, grp, len(combos))
