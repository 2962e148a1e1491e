"""One pass of the whole hot path over a resident workload:
ds_characterize -> ds_simulate -> ds_latency_stats (fused; or ds_latencies -> 4 x ds_tail_stats with fused=False). Orchestration and buffer ownership only;
every computation happens inside libdriftsched.so."""
from __future__ import annotations

import numpy as np
import torch

from . import _lib, api


class HotPath:
    """Device-resident buffers for one workload (see workload.Workload) and the step that runs the path."""

    def __init__(self, wl_obj, device="cuda:0", pct=(50, 99), fused=True, share=None):
        """share: another HotPath of the same workload whose OUTPUT buffers and workspaces this one reuses (only the
        inputs are private): the slots of a HostPipeline whose outputs do not fit twice (configs[3]: 98 GB)."""
        c = wl_obj
        self.c = c
        self.dev = torch.device(device)
        self.pct = tuple(pct)
        self.fused = fused
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(self.dev)
        self.text = up(c.text) if c.text is not None else None
        self.offsets = up(c.offsets) if c.offsets is not None else None
        self.trace_off = up(c.trace_off)
        self.arrival = up(c.arrival)
        self.tier = up(c.tier)
        self.out_len = up(c.out_len)
        self.words = up(c.words)     # overwritten by ds_characterize every step when text is present
        self.tokens = up(c.tokens)
        self.inst = api.instances_to_device(c.instances, self.dev)
        self.out_off = up(c.out_off)
        self.group = up(c.group)
        self.t_mid = up(c.t_mid) if c.t_mid is not None else None
        self.n_total = int(c.out_off[-1])
        self.n_inst = c.n_inst
        self.n_groups = c.n_groups * (2 if c.t_mid is not None else 1)
        n, dev = self.n_total, self.dev
        self.n_text_prompts = 0 if self.offsets is None else self.offsets.numel() - 1   # (a text sample may cover fewer prompts)
        if share is not None:
            for k in ("start", "done", "ema_final", "traj_off", "ema_traj", "ws_char", "ws_sim", "ws_tail", "e2e_stats", "qd_stats",
                      "counts4", "stats", "counts", "e2e", "qdelay", "seg_tier", "seg_all"):
                setattr(self, k, getattr(share, k))
            return
        self.start = torch.empty(n, dtype=torch.int64, device=dev)
        self.done = torch.empty(n, dtype=torch.int64, device=dev)
        self.ema_final = torch.empty((self.n_inst, 3), dtype=torch.float64, device=dev)
        self.traj_off = self.ema_traj = None
        if c.server.traj_every > 0:
            k = (np.diff(c.trace_off)[c.instances["trace"]] // c.server.traj_every).astype(np.int64)
            toff = np.concatenate([[0], np.cumsum(k)]).astype(np.int64)
            self.traj_off = up(toff)
            self.ema_traj = torch.zeros((int(toff[-1]), 3), dtype=torch.float64, device=dev)
        ws = lambda which, a, b: torch.empty(api.workspace_bytes(which, a, b), dtype=torch.uint8, device=dev)
        self.ws_char = ws(_lib.WS_CHARACTERIZE, 0 if self.text is None else self.text.numel(), self.n_text_prompts)
        self.ws_sim = torch.empty(api.simulate_workspace_bytes(n, self.n_inst, self.arrival.numel()), dtype=torch.uint8, device=dev)
        G = self.n_groups
        # histograms, and for the fused call the staging area behind them (5 bytes per simulated request: 32-bit keys + segment codes)
        nb = api.workspace_bytes(_lib.WS_TAIL_STATS, 4 * G, len(self.pct))
        if fused:
            nb += api.workspace_bytes(_lib.WS_LATENCY_STAGE, n, 0)
        self.ws_tail = torch.empty(nb, dtype=torch.uint8, device=dev)
        # percentiles: rows [0,3G) = (group, tier) segments, rows [3G,4G) = per-group overall (ds_latency_stats layout)
        self.e2e_stats = torch.empty((4 * G, len(self.pct)), dtype=torch.int64, device=dev)
        self.qd_stats = torch.empty((4 * G, len(self.pct)), dtype=torch.int64, device=dev)
        self.counts4 = torch.empty(4 * G, dtype=torch.int64, device=dev)
        self.stats = {"e2e_tier": self.e2e_stats[:3 * G], "e2e_all": self.e2e_stats[3 * G:],
                      "qdelay_tier": self.qd_stats[:3 * G], "qdelay_all": self.qd_stats[3 * G:]}
        if fused:
            self.counts = {"e2e_tier": self.counts4[:3 * G], "e2e_all": self.counts4[3 * G:],
                           "qdelay_tier": self.counts4[:3 * G], "qdelay_all": self.counts4[3 * G:]}
            self.e2e = self.qdelay = self.seg_tier = self.seg_all = None
        else:
            self.counts = {k: torch.empty(v.shape[0], dtype=torch.int64, device=dev) for k, v in self.stats.items()}
            self.e2e = torch.empty(n, dtype=torch.int64, device=dev)
            self.qdelay = torch.empty(n, dtype=torch.int64, device=dev)
            self.seg_tier = torch.empty(n, dtype=torch.int32, device=dev)
            self.seg_all = torch.empty(n, dtype=torch.int32, device=dev)

    def step(self, timed_events=False):
        """Run the path once on the current stream. With timed_events, returns CUDA events bracketing each stage."""
        ev = []
        mark = (lambda: ev.append(self._rec())) if timed_events else (lambda: None)
        mark()
        if self.text is not None:
            k = self.n_text_prompts       # the prompts that exist as text (all of them, or the materialised sample)
            api.characterize(self.text, self.offsets, self.words[:k], self.tokens[:k], self.ws_char)
        mark()
        api.simulate(self.trace_off, self.arrival, self.tier, self.words, self.tokens, self.out_len, self.c.server, self.inst,
                     self.out_off, self.n_total, self.start, self.done, self.ema_final, self.traj_off, self.ema_traj, self.ws_sim)
        mark()
        if self.fused:
            api.latency_stats(self.trace_off, self.arrival, self.tier, self.words, self.tokens, self.out_len, self.inst,
                              self.out_off, self.start, self.done, self.group, self.c.n_groups, self.t_mid, self.pct,
                              self.e2e_stats, self.qd_stats, self.counts4, self.ws_tail)
        else:
            e2e, qd, seg_t, seg_a = api.latencies(self.trace_off, self.arrival, self.tier, self.words, self.tokens, self.out_len,
                                                  self.inst, self.out_off, self.n_total, self.start, self.done, self.group,
                                                  self.t_mid, out=(self.e2e, self.qdelay, self.seg_tier, self.seg_all))
            for name, vals, seg in (("e2e_tier", e2e, seg_t), ("e2e_all", e2e, seg_a), ("qdelay_tier", qd, seg_t),
                                    ("qdelay_all", qd, seg_a)):
                api.tail_stats(vals, seg, self.stats[name].shape[0], self.pct, self.stats[name], self.counts[name], self.ws_tail)
        mark()
        return ev

    @staticmethod
    def _rec():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e


class HostPipeline:
    """End-to-end path for HOST inputs and outputs: `depth` HotPath slots and three CUDA streams, so the host-to-device
    copy of step i+1, the kernels of step i and the device-to-host copy of step i-1 overlap (PCIe is the slowest of the
    three on configs[1]). Orchestration only: every computation still happens inside libdriftsched.so.

    result="ticks": every step returns start/done ticks of every simulated request, the EMA factors and the percentile
    tables; result="stats": only the factors, percentile tables and segment counts come back (the per-request ticks stay in
    device memory: 52 GB on configs[3]). share_outputs: the slots have private inputs but share one set of output
    buffers and workspaces (for workloads whose outputs do not fit twice); a step then starts only after the previous
    step's results have left the device."""

    def __init__(self, wl_obj, device="cuda:0", depth=2, share_outputs=False, result="ticks"):
        self.dev = torch.device(device)
        first = HotPath(wl_obj, device)
        self.slots = [first] + [HotPath(wl_obj, device, share=first if share_outputs else None) for _ in range(depth - 1)]
        self.share = share_outputs
        self.s_in, self.s_run, self.s_out = (torch.cuda.Stream(self.dev) for _ in range(3))
        mk = lambda: [torch.cuda.Event() for _ in range(depth)]
        self.ev_in, self.ev_run, self.ev_out = mk(), mk(), mk()
        ticks = (lambda hp: [hp.start, hp.done]) if result == "ticks" else (lambda hp: [])
        self.out_dev = [ticks(hp) + [hp.ema_final, hp.e2e_stats, hp.qd_stats, hp.counts4] for hp in self.slots]
        self.out_host = [[torch.empty(t.shape, dtype=t.dtype).pin_memory() for t in outs] for outs in self.out_dev]
        self.h2d_bytes = 0
        self.d2h_bytes = sum(t.numel() * t.element_size() for t in self.out_host[0])
        # per-step inputs: the text and the trace records; (words, tokens) too when the text does not cover every prompt
        self.in_fields = ("text", "offsets", "arrival", "tier", "out_len")
        if first.text is None or first.n_text_prompts < first.words.numel():
            self.in_fields += ("words", "tokens")

    def pin_inputs(self, wl_obj):
        """Pinned host copies of the per-step inputs (what a caller would hand over)."""
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h = {f: pin(getattr(wl_obj, f)) for f in self.in_fields if getattr(wl_obj, f) is not None}
        self.h2d_bytes = sum(t.numel() * t.element_size() for t in h.values())
        return h

    def run(self, host_inputs, n_steps):
        """n_steps passes of the hot path, each with its inputs copied from `host_inputs` and its outputs copied to
        pinned host memory. Returns the host output tensors of the last step. Synchronises at the end."""
        cur = torch.cuda.current_stream(self.dev)
        start = torch.cuda.Event()
        start.record(cur)
        for s in (self.s_in, self.s_run, self.s_out):
            s.wait_event(start)
        depth = len(self.slots)
        for i in range(n_steps):
            k = i % depth
            hp = self.slots[k]
            if i >= depth:
                self.s_in.wait_event(self.ev_run[k])      # the kernels that last read this slot's inputs are done
                self.s_run.wait_event(self.ev_out[k])     # and its outputs have left the device
            if self.share and i >= 1:
                self.s_run.wait_event(self.ev_out[(i - 1) % depth])   # shared outputs: the previous step's results are out
            with torch.cuda.stream(self.s_in):
                for f, h in host_inputs.items():
                    getattr(hp, f).copy_(h, non_blocking=True)
                self.ev_in[k].record(self.s_in)
            self.s_run.wait_event(self.ev_in[k])
            with torch.cuda.stream(self.s_run):
                hp.step()
                self.ev_run[k].record(self.s_run)
            self.s_out.wait_event(self.ev_run[k])
            with torch.cuda.stream(self.s_out):
                for h, d in zip(self.out_host[k], self.out_dev[k]):
                    h.copy_(d, non_blocking=True)
                self.ev_out[k].record(self.s_out)
        for s in (self.s_in, self.s_run, self.s_out):
            done = torch.cuda.Event()
            done.record(s)
            cur.wait_event(done)
        return self.out_host[(n_steps - 1) % depth]
