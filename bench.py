#!/usr/bin/env python
"""bench.py — whole-hot-path throughput of the B200-native DriftSched evaluation path.

A step = one pass of every SURVEY.md §8(a) row over BASELINE.json:configs[1] (policy sweep: 1024 traces x 2000
requests x 5 policies x 2 estimators = 10 240 instances, 20.48 M simulated requests, 1.13 GB of prompt text):
ds_characterize -> ds_simulate -> ds_latency_stats (fused latencies + percentiles).  Prints ONE JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--traces T]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "simulated requests/sec (policy x trace)"
UNIT = "req/s"
# The issue-slot roofline of ds_simulate uses the executed warp instructions per simulated request measured with ncu
# (paper_2606_02982_b200/k2_inst_per_simreq.txt, from profiles/r01_ncu_k2_v4.txt); DRAM traffic per launch comes from
# the same captures (profiles/r01_traffic.json.txt).


def _peaks():
    try:
        pk = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(pk["hbm_gbs"]), "measured", float(pk.get("sm_max_mhz", 1965.0))
    except Exception:
        return 6650.0, "fallback", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True).start()
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def build_workload(n_traces, seed, characterize):
    from paper_2606_02982_b200 import workload as wl
    return wl.config1(characterize, n_traces=n_traces, n_req=2000, seed=seed)


def gpu_characterize_fn(device):
    import torch
    import paper_2606_02982_b200 as ds

    def f(text, offsets):
        t = torch.from_numpy(text).to(device)
        o = torch.from_numpy(offsets).to(device)
        w, k = ds.characterize(t, o)
        torch.cuda.synchronize()
        return w.cpu().numpy(), k.cpu().numpy()
    return f


def oracle_step(c, sl):
    """The oracle, as it stands, over the traces in slice sl (whole path). Returns (sim_requests, seconds)."""
    import oracle
    from paper_2606_02982_b200 import workload as wl
    t0, t1 = sl
    nr = c.n_req
    lo, hi = c.offsets[t0 * nr], c.offsets[t1 * nr]
    text, off = c.text[lo:hi], c.offsets[t0 * nr:t1 * nr + 1] - lo
    rs = slice(t0 * nr, t1 * nr)
    inst, grp = wl.make_instances(t1 - t0, c.extra["combos"])
    trace_off = np.arange(t1 - t0 + 1, dtype=np.int64) * nr
    out_off = np.arange(len(inst) + 1, dtype=np.int64) * nr
    tic = time.perf_counter()
    w, k = oracle.characterize(text, off)
    st, dn, ema = oracle.simulate(trace_off, c.arrival[rs], c.tier[rs], w, k, c.out_len[rs], c.server, inst, out_off)
    e2e, qd, seg_t, seg_a = oracle.latencies(trace_off, c.arrival[rs], c.tier[rs], w, k, c.out_len[rs], inst, out_off, st, dn, grp)
    for vals in (e2e, qd):
        oracle.tail_stats(vals, seg_t, 3 * c.n_groups)
        oracle.tail_stats(vals, seg_a, c.n_groups)
    return len(inst) * nr, time.perf_counter() - tic


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    n_sample = min(args.traces, 64)
    c = build_workload(n_sample, 1, oracle.characterize)
    for _ in range(min(args.warmup, 1)):
        oracle_step(c, (0, min(4, n_sample)))
    tic = time.perf_counter()
    total = 0
    for _ in range(args.steps):
        n, _s = oracle_step(c, (0, n_sample))
        total += n
    el = time.perf_counter() - tic
    v = total / el
    sample = f"{n_sample} of {args.traces} traces of configs[1] ({n_sample * 10} instances, {n_sample * 20000} sim-requests) per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": "configs[1] policy sweep (bounded sample, CPU oracle)", "traces": args.traces, "requests_per_trace": 2000},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def max_over_ranks(ms, world, device):
    """Timing rule of the bench contract: the job's time is the slowest rank's (all_reduce MAX); identity at N=1."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def rank_seed(rank):
    """Weak scaling: rank r simulates its own 1024 traces, generated with seed 1+r (no data-path exchange)."""
    return 1 + rank


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200.pipeline import HotPath

    # ---- setup (untimed): seeded inputs; W,P of the generated text come from ds_characterize itself ----
    c = build_workload(args.traces, rank_seed(rank), gpu_characterize_fn(dev))   # weak scaling: every rank its own traces
    hp = HotPath(c, dev)
    n_sim = c.sim_requests
    text_bytes = int(c.text.size)
    n_prompts = c.n_traces * c.n_req

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        hp.step()
    st = ds.device_status()
    assert st == 0, f"device status {st}"
    sync_all()

    # ---- timed region: K steps, inputs resident in HBM (1.13 GB of text per step >> 126 MB L2) ----
    sampler = ClockSampler(local)
    sampler.start()
    l0 = ds.launch_count()
    sync_all()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    stage_ev = []
    e0.record()
    for _ in range(args.steps):
        stage_ev.append(hp.step(timed_events=True))
    e1.record()
    sync_all()
    launches = ds.launch_count() - l0
    clocks = sampler.stop()
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    st_ms = np.array([[ev[i].elapsed_time(ev[i + 1]) for i in range(3)] for ev in stage_ev])   # characterize, simulate, stats
    char_ms, sim_ms, stat_ms = st_ms.mean(axis=0)

    # ---- end to end through the public API with HOST buffers (pinned): every step copies its inputs H2D and its outputs
    # D2H inside the timed region; pipeline.HostPipeline overlaps copy-in, kernels and copy-out of neighbouring steps ----
    from paper_2606_02982_b200.pipeline import HostPipeline
    del hp
    torch.cuda.empty_cache()
    pipe = HostPipeline(c, dev, depth=2)
    h_in = pipe.pin_inputs(c)
    h2d, d2h = pipe.h2d_bytes, pipe.d2h_bytes
    pipe.run(h_in, 2)
    sync_all()
    k2 = max(2, args.steps)
    e0.record()
    out = pipe.run(h_in, k2)
    e1.record()
    sync_all()
    assert int(out[0].numel()) == n_sim and bool((out[1][:1000] > out[0][:1000]).all())     # done > start came back
    e2e_val = world * n_sim * k2 / (max_over_ranks(e0.elapsed_time(e1), world, dev) * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, which, sm_max = _peaks()
    value = world * n_sim * args.steps / (ms_total * 1e-3)
    # K1 roofline: algorithmic bytes = text + 8 B offset + 8 B outputs per prompt
    k1_bytes = text_bytes + 16 * n_prompts
    k1_gbs = k1_bytes / (char_ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": "configs[1] policy sweep: %d traces x 2000 requests x 5 policies x 2 estimators, max_batch 32, "
                               "KV 16384, rho 0.85" % args.traces, "instances": c.n_inst, "sim_requests_per_step": n_sim,
                   "text_bytes": text_bytes, "l2": "inputs_exceed_l2 (text re-read every step)", "per_rank": "own traces (seed 1+rank)"},
        "stage_ms": {"characterize": float(char_ms), "simulate": float(sim_ms), "latencies+tail_stats": float(stat_ms)},
        "characterization_gbs": k1_gbs,
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": k2},
        "gpu_launches": int(launches),
        "roofline_scan": {"kernel": "characterize_kernel", "bound": "hbm", "achieved": k1_gbs, "peak": hbm_peak, "unit": "GB/s",
                          "frac": k1_gbs / hbm_peak, "peak_source": which, "frac_of_8TBps": k1_gbs / 8000.0, "traffic": None},
    }
    line["roofline_scan"]["traffic"] = _traffic().get("characterize_kernel")
    if world == 1 and args.scan_gib > 0:
        line["scan_configs2"] = scan_leg(dev, args.scan_gib, hbm_peak)
    # K2 roofline (dominant kernel): plain-ALU issue slots. peak = 148 SMs x 4 schedulers x 1 warp-inst/clk x max SM clock.
    ipr = _k2_inst_per_simreq()
    issue_peak = 148 * 4 * sm_max * 1e6 / 1e9
    if ipr is not None:
        ach = ipr * n_sim / (sim_ms * 1e-3) / 1e9
        line["roofline"] = {"kernel": "simulate_kernel<1>", "bound": "alu", "achieved": ach, "peak": issue_peak,
                            "unit": "Gwarp-inst/s", "frac": ach / issue_peak, "traffic": _traffic().get("simulate_kernel"),
                            "note": "achieved = ncu-counted executed warp instructions per sim-request x sim-requests / live duration"}
        alu = _k2_inst_per_simreq(1)
        if alu is not None:
            # DESIGN.md §6.1/§6.2: measured on this GPU, an ALU-pipe instruction (16 lanes/clk per scheduler) holds the issue
            # port for two cycles, everything else for one: issue cycles per request = instructions + ALU instructions.
            cyc = (ipr + alu) * n_sim / (sim_ms * 1e-3) / 1e9
            line["roofline"]["issue_cycles"] = {"achieved": cyc, "peak": issue_peak, "unit": "Gcycle/s", "frac": cyc / issue_peak,
                                                "alu_inst_per_request": alu}
    else:
        line["roofline"] = {"kernel": "simulate_kernel<1>", "bound": "alu", "achieved": None, "peak": issue_peak,
                            "unit": "Gwarp-inst/s", "frac": None, "traffic": None}
    # CPU baseline: the oracle as it stands on a bounded sample (host cores of this box), rank 0, N=1 only
    if world == 1 and not args.no_cpu_baseline:
        ns = min(args.traces, args.cpu_traces)
        n, s = oracle_step(c, (0, ns))
        line["cpu_baseline"] = {"value": n / s, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"first {ns} of {args.traces} traces ({n} sim-requests, whole path), {s:.1f} s",
                                "host_cores_available": os.cpu_count()}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def _traffic():
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "r01_traffic.json.txt")))
    except Exception:
        return {}


def scan_leg(dev, gib, hbm_peak):
    """configs[2]: characterization-only scan of `gib` GiB of packed text (8 GiB = the full configuration)."""
    import torch
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import workload as wl
    buf, off = wl.config2(int(gib * (1 << 30)))
    t = torch.from_numpy(buf).to(dev)
    o = torch.from_numpy(off).to(dev)
    n = len(off) - 1
    w = torch.empty(n, dtype=torch.int32, device=dev)
    k = torch.empty_like(w)
    for _ in range(3):
        ds.characterize(t, o, w, k)
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    reps = 5
    e0.record()
    for _ in range(reps):
        ds.characterize(t, o, w, k)                      # 8 GiB of input per call >> 126 MB L2
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    nbytes = buf.size + 16 * n
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"workload": "configs[2] scan, %.2f GiB packed text" % gib, "bytes": int(buf.size), "prompts": int(n), "ms": ms,
            "achieved": gbs, "unit": "GB/s", "frac": gbs / hbm_peak, "frac_of_8TBps": gbs / 8000.0,
            "algorithmic_bytes": int(nbytes)}


def _k2_inst_per_simreq(col=0):
    """col 0: executed warp instructions per simulated request; col 1: those of them on the ALU pipe (ncu SASS counts)."""
    p = os.path.join(ROOT, "paper_2606_02982_b200", "k2_inst_per_simreq.txt")
    try:
        return float(open(p).read().split()[col])
    except Exception:
        return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--traces", type=int, default=1024, help="traces per GPU (configs[1] = 1024)")
    ap.add_argument("--cpu-traces", type=int, default=1024, help="traces in the bounded oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scan-gib", type=float, default=8.0, help="size of the configs[2] scan leg in GiB (0 = skip)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
