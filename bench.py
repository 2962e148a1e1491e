#!/usr/bin/env python
"""bench.py — whole-hot-path throughput of the B200-native DriftSched evaluation path.

Headline workload (N = 1): BASELINE.json:configs[3], the largest single-GPU configuration (heavy contention: 16 384 traces
x 10^4 requests x 5 policies x 4 EMA rates = 327 680 instances, 3.2768 G simulated requests, max batch 128, KV 65 536,
Pareto outputs, rho 0.95). A step = one pass of every SURVEY.md §8(a) row over it:
  ds_characterize (the materialised prompt text of the first --text-traces traces, 5.7 GB; SURVEY.md §8(d) draws the other
  traces' (W, P) numerically, their text would be 90 GB) -> ds_simulate (all instances) -> ds_latency_stats (fused
  latencies + p50/p99 per (policy, alpha) x tier and overall).
Extra legs at N = 1 (own keys, not the headline): the configs[1] step of round 1 (`step_configs1`), configs[4]
(`sim_configs4`: simulate with EMA trajectories + pre/post-drift percentiles) and the configs[2] 8 GiB scan (`scan_configs2`).
Prints ONE JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--traces T] [--legs cfg1,cfg4,cfg2]
"""
from __future__ import annotations

import argparse
import hashlib
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
K2_COUNTS = os.path.join(ROOT, "profiles", "r02_k2_counts.json.txt")     # ncu-counted instructions per simulated request (see its "how")
TRAFFIC = os.path.join(ROOT, "profiles", "r02_traffic.json.txt")         # ncu dram bytes per launch of the dominant kernels
SIM_CU = os.path.join(ROOT, "paper_2606_02982_b200", "csrc", "simulate.cu")


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


def build_cfg3(n_traces, text_traces, seed, characterize):
    from paper_2606_02982_b200 import workload as wl
    return wl.config3(characterize, n_traces=n_traces, seed=seed, text_traces=min(text_traces, n_traces))


def oracle_step(c, t0, t1):
    """The oracle, as it stands, over traces [t0, t1) of a trace workload (whole path: characterize the traces' text where
    it exists, simulate, latencies, percentiles). Returns (sim_requests, seconds)."""
    import oracle
    from paper_2606_02982_b200 import workload as wl
    nr = c.n_req
    rs = slice(t0 * nr, t1 * nr)
    inst, grp = wl.make_instances(t1 - t0, c.extra["combos"])
    trace_off = np.arange(t1 - t0 + 1, dtype=np.int64) * nr
    out_off = np.arange(len(inst) + 1, dtype=np.int64) * nr
    w, k = c.words[rs].copy(), c.tokens[rs].copy()
    tic = time.perf_counter()
    if c.offsets is not None:
        nt = min(t1, (len(c.offsets) - 1) // nr)               # traces whose prompts exist as text
        if nt > t0:
            lo, hi = c.offsets[t0 * nr], c.offsets[nt * nr]
            ww, kk = oracle.characterize(c.text[lo:hi], c.offsets[t0 * nr:nt * nr + 1] - lo)
            w[:len(ww)], k[:len(kk)] = ww, kk
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
    n_sample = min(args.traces, args.ref_traces)
    c = build_cfg3(n_sample, args.text_traces, rank_seed(0), oracle.characterize)
    for _ in range(min(args.warmup, 1)):
        oracle_step(c, 0, min(2, n_sample))
    tic = time.perf_counter()
    total = 0
    for _ in range(args.steps):
        n, _s = oracle_step(c, 0, n_sample)
        total += n
    el = time.perf_counter() - tic
    v = total / el
    sample = (f"first {n_sample} of {args.traces} traces of configs[3] ({n_sample * 20} instances, {n_sample * 200000} sim-requests, "
              f"whole path incl. the text of those traces) per step")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": workload_config(args.traces, min(args.text_traces, args.traces), None, note="bounded sample, CPU oracle, 1 core"),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def workload_config(n_traces, text_traces, c, note=None):
    cfg = {"workload": "configs[3] heavy contention: %d traces x 10000 requests x 5 policies x 4 EMA rates (split()+EMA), max_batch 128, "
                       "KV 65536, Pareto outputs, rho 0.95, aging 250 ms; whole hot path per step: ds_characterize over the materialised "
                       "prompt text of the first %d traces (the other traces' (W,P) are drawn numerically, SURVEY.md §8(d)) -> "
                       "ds_simulate -> ds_latency_stats" % (n_traces, text_traces),
           "l2": "inputs_exceed_l2 (%.2f GB of trace records + %.1f GB of text re-read every step)"
                 % (n_traces * 10000 * 21 / 1e9, c.text.size / 1e9 if c is not None and c.text is not None else 5.5 * text_traces / 1000.0),
           "per_rank": "own traces (seed 3 + 1000*rank)"}
    if c is not None:
        cfg.update({"instances": c.n_inst, "sim_requests_per_step": c.sim_requests,
                    "text_bytes": int(c.text.size) if c.text is not None else 0})
    if note:
        cfg["note"] = note
    return cfg


def pin_workload(c):
    """Move the per-step input arrays of a workload into pinned host memory ONCE and let the workload's numpy arrays be views
    of it: the end-to-end leg then copies from these very buffers (Tensor.pin_memory() of an already pinned array is the
    array itself), so a rank holds its 9.2 GB of inputs once instead of twice (8 ranks on one host: 75 GB, not 150 GB)."""
    import torch
    for f in ("text", "offsets", "arrival", "tier", "out_len", "words", "tokens"):
        a = getattr(c, f)
        if a is not None:
            setattr(c, f, torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy())


def max_over_ranks(ms, world, device):
    """Timing rule of the bench contract: the job's time is the slowest rank's (all_reduce MAX); identity at N=1."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def rank_seed(rank):
    """Weak scaling: rank r simulates its own traces of configs[3], generated with seed 3 + 1000 r (no data-path exchange)."""
    return 3 + 1000 * rank


def _json(path):
    try:
        return json.load(open(path))
    except Exception:
        return {}


def k2_roofline(kernel_key, n_sim, sim_ms, sm_max):
    """Issue-slot roofline of ds_simulate (plain ALU issue): peak = SMs x 4 schedulers x 1 warp-instruction per
    clock; achieved = (ncu-counted executed warp instructions per simulated request, from the committed capture) x requests
    / live kernel time. The capture names the simulate.cu it was taken from; when the source has changed since, the
    instruction count is stale and no fraction is printed. `algorithmic` puts the same time against the instruction floor
    DESIGN.md §6.2 derives for one request, which does not move with the kernel's own instruction count."""
    peak = 148 * 4 * sm_max * 1e6 / 1e9
    out = {"kernel": "simulate_kernel<%s>" % {"slots1": 1, "slots4": 4, "slots8": 8}[kernel_key], "bound": "alu", "achieved": None,
           "peak": peak, "unit": "Gwarp-inst/s", "frac": None, "traffic": None}
    tr = _json(TRAFFIC).get("simulate_" + kernel_key)
    if tr:   # dram read + write bytes of one launch of this size, from the ncu capture's bytes per simulated request
        out["traffic"] = tr["dram_bytes_per_simreq"] * n_sim
        out["traffic_source"] = "profiles/r02_traffic.json.txt: %.1f DRAM bytes per simulated request (ncu --set full, %s) x requests of this launch; algorithmic: 37 B (DESIGN.md §6.2)" % (
            tr["dram_bytes_per_simreq"], tr["per_launch_of"])
    cap = _json(K2_COUNTS)
    ent = cap.get(kernel_key)
    if not ent:
        out["reason"] = "no ncu capture of this instantiation in profiles/r02_k2_counts.json.txt"
        return out
    try:
        sha = hashlib.sha256(open(SIM_CU, "rb").read()).hexdigest()
    except OSError:
        sha = None
    out["capture"] = {"commit": cap.get("commit"), "simulate_cu_sha256": cap.get("simulate_cu_sha256"),
                      "ncu_issue_active_pct": ent.get("issue_active_pct"), "ncu_achieved_occupancy_pct": ent.get("achieved_occupancy_pct"),
                      "ncu_inst_per_simreq": ent.get("inst_per_simreq"), "file": "profiles/r02_k2_counts.json.txt"}
    floor = ent.get("floor_inst_per_simreq")
    if floor:
        fa = floor * n_sim / (sim_ms * 1e-3) / 1e9
        out["algorithmic"] = {"inst_per_simreq_floor": floor, "achieved": fa, "frac": fa / peak, "source": "DESIGN.md §6.2"}
    if sha is None or sha != cap.get("simulate_cu_sha256"):
        out["reason"] = "simulate.cu differs from the captured source: instruction count is stale, fraction withheld"
        return out
    ach = ent["inst_per_simreq"] * n_sim / (sim_ms * 1e-3) / 1e9
    out["achieved"], out["frac"] = ach, ach / peak
    out["note"] = "achieved = ncu-counted executed warp instructions per sim-request x sim-requests / live duration (issue-slot utilisation over the launch)"
    return out


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
    from paper_2606_02982_b200.pipeline import HotPath, HostPipeline

    # ---- setup (untimed): seeded inputs; W,P of the materialised text come from ds_characterize itself ----
    c = build_cfg3(args.traces, args.text_traces, rank_seed(rank), gpu_characterize_fn(dev))   # weak scaling: every rank its own traces
    pin_workload(c)
    hp = HotPath(c, dev)
    n_sim = c.sim_requests
    text_bytes = int(c.text.size) if c.text is not None else 0
    n_prompts = hp.n_text_prompts

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    warm = max(args.warmup, 3)
    for _ in range(warm):
        hp.step()
    st = ds.device_status()
    assert st == 0, f"device status {st}"
    sync_all()

    # ---- timed region: K steps, inputs resident in HBM (9 GB of inputs per step >> 126 MB L2) ----
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
    del hp
    torch.cuda.empty_cache()

    # ---- end to end through the public API with HOST buffers (pinned): every step copies its inputs (text, offsets, trace
    # records) H2D and its results (EMA factors, percentile tables, segment counts) D2H inside the timed region. The
    # per-request ticks (52 GB) stay in device memory; two input slots share one set of outputs, so the copy-in of step i+1
    # overlaps the kernels of step i ----
    e2e = None
    if not args.no_e2e:
        pipe = HostPipeline(c, dev, depth=2, share_outputs=True, result="stats")
        h_in = pipe.pin_inputs(c)
        h2d, d2h = pipe.h2d_bytes, pipe.d2h_bytes
        pipe.run(h_in, 2)
        sync_all()
        k2 = max(2, args.steps)
        e0.record()
        out = pipe.run(h_in, k2)
        e1.record()
        sync_all()
        assert bool((out[0] > 0).all()) and int(out[3].sum()) == 2 * n_sim          # factors came back; every request counted (tier + overall)
        e2e = {"value": world * n_sim * k2 / (max_over_ranks(e0.elapsed_time(e1), world, dev) * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": k2,
               "result": "EMA factors + p50/p99 tables + segment counts to pinned host memory; per-request ticks stay on the device"}
        del pipe, h_in, out
        torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, which, sm_max = _peaks()
    value = world * n_sim * args.steps / (ms_total * 1e-3)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": workload_config(args.traces, min(args.text_traces, args.traces), c),
        "stage_ms": {"characterize": float(char_ms), "simulate": float(sim_ms), "latencies+tail_stats": float(stat_ms)},
        "simulate_req_per_s": n_sim / (sim_ms * 1e-3),
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": int(launches),
        "roofline": k2_roofline("slots4", n_sim, sim_ms, sm_max),
    }
    if text_bytes:
        # K1 roofline: algorithmic bytes = text + 8 B offset + 8 B outputs per prompt
        k1_gbs = (text_bytes + 16 * n_prompts) / (char_ms * 1e-3) / 1e9
        line["characterization_gbs"] = k1_gbs
        line["roofline_scan"] = {"kernel": "characterize_kernel", "bound": "hbm", "achieved": k1_gbs, "peak": hbm_peak, "unit": "GB/s",
                                 "frac": k1_gbs / hbm_peak, "peak_source": which, "frac_of_8TBps": k1_gbs / 8000.0,
                                 "traffic": None, "workload": "text sample of the headline step"}
        tk = _json(TRAFFIC).get("characterize_kernel")
        if tk:
            line["roofline_scan"]["traffic"] = tk["dram_bytes_per_text_byte"] * text_bytes
            line["roofline_scan"]["traffic_source"] = "profiles/r02_traffic.json.txt: %.4f DRAM bytes per text byte (ncu --set full, %s)" % (
                tk["dram_bytes_per_text_byte"], tk["per_launch_of"])
    legs = [x for x in args.legs.split(",") if x] if world == 1 else []
    # CPU baseline first (it needs c): the oracle as it stands on a bounded sample (host cores of this box), rank 0, N=1 only
    if world == 1 and not args.no_cpu_baseline:
        ns = min(args.traces, args.cpu_traces)
        n, s = oracle_step(c, 0, ns)
        line["cpu_baseline"] = {"value": n / s, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"first {ns} of {args.traces} traces of configs[3] ({n} sim-requests, whole path incl. their text), {s:.1f} s",
                                "host_cores_available": os.cpu_count()}
    del c
    if "cfg1" in legs:
        line["step_configs1"] = step1_leg(dev, sm_max, hbm_peak)
    if "cfg4" in legs:
        line["sim_configs4"] = sim4_leg(dev, sm_max, n_traces=args.cfg4_traces)
    if "cfg2" in legs:
        line["scan_configs2"] = scan_leg(dev, args.scan_gib, hbm_peak)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def step1_leg(dev, sm_max, hbm_peak, reps=5):
    """configs[1] (round 1's headline step): 1024 traces x 2000 requests x 10 instances, text of every prompt materialised."""
    import torch
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import workload as wl
    from paper_2606_02982_b200.pipeline import HotPath
    c = wl.config1(gpu_characterize_fn(dev), n_traces=1024, n_req=2000, seed=1)
    hp = HotPath(c, dev)
    for _ in range(3):
        hp.step()
    assert ds.device_status() == 0
    ev = [hp.step(timed_events=True) for _ in range(reps)]
    torch.cuda.synchronize()
    ms = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(3)] for e in ev]).mean(axis=0)
    n_sim, tb, npmt = c.sim_requests, int(c.text.size), c.n_traces * c.n_req
    gbs = (tb + 16 * npmt) / (ms[0] * 1e-3) / 1e9
    return {"workload": "configs[1] policy sweep: 1024 traces x 2000 requests x 5 policies x 2 estimators, max_batch 32, KV 16384, rho 0.85",
            "sim_requests": n_sim, "ms_per_step": float(ms.sum()), "value": n_sim / (ms.sum() * 1e-3), "unit": UNIT,
            "stage_ms": {"characterize": float(ms[0]), "simulate": float(ms[1]), "latencies+tail_stats": float(ms[2])},
            "simulate_req_per_s": n_sim / (ms[1] * 1e-3), "characterization_gbs": gbs, "characterization_frac": gbs / hbm_peak,
            "roofline": k2_roofline("slots1", n_sim, ms[1], sm_max)}


def sim4_leg(dev, sm_max, reps=3, n_traces=4096):
    """configs[4]: 4096 traces x 50000 requests x 10 instances (2.048 G simulated requests), batch 256, EMA trajectories every
    1000 completions, pre/post-drift percentiles. Text-free: simulate + latency_stats."""
    import torch
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import workload as wl
    from paper_2606_02982_b200.pipeline import HotPath
    c = wl.config4(n_traces=n_traces)
    hp = HotPath(c, dev)
    for _ in range(2):
        hp.step()
    assert ds.device_status() == 0
    ev = [hp.step(timed_events=True) for _ in range(reps)]
    torch.cuda.synchronize()
    ms = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(3)] for e in ev]).mean(axis=0)
    n_sim = c.sim_requests
    return {"workload": "configs[4] runtime token drift: %d traces x 50000 requests x 5 policies x 2 estimators, max_batch 256, KV 131072, "
                        "rho 0.9, trajectories every 1000 completions, pre/post-drift p50/p99" % n_traces,
            "sim_requests": n_sim, "ms_per_step": float(ms[1] + ms[2]), "value": n_sim / ((ms[1] + ms[2]) * 1e-3), "unit": UNIT,
            "stage_ms": {"simulate": float(ms[1]), "latencies+tail_stats": float(ms[2])},
            "simulate_req_per_s": n_sim / (ms[1] * 1e-3), "roofline": k2_roofline("slots8", n_sim, ms[1], sm_max)}


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
    # CUDA events, best of >= 5 launches after warm-up, inputs resident; every launch has its own event pair
    # (8 GiB of input per call >> 126 MB L2, so no launch finds its input in cache). The mean is reported beside the best.
    reps = 7
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in evs:
        a.record()
        ds.characterize(t, o, w, k)
        b.record()
    torch.cuda.synchronize()
    times = [a.elapsed_time(b) for a, b in evs]
    ms, ms_mean = min(times), float(np.mean(times))
    nbytes = buf.size + 16 * n
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"workload": "configs[2] scan, %.2f GiB packed text" % gib, "bytes": int(buf.size), "prompts": int(n), "ms": ms, "ms_mean": ms_mean,
            "timing": "best of %d single launches (SURVEY.md 8(d)); mean beside it" % reps, "achieved_mean": nbytes / (ms_mean * 1e-3) / 1e9,
            "achieved": gbs, "unit": "GB/s", "frac": gbs / hbm_peak, "frac_of_8TBps": gbs / 8000.0,
            "algorithmic_bytes": int(nbytes)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--traces", type=int, default=16384, help="traces per GPU (configs[3] = 16384)")
    ap.add_argument("--text-traces", type=int, default=1024, help="traces of the headline workload whose prompts are materialised as text")
    ap.add_argument("--cpu-traces", type=int, default=128, help="traces in the bounded oracle sample of the cpu_baseline leg")
    ap.add_argument("--ref-traces", type=int, default=24, help="traces per step of --impl reference (bounded sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--legs", default="cfg1,cfg4,cfg2", help="extra legs at N=1: any of cfg1,cfg4,cfg2 (empty = none)")
    ap.add_argument("--cfg4-traces", type=int, default=4096, help="traces of the configs[4] leg (4096 = the full configuration)")
    ap.add_argument("--scan-gib", type=float, default=8.0, help="size of the configs[2] scan leg in GiB")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
