#!/usr/bin/env python
"""bench.py -- paged decode-attention KV GB/s on one B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (translation + split-KV partial attention + LSE
combine, all inside one persistent launch) over one synthetic batch: one
cp_decode_attention call.  Default workload: BASELINE.json configs[1], the shared pool of
4 cold GQA models (344 MB of KV per step = 2.7 x the 126 MB L2): K steps back to back inside one
CUDA-event pair; the same steps with a read-only L2 flush before each are reported beside it, and the
other four BASELINE configs go through the same protocol in the `per_config` block (class StepTimer).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]
                    [--probe timeline|stream|launch]

Prints ONE JSON line (see DESIGN.md 7 for every field).  N > 1 = independent replicas
(the path does not shard: BASELINE north_star fixes one GPU).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the decode kernel, from the committed `ncu --set full`
# captures profiles/r2_ncu_full_cfg{2,3,4,5}.txt (cfg1, 0.66 MB, has no capture: its launch is latency, not traffic)
NCU_TRAFFIC_BYTES = {2: 344.68e6 + 7.64e6, 3: 293.21e6 + 16.84e6, 4: 135.82e6 + 7.35e6, 5: 806.45e6 + 7.51e6}
NCU_TENSOR_PIPE_PCT = {3: 47.0}       # sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active

METRIC = "paged decode-attention KV GB/s"
UNIT = "GB/s"
L2_BYTES = 126 * 1024 * 1024


def reduce_max_over_ranks(x: float, device="cpu") -> float:
    """Max over ranks of a per-rank time (the contract: time on the device, take the MAX)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(bytes_per_rank: int, world: int, step_ms: float) -> float:
    """Replicas only: every rank processes its own copy of the batch; the
    whole-job throughput is the bytes of all ranks over the slowest rank's step time."""
    return world * bytes_per_rank / (step_ms * 1e-3) / 1e9


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d.get("bf16_tflops", 1590.0)),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", 1400.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def workload_desc(w, k):
    return {"workload": "cfg%d:%s" % (k, w.name), "requests": len(w.requests),
            "tokens": w.total_tokens(), "page_tokens": w.page_tokens,
            "kv_bytes_per_step": w.algorithmic_bytes(), "flops_per_step": w.flops(),
            "l2": ("inputs %.0f MB > 2 x L2 (126 MB): K steps back to back, no flush; the flushed number is reported beside it"
                   % (w.algorithmic_bytes() / 1e6)) if w.algorithmic_bytes() > 2 * L2_BYTES else
                  "L2 flushed before every timed step (read-only pass over 512 MB, outside the step's event pair)"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed regions run."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            import shutil
            cmd = ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                   "--format=csv,noheader,nounits", "-lms", "5"]
            if shutil.which("stdbuf"):
                cmd = ["stdbuf", "-oL"] + cmd          # line-buffered: samples arrive while we run
            self.proc = subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        self.t.join(timeout=2)
        # nvidia-smi's own timestamp decides whether a sample lies in the window (its stdout reaches
        # us through a pipe in bursts, so the arrival time says little)
        import datetime
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        parsed = []
        for _, r in self.rows:
            f = [x.strip() for x in r.split(",")]
            try:
                ts = datetime.datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                parsed.append((ts, float(f[1]), float(f[2]), f[4:8]))
            except Exception:
                continue
        inside = [x for x in parsed if t0 - 0.05 <= x[0] <= t1 + 0.05] or parsed
        for _, a, b, fl in inside:
            sm.append(a); mx.append(b)
            for n, v in zip(names, fl):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample_plan(w, budget_s: float):
    """Pick a bounded sample of (request, head) pairs for the CPU oracle: every request, an
    evenly spaced subset of heads, sized from a quick calibration so one pass costs about
    budget_s.  Returns (heads_per_request, fraction_of_heads)."""
    import oracle
    r = min(range(len(w.requests)), key=lambda i: w.requests[i].context_len)
    m = w.models[w.requests[r].model_id]
    t = time.perf_counter()
    oracle.decode_workload(w, request_indices=[r], heads_per_request=[[0]])
    dt = max(time.perf_counter() - t, 1e-4)
    per_head_token = dt / w.requests[r].context_len / ((m.head_dim_qk + m.head_dim_v) / 256.0)
    cores = oracle.num_threads()
    full = sum(w.requests[i].context_len * w.models[w.requests[i].model_id].n_q_heads *
               (w.models[w.requests[i].model_id].head_dim_qk + w.models[w.requests[i].model_id].head_dim_v) / 256.0
               for i in range(len(w.requests))) * per_head_token / cores
    frac = min(1.0, budget_s / max(full, 1e-9))
    heads, used, total = [], 0, 0
    for rq in w.requests:
        hq = w.models[rq.model_id].n_q_heads
        n = max(1, int(round(hq * frac)))
        hs = sorted(set(int(x) for x in np.linspace(0, hq - 1, n)))
        heads.append(hs)
        used += len(hs) * rq.context_len
        total += hq * rq.context_len
    return heads, used / total


def run_reference(args, w, k):
    """--impl reference: the CPU oracle, as it stands, timed on the host cores."""
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    budget = min(1.5, 150.0 / max(1, args.steps + args.warmup))
    heads, frac = oracle_sample_plan(w, budget)
    for _ in range(args.warmup):
        oracle.decode_workload(w, heads_per_request=heads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.decode_workload(w, heads_per_request=heads)
    dt = time.perf_counter() - t0
    value = frac * w.algorithmic_bytes() * args.steps / dt / 1e9
    sample = "every request, %.1f%% of the (head, token) pairs (evenly spaced heads) per step" % (100 * frac)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps / frac,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_desc(w, k),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "note": "ms_per_step is extrapolated to the full step from the sampled fraction"}
    print(json.dumps(line))


class StepTimer:
    """Timing protocol of one workload.  All numbers come from CUDA events on the launching stream.

    region      K steps back to back inside ONE event pair: the contract's number.  Legitimate as an HBM
                measurement only when a step's inputs exceed the L2 (126 MB) several times over, so that nothing
                of step i is left when step i + 1 asks for it (cfg2, cfg3, cfg5).
    flushed     every step bracketed by its own event pair, a read-only pass over 512 MB (clean lines only: a
                write would leave dirty lines the timed kernel has to evict) and a short device-side spin
                before it; p10 / p50 / p90, p50 is "the" flushed number.  The number for inputs near or below
                the L2 size (cfg1, cfg4); reported for every config.  An event pair around an EMPTY kernel
                already reads ~6 us on this box and a kernel boundary inside a region ~2 us (both measured
                beside it: empty_kernel_events_us, empty_kernel_region_us), so a flushed number carries ~4 us that a
                region number does not; flushed_calibrated_us subtracts that difference and is reported
                only as a reading aid.
    device      %globaltimer stamps written by the kernel itself (CP_OPT_TIMELINE): first CTA entry to last
                CTA exit of flushed steps; where the launch and event overheads are not.
    """

    def __init__(self, torch, cp, dev, stream):
        self.torch, self.cp, self.dev, self.stream = torch, cp, dev, stream
        self.flush_buf = torch.zeros(512 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)
        self.flush_sink = torch.zeros((), dtype=torch.float32, device=dev)
        self.stamp = torch.zeros(2, dtype=torch.int64, device=dev)
        self.event_overhead_us = 0.0      # empty_kernel_events_us - empty_kernel_region_us, set by the caller

    def l2_flush(self):
        self.torch.sum(self.flush_buf, dim=(0,), out=self.flush_sink)

    def _region(self, steps, fn):
        torch = self.torch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        torch.cuda._sleep(4000000)          # ~2 ms: the host enqueues the whole region behind a device-side spin
        e0.record()
        for i in range(steps):
            fn(i)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps  # ms per step

    def region(self, steps, step_fn):
        return self._region(steps, lambda i: step_fn())

    def per_step(self, steps, step_fn):
        torch = self.torch
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps)]
        torch.cuda.synchronize()
        for i in range(steps):
            self.l2_flush()
            torch.cuda._sleep(100000)       # ~50 us: keeps the host a step ahead
            ev[2 * i].record()
            step_fn()
            ev[2 * i + 1].record()
        torch.cuda.synchronize()
        return [ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(steps)]

    def empty_kernel_events_us(self, reps=20):
        """What an event pair around a one-thread kernel reads: the floor of every per-step number."""
        return 1e3 * float(np.median(self.per_step(reps, lambda: self.cp.probe_globaltimer(self.stamp, self.stream))))

    def empty_kernel_region_us(self, reps=50):
        """Back-to-back one-thread kernels inside one event pair: what a kernel boundary costs."""
        return 1e3 * self.region(reps, lambda: self.cp.probe_globaltimer(self.stamp, self.stream))


TL = {"entry": 0, "after_sync": 14, "sched_has_rec": 15, "producer_has_meta": 1, "first_tma": 9, "first_slice_landed": 2, "last_page_issued": 3, "last_slice_landed": 10,
      "softmax_done": 4, "published": 5, "poll_ok": 12, "partials_loaded": 13, "combine_done": 7}


def device_timeline(timer, dw, cp, reps=5):
    """Per-CTA %globaltimer stamps of flushed steps of the tcgen05 K/V kernel (cp_pool_read_timeline): kernel
    duration on the device and where it goes, as [min, median, max] over the CTAs, us after the first CTA's entry."""
    torch = timer.torch
    dw.pool.set_option(cp.CP_OPT_TIMELINE, 1)
    dur, phases = [], {k: [] for k in TL}
    try:
        for _ in range(reps):
            timer.l2_flush()
            torch.cuda._sleep(100000)
            dw.decode()
            torch.cuda.synchronize()
            t = dw.pool.read_timeline().astype(np.int64)
            t = t[t[:, 0] > 0]
            if t.size == 0 or t[:, 7].max() == 0:
                return None                 # a kernel that does not stamp
            t0 = t[:, 0].min()
            dur.append((t[:, 7].max() - t0) / 1e3)
            for name, slot in TL.items():
                col = t[:, slot][t[:, slot] > 0]
                if col.size:
                    phases[name].append([(col.min() - t0) / 1e3, (float(np.median(col)) - t0) / 1e3, (col.max() - t0) / 1e3])
    finally:
        dw.pool.set_option(cp.CP_OPT_TIMELINE, 0)
    return {"kernel_us": float(np.median(dur)), "reps": reps,
            "phases_us_min_med_max_over_ctas": {k: [round(float(x), 2) for x in np.median(np.array(v), axis=0)] for k, v in phases.items() if v},
            "note": "first CTA entry to last CTA's combine done; stamps taken right after a barrier show the arrival"}


def parity_sample(w, got, budget_s=1.5):
    """Achieved error of this run's outputs against the CPU oracle on a bounded sample of (request, head) pairs."""
    import oracle
    heads, frac = oracle_sample_plan(w, budget_s)
    ref = oracle.decode_workload(w, heads_per_request=heads)
    worst = {"max_abs": 0.0, "rel_fro": 0.0, "lse_abs": 0.0}
    for (o, l), (ro, rl), hs in zip(got, ref, heads):
        o, l = o[hs].astype(np.float64), l[hs].astype(np.float64)
        worst["max_abs"] = max(worst["max_abs"], float(np.abs(o - ro).max()))
        worst["rel_fro"] = max(worst["rel_fro"], float(np.linalg.norm(o - ro) / np.linalg.norm(ro)))
        worst["lse_abs"] = max(worst["lse_abs"], float(np.abs(l - rl).max()))
    worst["sample"] = "%.1f%% of the (head, token) pairs, every request" % (100 * frac)
    return worst


def measure_config(timer, cp, k, w, dw, steps, peaks, with_parity=True):
    """One workload through the whole protocol; returns the per_config entry."""
    abytes = w.algorithmic_bytes()
    dw.ensure_workspace()
    for _ in range(5):
        dw.decode()
    region_ms = min(timer.region(steps, dw.decode) for _ in range(2))
    ps = timer.per_step(max(steps // 2, 20), dw.decode)
    flushed_ms = float(np.median(ps))
    big = abytes > 2 * L2_BYTES
    used_ms = region_ms if big else flushed_ms
    achieved = abytes / (used_ms * 1e-3) / 1e9
    entry = {"workload": "cfg%d:%s" % (k, w.name), "kv_bytes_per_step": abytes,
             "region_us": 1e3 * region_ms, "flushed_us": 1e3 * flushed_ms,
             "flushed_us_p10_p50_p90": [1e3 * float(x) for x in np.percentile(ps, [10, 50, 90])],
             "flushed_calibrated_us": 1e3 * flushed_ms - timer.event_overhead_us,
             "roofline_uses": "region (inputs %.0f MB > 2 x L2)" % (abytes / 1e6) if big else "flushed (inputs %.0f MB fit or nearly fit the 126 MB L2)" % (abytes / 1e6),
             "kernel_us": 1e3 * used_ms, "gbs": achieved, "frac_of_measured_peak": achieved / peaks["hbm_gbs"],
             "frac_of_nominal_8000": achieved / 8000.0, "flushed_gbs": abytes / (flushed_ms * 1e-3) / 1e9,
             "traffic": NCU_TRAFFIC_BYTES.get(k)}
    tl = device_timeline(timer, dw, cp)
    if tl:
        entry["device"] = tl
        entry["device_gbs"] = abytes / (tl["kernel_us"] * 1e-6) / 1e9
    if any(m.kind == 1 for m in w.models):
        tf = w.flops() / (used_ms * 1e-3) / 1e12
        entry["tensor"] = {"achieved_tflops": tf, "peak_burst": peaks["bf16_tflops"], "frac_burst": tf / peaks["bf16_tflops"],
                           "frac_sustained": tf / peaks["bf16_tflops_sustained"], "tensor_pipe_pct_ncu": NCU_TENSOR_PIPE_PCT.get(k)}
    if with_parity:
        dw.out.fill_(float("nan"))
        dw.lse.fill_(float("nan"))
        dw.decode()
        entry["parity_vs_oracle"] = parity_sample(w, dw.results())
    return entry


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--kernel", type=int, default=0, help="CP_OPT_KERNEL (0 auto, 1 generic)")
    ap.add_argument("--waves-x16", type=int, default=0, help="CP_OPT_WAVES_X16 (0 = library default)")
    ap.add_argument("--min-tile-pages", type=int, default=0, help="CP_OPT_MIN_TILE_PAGES (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (tuning sweeps only)")
    ap.add_argument("--no-vmm", action="store_true", help="skip the CUDA-VMM arena leg (SURVEY 8(f) N2)")
    ap.add_argument("--no-planner", action="store_true", help="skip the KV-cache planner leg (SURVEY 8(f) N3)")
    ap.add_argument("--no-stages", action="store_true", help="skip the multi-stage launch leg (SURVEY 8(f) N4)")
    ap.add_argument("--stage-layers", type=int, default=4, help="layers per batch in the multi-stage leg")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (the other four BASELINE configs)")
    ap.add_argument("--probe", default="", choices=["", "timeline", "stream", "launch"],
                    help="measurement aids: per-CTA timeline of the K/V kernel, read-only HBM ceiling, launch / event floor")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    import workloads as W
    if args.impl == "reference":
        if rank != 0:
            return 0
        run_reference(args, W.config(args.config), args.config)
        return 0

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    import paper_2606_24506_b200 as cp
    from paper_2606_24506_b200.harness import DeviceWorkload

    dev = "cuda:%d" % local_rank
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    k = args.config
    w = W.config(k)
    # room in the page lists for the tokens the append / decode-loop legs add (16 + 2 loops of max(2 P, 64) tokens)
    loop_tokens = 16 + 2 * max(2 * w.page_tokens, 64) + 8
    dw = DeviceWorkload(w, dev, page_list_slack=(-(-loop_tokens // w.page_tokens) + 2) * max(m.n_kv_heads for m in w.models))
    dw.pool.set_option(cp.CP_OPT_KERNEL, args.kernel)
    if args.waves_x16 > 0:
        dw.pool.set_option(cp.CP_OPT_WAVES_X16, args.waves_x16)
    if args.min_tile_pages > 0:
        dw.pool.set_option(cp.CP_OPT_MIN_TILE_PAGES, args.min_tile_pages)
    dw.ensure_workspace()
    abytes = w.algorithmic_bytes()
    peaks = measured_peaks()
    timer = StepTimer(torch, cp, dev, dw.stream())
    l2_flush = timer.l2_flush

    def spacer(i):
        """Before a per-step-timed call of the side legs: L2 flush (read-only), then a short device-side spin
        that keeps the host a step ahead, so that host launch latency never lands inside a measurement."""
        l2_flush()
        torch.cuda._sleep(100000)       # ~50 us at 1.9 GHz

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank) if rank == 0 else None

    # ---------------- probes (measurement aids; one JSON line each, then exit)
    if args.probe:
        if args.probe == "timeline":
            out = {"probe": "timeline", "config": workload_desc(w, k), "device": device_timeline(timer, dw, cp, reps=8)}
        elif args.probe == "stream":
            buf = torch.zeros(1 << 30, dtype=torch.uint8, device=dev)
            sink = torch.zeros(1, dtype=torch.int32, device=dev)
            res = {}
            for n_ctas in (148, 296, 592, 1184, 2368):
                ms = min(timer.region(10, lambda: cp.probe_read_stream(buf, buf.numel(), n_ctas, sink, dw.stream())) for _ in range(3))
                res[str(n_ctas)] = buf.numel() / (ms * 1e-3) / 1e9
            out = {"probe": "stream", "what": "read-only pass over 1 GiB, 16-byte loads, CTAs of 512 threads (cp_probe_read_stream)",
                   "gbs_by_ctas": res, "copy_peak_gbs": peaks["hbm_gbs"]}
        else:
            out = {"probe": "launch", "empty_kernel_event_pair_us": timer.empty_kernel_events_us(),
                   "back_to_back_empty_kernels_us": 1e3 * timer.region(50, lambda: cp.probe_globaltimer(timer.stamp, dw.stream()))}
        print(json.dumps(out))
        dw.close()
        return 0

    # ---------------- device-resident leg: K steps, inputs already in HBM, back to back inside one event pair
    t_wall0 = time.time()               # clocks are sampled from the warm-up on (the timed region is a few ms)
    for _ in range(args.warmup):
        dw.decode()
    barrier()
    c0 = dw.pool.counters()
    e_start, e_stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda._sleep(4000000)          # the host enqueues the K steps behind a ~2 ms device-side spin
    e_start.record()
    for i in range(args.steps):
        dw.decode()
    e_stop.record()
    barrier()
    c1 = dw.pool.counters()
    region_ms = e_start.elapsed_time(e_stop) / args.steps
    launches = c1["kernel_launches"] - c0["kernel_launches"]
    big = abytes > 2 * L2_BYTES
    # the same steps, each after a read-only L2 flush and bracketed by its own event pair (see StepTimer)
    per_step = timer.per_step(max(args.steps // 2, 20), dw.decode)
    flushed_ms = float(np.median(per_step))
    empty_us = timer.empty_kernel_events_us()
    empty_region_us = timer.empty_kernel_region_us()
    timer.event_overhead_us = max(empty_us - empty_region_us, 0.0)
    kern_ms = region_ms if big else flushed_ms         # the kernel's launch duration the roofline uses
    step_ms = reduce_max_over_ranks(kern_ms, dev)
    back_to_back_us = 1e3 * region_ms
    device_tl = device_timeline(timer, dw, cp) if rank == 0 else None
    headline_parity = None
    if rank == 0 and world == 1 and not args.no_per_config:
        dw.out.fill_(float("nan"))
        dw.lse.fill_(float("nan"))
        dw.decode()
        headline_parity = parity_sample(w, dw.results())

    # ---------------- end-to-end leg: host buffers through cp_decode_attention_host
    need = dw.pool.decode_workspace_bytes_host(dw.ids)
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    q_host = torch.from_numpy(w.q_packed().view(np.int16)).pin_memory()
    ol_host = torch.empty(dw.out.numel() + dw.lse.numel(), dtype=torch.float32).pin_memory()
    o_host, l_host = ol_host[:dw.out.numel()], ol_host[dw.out.numel():]     # adjacent: one device->host copy
    e2e_steps = 1 if args.no_e2e else args.steps
    # what a caller's serving loop holds between steps: the batch's ids as an int32 array and the stream handle (looking
    # the torch stream up and converting a Python list cost 6 us per call, a tenth of the step)
    e2e_ids, e2e_stream = np.ascontiguousarray(dw.ids, dtype=np.int32), dw.stream()
    for _ in range(1 if args.no_e2e else 3):
        dw.pool.decode_attention_host(e2e_ids, q_host, o_host, l_host, ws, need, e2e_stream)
    barrier()
    e2e_s = 0.0
    for i in range(e2e_steps):
        if not big:
            l2_flush()
        torch.cuda.synchronize()
        t0 = time.perf_counter()       # the call copies q H2D, runs the step, copies O/LSE D2H and syncs
        dw.pool.decode_attention_host(e2e_ids, q_host, o_host, l_host, ws, need, e2e_stream)
        e2e_s += time.perf_counter() - t0
    e2e_ms = 1e3 * e2e_s / e2e_steps
    e2e_ms = reduce_max_over_ranks(e2e_ms, dev)
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---------------- step a2 alone: translation + KV gather of the longest request (rank 0 only)
    gather = None
    if rank == 0:
        ri = max(range(len(w.requests)), key=lambda i: w.requests[i].context_len)
        rq = w.requests[ri]
        m = w.models[rq.model_id]
        gk = torch.empty((rq.context_len, m.n_kv_heads, m.head_dim_qk), dtype=torch.int16, device=dev)
        gv = torch.empty((rq.context_len, m.n_kv_heads, m.head_dim_v), dtype=torch.int16, device=dev)
        for _ in range(3):
            dw.pool.gather_kv(rq.request_id, gk, gv, dw.stream())
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 20
        torch.cuda.synchronize()
        g0.record()
        for _ in range(reps):
            dw.pool.gather_kv(rq.request_id, gk, gv, dw.stream())
        g1.record()
        torch.cuda.synchronize()
        g_ms = g0.elapsed_time(g1) / reps
        g_bytes = 2 * (gk.numel() + gv.numel()) * 2          # read + written
        gather = {"request": ri, "context_len": rq.context_len, "us": 1e3 * g_ms,
                  "traffic_gbs": g_bytes / (g_ms * 1e-3) / 1e9, "bytes_read_plus_written": g_bytes,
                  "note": "back-to-back launches (the gathered copy of a long request exceeds L2)"}
        del gk, gv

    # ---------------- CUDA-VMM-backed arena: the same step on an arena the library maps chunk
    # by chunk, page ids by arithmetic (no table) and with the identity table read anyway; and what the
    # slow path costs: mapping / unmapping the longest request's pages, against the software table's
    vmm = None
    if rank == 0 and world == 1 and not args.no_vmm:
        dv = DeviceWorkload(w, dev, vmm=True)
        dv.pool.set_option(cp.CP_OPT_KERNEL, args.kernel)
        dv.ensure_workspace()
        vmm = {"chunk_bytes": dv.pool.vmm_info()["chunk_bytes"], "chunks_mapped": dv.pool.vmm_info()["chunks_mapped"]}
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for table, name in ((0, "us_per_step_no_table"), (1, "us_per_step_identity_table")):
            dv.pool.set_option(cp.CP_OPT_VMM_TABLE, table)
            for _ in range(3):
                dv.decode()
            ts = []
            for i in range(min(args.steps, 50)):
                spacer(i)
                e0.record()
                dv.decode()
                e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            vmm[name] = 1e3 * float(np.median(ts))
        dv.close()
        del dv
        ri = max(range(len(w.requests)), key=lambda i: w.requests[i].page_ids.size)
        rq = w.requests[ri]
        n_pg = int(rq.page_ids.size)
        vp = cp.Pool.create_vmm(n_pg * w.page_bytes + (4 << 20), w.page_tokens, w.page_bytes, w.models, 2, n_pg)

        def wall_us(fn):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            fn()
            return 1e6 * (time.perf_counter() - t0)

        cold = wall_us(lambda: vp.map_pages(0, rq.model_id, None, rq.context_len, n_allocate=n_pg))
        chunks = vp.vmm_info()["chunks_mapped"]
        unmap = wall_us(lambda: vp.unmap_request(0))
        warm = wall_us(lambda: vp.map_pages(0, rq.model_id, None, rq.context_len, n_allocate=n_pg))
        vp.close()
        sp = cp.Pool(dw.arena, dw.arena.numel() * 2, w.page_tokens, w.page_bytes, w.num_pages, w.models, 2, n_pg)
        # (bookkeeping only: this pool never launches, the arena is not touched)
        soft = wall_us(lambda: sp.map_pages(0, rq.model_id, None, rq.context_len, n_allocate=n_pg))
        soft_unmap = wall_us(lambda: sp.unmap_request(0))
        sp.close()
        vmm["map_unmap_host_us"] = {
            "pages": n_pg, "chunks": chunks,
            "vmm_map_cold": cold, "vmm_map_parked_chunks": warm, "vmm_unmap": unmap,
            "software_table_map": soft, "software_table_unmap": soft_unmap,
            "note": "host wall clock of one cp_pool_map_pages / cp_pool_unmap_request call for the longest "
                    "request; cold = cuMemCreate + cuMemMap + cuMemSetAccess per chunk, parked = cuMemMap + "
                    "cuMemSetAccess; the software table's device upload is deferred to the next compute call"}

    # ---------------- multi-stage persistent launch: L layers in ONE launch against L
    # launches.  Every layer has its own copy of the workload's KV (distinct memory, L x the arena), so
    # nothing is re-read from L2.  (a) one batch of all requests, L dependent layers; (b) one batch per
    # model, two in flight, served in turn (the paper's layer-wise state machine), L layers each.
    stages_leg = None
    if rank == 0 and world == 1 and not args.no_stages and all(m.kind == 0 and m.head_dim_qk == 128 and m.head_dim_v == 128 for m in w.models):
        L = args.stage_layers
        nreq = len(w.requests)
        arena_l = dw.arena.repeat(L)
        max_ppr = max(r.page_ids.size for r in w.requests)
        pool_l = cp.Pool(arena_l, arena_l.numel() * 2, w.page_tokens, w.page_bytes, w.num_pages * L, w.models,
                         max_requests=nreq * L, max_pages_per_request=max_ppr)
        for l in range(L):
            for r in w.requests:
                pool_l.map_pages(l * nreq + r.request_id, r.model_id, r.page_ids + l * w.num_pages, r.context_len)
        sep_pools = {}

        def sep_pool(batch_key, l, ids):
            """Pool of one (batch, layer) for the separate launches: its plan stays cached."""
            if (batch_key, l) not in sep_pools:
                pl = cp.Pool(arena_l, arena_l.numel() * 2, w.page_tokens, w.page_bytes, w.num_pages * L, w.models,
                             max_requests=nreq, max_pages_per_request=max_ppr)
                for i in ids:
                    r = w.requests[i]
                    pl.map_pages(r.request_id, r.model_id, r.page_ids + l * w.num_pages, r.context_len)
                sep_pools[(batch_key, l)] = pl
            return sep_pools[(batch_key, l)]

        req_ids = [r.request_id for r in w.requests]
        by_model = [[r.request_id for r in w.requests if r.model_id == mi] for mi in range(len(w.models))]
        by_model = [b for b in by_model if b]

        def pipeline(layers, slots=2):
            queue = list(range(len(layers)))
            live = [queue.pop(0) for _ in range(min(slots, len(queue)))]
            cur = {b: 0 for b in live}
            order = []
            while any(b is not None for b in live):
                for i, b in enumerate(live):
                    if b is None:
                        continue
                    order.append((b, cur[b]))
                    cur[b] += 1
                    if cur[b] == layers[b]:
                        live[i] = queue.pop(0) if queue else None
                        if live[i] is not None:
                            cur[live[i]] = 0
            return order

        def rows_of(ids):
            return sum(w.models[w.requests[i].model_id].n_q_heads for i in ids)     # request_id == index

        def run_case(batches):
            order = pipeline([L] * len(batches))
            pos = {bl: s for s, bl in enumerate(order)}
            stages = [[l * nreq + i for i in batches[b]] for b, l in order]
            deps = [pos[(b, l - 1)] if l > 0 else -1 for b, l in order]
            rows = sum(rows_of(batches[b]) for b, _ in order)
            qs = torch.randn(rows * 128, device=dev).to(torch.bfloat16).view(torch.int16)
            outs = torch.empty(rows * 128, dtype=torch.float32, device=dev)
            lses = torch.empty(rows, dtype=torch.float32, device=dev)
            wsb = max(pool_l.decode_stages_workspace_bytes(stages, deps), 256)
            wss = torch.empty(wsb, dtype=torch.uint8, device=dev)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            one, sep = [], []
            for i in range(3 + 15):
                spacer(i)
                e0.record()
                pool_l.decode_attention_stages(stages, deps, 1.0, qs, outs, lses, wss, wsb, dw.stream())
                e1.record()
                torch.cuda.synchronize()
                one.append(e0.elapsed_time(e1))
            # the same stages through the request queue (cp_queue_*): nothing is known to the kernel at launch, the
            # planner warp on the GPU cuts every stage into tiles as it reads it from the ring.  All stages are
            # pushed before the launch here, so this times the device-side planning, not the host's push rate.
            qtimes, qst = [], {"error": None}
            ids_l = [[int(x) for x in st] for st in stages]
            use_queue = max(len(st) for st in stages) <= 12          # a queue entry holds at most 12 requests
            wsq = torch.empty(max(4 * wsb, 64 << 20), dtype=torch.uint8, device=dev)
            for i in range(3 + 10 if use_queue else 0):
                qu = cp.Queue(pool_l, max_stages=len(stages) + 1)
                for st_ids, dp in zip(ids_l, deps):
                    qu.push(st_ids, dp, 1.0)
                qu.close_queue()
                spacer(i)
                e0.record()
                qu.launch(qs, outs, lses, wsq, wsq.numel(), 2000, dw.stream())
                e1.record()
                torch.cuda.synchronize()
                qtimes.append(e0.elapsed_time(e1))
                qst = qu.status(dw.stream())
                qu.free()
            del wsq
            # the same stages as separate launches (plain steps, no dependency between them)
            offs, ro = [], 0
            for b, l in order:
                offs.append(ro)
                ro += rows_of(batches[b])
            pools = [sep_pool((len(batches), b), l, batches[b]) for b, l in order]
            wsb1 = max(max(pl.decode_workspace_bytes(batches[b]) for pl, (b, l) in zip(pools, order)), 256)
            ws1 = torch.empty(wsb1, dtype=torch.uint8, device=dev)
            for i in range(3 + 15):
                spacer(i)
                e0.record()
                for s, (b, l) in enumerate(order):
                    pools[s].decode_attention(batches[b], qs[offs[s] * 128:], outs[offs[s] * 128:], lses[offs[s]:],
                                              ws1, wsb1, dw.stream())
                e1.record()
                torch.cuda.synchronize()
                sep.append(e0.elapsed_time(e1))
            # host-driven: the host sees every stage complete before it launches the next (Fig. 5a)
            host = []
            for i in range(2 + 8):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for s, (b, l) in enumerate(order):
                    pools[s].decode_attention(batches[b], qs[offs[s] * 128:], outs[offs[s] * 128:], lses[offs[s]:],
                                              ws1, wsb1, dw.stream())
                    torch.cuda.synchronize()
                host.append(1e3 * (time.perf_counter() - t0))
            t3 = float(np.median(host[2:]))
            kv_bytes = sum(w.requests[i].context_len * w.models[w.requests[i].model_id].n_kv_heads * 512
                           for b, _ in order for i in batches[b])
            t1, t2 = float(np.median(one[3:])), float(np.median(sep[3:]))
            tq = float(np.median(qtimes[3:])) if use_queue else None
            return {"stages": len(order), "kv_bytes": int(kv_bytes), "one_launch_us": 1e3 * t1,
                    "queue_launch_us": 1e3 * tq if use_queue else None,
                    "queue_us_per_stage": 1e3 * tq / len(order) if use_queue else None, "queue_device_error": qst["error"],
                    "separate_launches_us": 1e3 * t2, "one_launch_us_per_stage": 1e3 * t1 / len(order),
                    "separate_us_per_stage": 1e3 * t2 / len(order),
                    "host_driven_us_per_stage_wall": 1e3 * t3 / len(order), "one_launch_gbs": kv_bytes / (t1 * 1e-3) / 1e9,
                    "separate_gbs": kv_bytes / (t2 * 1e-3) / 1e9}

        stages_leg = {"layers": L,
                      "one_batch_of_all_requests": run_case([req_ids]),
                      "one_batch_per_model_two_in_flight": run_case(by_model),
                      "note": "separate launches: the same stages as back-to-back cp_decode_attention calls, each on a "
                              "pool of its own so that its plan stays cached (no dependency between them)"}
        pool_l.close()
        for pl in sep_pools.values():
            pl.close()
        del arena_l

    # ---------------- q_len > 1 (SURVEY §8(f) N4 variant): the same KV, four query tokens per request
    qlen_leg = None
    if rank == 0 and world == 1 and not args.no_stages and all(m.kind == 0 and m.head_dim_qk == 128 and m.head_dim_v == 128 and
                                                m.n_q_heads // m.n_kv_heads * 4 <= 128 for m in w.models):
        ql = 4
        rows = w.out_rows() * ql
        qq = torch.randn(rows * 128, device=dev).to(torch.bfloat16).view(torch.int16)
        oq = torch.empty(rows * 128, dtype=torch.float32, device=dev)
        lq = torch.empty(rows, dtype=torch.float32, device=dev)
        wsb = max(dw.pool.decode_workspace_bytes_qlen(dw.ids, ql), 256)
        wsq = torch.empty(wsb, dtype=torch.uint8, device=dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ts = []
        for i in range(3 + 20):
            spacer(i)
            e0.record()
            dw.pool.decode_attention_qlen(dw.ids, ql, qq, oq, lq, wsq, wsb, dw.stream())
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        t = float(np.median(ts[3:]))
        qlen_leg = {"q_len": ql, "us_per_step": 1e3 * t, "kv_gbs": abytes / (t * 1e-3) / 1e9}
        del qq, oq, lq, wsq

    # ---------------- KV-cache planner (Eq. (1)-(2)): pool demand at 100 000 observation
    # times of a two-hour synthetic trace of 8 cold models, then P95 / P99 and the page budgets
    planner = None
    if rank == 0 and world == 1 and not args.no_planner:
        from workloads.planner_traces import planner_trace
        tr = planner_trace(1)
        td = [torch.from_numpy(a).to(dev) for a in (tr.arrival, tr.o_p, tr.o_d, tr.t_res, tr.t_obs)]
        kp = torch.empty(tr.t_obs.size, dtype=torch.float64, device=dev)
        wsb = cp.planner_workspace_bytes(tr.n_requests)
        pws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        st = dw.stream()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d_us, q_us = [], []
        for i in range(6):
            p0.record()
            cp.planner_pool_demand(tr.offsets, tr.kappa, td[0], td[1], td[2], td[3], tr.t_obs.size, td[4], kp, pws, wsb, st)
            p1.record()
            torch.cuda.synchronize()
            d_us.append(1e3 * p0.elapsed_time(p1))
            t0 = time.perf_counter()
            budgets = {q: cp.planner_quantile(kp, tr.t_obs.size, q, float(w.page_bytes), pws, wsb, st) for q in (0.95, 0.99)}
            q_us.append(1e6 * (time.perf_counter() - t0) / 2)
        planner = {"models": tr.n_models, "trace_requests": tr.n_requests, "observations": int(tr.t_obs.size),
                   "demand_us": float(np.median(d_us[1:])), "quantile_us_host_wall": float(np.median(q_us[1:])),
                   "observations_per_s": tr.t_obs.size / (float(np.median(d_us[1:])) * 1e-6),
                   "p95_gib": budgets[0.95][0] / 2 ** 30, "p99_gib": budgets[0.99][0] / 2 ** 30,
                   "p95_pages": budgets[0.95][1], "p99_pages": budgets[0.99][1], "page_bytes": int(w.page_bytes),
                   "dtype": "f64"}
        if not args.no_cpu_baseline:
            import oracle
            n_s = 2000
            t0 = time.perf_counter()
            oracle.pool_demand(tr.offsets, tr.kappa, tr.arrival, tr.o_p, tr.o_d, tr.t_res, tr.t_obs[:n_s])
            planner["cpu_oracle_observations_per_s"] = n_s / (time.perf_counter() - t0)
            planner["cpu_oracle_sample"] = "%d of the observation times, one core" % n_s
        del td, kp, pws

    # ---------------- KV append step, last because it grows the contexts: one new token
    # per request per call, launch-bound (a few KB per call); reported as us per call on the device
    append = None
    if rank == 0:
        kn = sum(m.n_kv_heads * m.head_dim_qk for m in (w.models[r.model_id] for r in w.requests))
        vn = sum(m.n_kv_heads * m.head_dim_v for m in (w.models[r.model_id] for r in w.requests) if m.kind == 0)
        k_new = torch.zeros(kn, dtype=torch.int16, device=dev)
        v_new = torch.zeros(max(vn, 8), dtype=torch.int16, device=dev)
        reps = 8
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        dw.pool.append_kv(dw.ids, k_new, v_new, dw.stream())
        torch.cuda._sleep(400000)          # keep the device busy while the host enqueues the calls
        a0.record()
        for _ in range(reps):
            dw.pool.append_kv(dw.ids, k_new, v_new, dw.stream())
        a1.record()
        torch.cuda.synchronize()
        append = {"us_per_call": 1e3 * a0.elapsed_time(a1) / reps, "requests": len(w.requests),
                  "bytes_per_call": 2 * (kn + vn)}
        # a decode LOOP as a serving engine runs it (one new token per request per iteration, page boundaries
        # included, so the tile plan is rebuilt and re-uploaded whenever a request opens a page):
        #   fused   cp_decode_step: append + attention, one launch per iteration on the tcgen05 K/V kernel
        #   two     cp_pool_append_kv then cp_decode_attention
        # wall clock of the free-running loop (host and device as a server would run them: whichever is slower
        # sets the pace) and the host's enqueue time per iteration.
        n_loop = max(2 * w.page_tokens, 64)
        need = max(dw.pool.decode_step_workspace_bytes(dw.ids), dw.ws_bytes, 256)
        wsl = torch.empty(need + (1 << 20), dtype=torch.uint8, device=dev)

        def loop(fused, steps):
            c0 = dw.pool.counters()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0.record()
            for _ in range(steps):
                if fused:
                    dw.pool.decode_step(dw.ids, k_new, v_new, dw.q, dw.out, dw.lse, wsl, wsl.numel(), dw.stream())
                else:
                    dw.pool.append_kv(dw.ids, k_new, v_new, dw.stream())
                    dw.pool.decode_attention(dw.ids, dw.q, dw.out, dw.lse, wsl, wsl.numel(), dw.stream())
            e1.record()
            t_enq = time.perf_counter() - t0
            torch.cuda.synchronize()
            t_all = time.perf_counter() - t0
            c1 = dw.pool.counters()
            return {"us_per_iteration": 1e6 * t_all / steps,
                    "stream_us_per_iteration": 1e3 * e0.elapsed_time(e1) / steps,
                    "host_enqueue_us_per_iteration": 1e6 * t_enq / steps,
                    "launches_per_iteration": (c1["kernel_launches"] - c0["kernel_launches"]) / steps,
                    "plan_builds": c1["plan_builds"] - c0["plan_builds"]}
        loop(True, 4)

        def single_step_device_us(reps=8):
            """Kernel duration on the device (first CTA entry to last CTA done, CP_OPT_TIMELINE) of single steps, one at a
            time, no flush: the plain step and the fused step alternate, so both see the same cache state."""
            dw.pool.set_option(cp.CP_OPT_TIMELINE, 1)
            res = {"plain": [], "fused": []}
            try:
                for _ in range(reps):
                    for name in ("plain", "fused"):
                        if name == "plain":
                            dw.pool.decode_attention(dw.ids, dw.q, dw.out, dw.lse, wsl, wsl.numel(), dw.stream())
                        else:
                            dw.pool.decode_step(dw.ids, k_new, v_new, dw.q, dw.out, dw.lse, wsl, wsl.numel(), dw.stream())
                        torch.cuda.synchronize()
                        t = dw.pool.read_timeline().astype(np.int64)
                        t = t[t[:, 0] > 0]
                        if t.size == 0 or t[:, 7].max() == 0:
                            return None              # a kernel that does not stamp (MLA, generic)
                        res[name].append((t[:, 7].max() - t[:, 0].min()) / 1e3)
            finally:
                dw.pool.set_option(cp.CP_OPT_TIMELINE, 0)
            return {k: float(np.median(v)) for k, v in res.items()}
        dev_cmp = single_step_device_us()
        append["decode_loop"] = {"iterations": n_loop,
                                 "fused_cp_decode_step": loop(True, n_loop),
                                 "append_then_attention": loop(False, n_loop),
                                 "single_step_kernel_us_on_device": dev_cmp,
                                 "plain_step_cached_plan_us": back_to_back_us,
                                 "note": "a free-running loop (no device-side spin in front): us_per_iteration is wall clock from the "
                                         "first enqueue to the final synchronise, i.e. max(host, device); every request crosses a "
                                         "page boundary at least once, so the plan is rebuilt and re-uploaded plan_builds times"}
        del wsl

    if gather:
        gather["frac_of_measured_copy_peak"] = gather["traffic_gbs"] / peaks["hbm_gbs"]
    value = whole_job_value(abytes, world, step_ms)
    achieved = abytes / (kern_ms * 1e-3) / 1e9
    mla = any(m.kind == 1 for m in w.models)
    roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
            "frac": achieved / peaks["hbm_gbs"], "traffic": NCU_TRAFFIC_BYTES.get(k), "peak_source": peaks["source"],
            "kernel_us": 1e3 * kern_ms,
            "kernel_us_is": ("K steps back to back inside one event pair (inputs %.0f MB > 2 x L2, no flush)" % (abytes / 1e6)) if big
                            else "median of K steps, each after a read-only L2 flush and inside its own event pair",
            "region_us": 1e3 * region_ms, "flushed_us": 1e3 * flushed_ms, "flushed_gbs": abytes / (flushed_ms * 1e-3) / 1e9,
            "flushed_us_p10_p50_p90": [float(x) * 1e3 for x in np.percentile(per_step, [10, 50, 90])],
            "flushed_calibrated_us": 1e3 * flushed_ms - timer.event_overhead_us,
            "empty_kernel_events_us": empty_us, "empty_kernel_region_us": empty_region_us,
            "device": device_tl, "device_gbs": (abytes / (device_tl["kernel_us"] * 1e-6) / 1e9) if device_tl else None,
            "frac_of_nominal_8000": achieved / 8000.0, "parity_vs_oracle": headline_parity}
    if mla:
        tf = w.flops() / (kern_ms * 1e-3) / 1e12
        roof["tensor"] = {"achieved_tflops": tf, "peak_burst": peaks["bf16_tflops"],
                          "frac_burst": tf / peaks["bf16_tflops"],
                          "tensor_pipe_pct_ncu": NCU_TENSOR_PIPE_PCT.get(k)}

    # ---------------- the other BASELINE configs through the same protocol (north_star: "all five configs")
    per_config = None
    if rank == 0 and world == 1 and not args.no_per_config and k == 2:
        per_config = {}
        for kk in (1, 3, 4, 5):
            wk = W.config(kk)
            dk = DeviceWorkload(wk, dev)
            dk.pool.set_option(cp.CP_OPT_KERNEL, args.kernel)
            try:
                per_config["cfg%d" % kk] = measure_config(timer, cp, kk, wk, dk, max(args.steps // 2, 30), peaks)
            finally:
                dk.close()
            del dk, wk

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "us_per_step": 1e3 * step_ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16 in, fp32 accumulate",
            "data": "synthetic", "config": workload_desc(w, k), "clocks": clocks,
            "e2e": {"value": whole_job_value(abytes, world, e2e_ms), "unit": UNIT,
                    "us_per_step": 1e3 * e2e_ms,
                    "h2d_bytes_per_step": int(q_host.numel() * 2),
                    "d2h_bytes_per_step": int(o_host.numel() * 4 + l_host.numel() * 4)},
            "gpu_launches": int(launches), "back_to_back_no_flush_us_per_step": back_to_back_us, "roofline": roof,
            "per_config": per_config, "gather": gather, "append": append, "vmm_arena": vmm, "planner": planner,
            "stages": stages_leg, "qlen": qlen_leg,
            "pct_of_hbm_peak": {"measured_copy": 100 * achieved / peaks["hbm_gbs"], "nominal_8TBs": 100 * achieved / 8000.0}}

    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        heads, frac = oracle_sample_plan(w, 8.0)
        t0 = time.perf_counter()
        n = 0
        while True:
            oracle.decode_workload(w, heads_per_request=heads)
            n += 1
            if time.perf_counter() - t0 > 10.0 or n >= 3:
                break
        dt = (time.perf_counter() - t0) / n
        line["cpu_baseline"] = {"value": frac * abytes / dt / 1e9, "unit": UNIT, "cores": oracle.num_threads(),
                                "kind": "oracle", "us_per_step": 1e6 * dt / frac,
                                "sample": "%d pass(es) over every request, %.1f%% of the (head, token) pairs" % (n, 100 * frac)}
    print(json.dumps(line))
    dw.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
