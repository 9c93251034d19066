#!/usr/bin/env python
"""bench.py -- events/sec of the whole hot path (event build, discretisation,
filter scan, smoother, log-likelihood, posterior at the observations) on BASELINE.json's headline
workload: config 3 (quasiperiodic kernel, n = 21, N = 100 000 exposures, K = 200 000 events, fp64).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 3]

One JSON line on stdout (rank 0).  `value` = events/s with inputs resident in HBM; `e2e` = the same
through the *_host C-ABI calls from pinned host buffers (copies inside the timed region).  Under
torchrun (N > 1) every rank runs an independent replica of the workload on its own GPU (the path
does not shard: DESIGN.md "Multi-GPU": replicas only, no collective) and `value` is the aggregate.
`--impl reference` times the CPU oracle (oracle/, fp64 build) on a bounded sample of the workload.
"""
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

from paper_2601_02527_b200 import workloads as W  # noqa: E402

FP64_PEAK_DERIVED_TFLOPS = 37.2  # 148 SM x 64 DFMA/clk x 2 flop x 1.965 GHz; the line's `peak` is MEASURED


def fp64_probe(device):
    """plain-ALU FP64 FMA throughput of this device, measured now (TFLOP/s): the roofline denominator.
    MEASURED_PEAKS.json has no FP64 entry; the probe is bench.py's own tool (csrc/probe_fp64.cu)."""
    import ctypes
    from paper_2601_02527_b200 import _build
    L = ctypes.CDLL(_build.build_probe())
    v = ctypes.c_double()
    rc = L.sgprobe_fp64(int(device), 5, ctypes.byref(v))
    if rc != 0:
        raise RuntimeError("fp64 probe failed: cuda error %d" % rc)
    return v.value


def hbm_peak_gbs():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json"
    except (OSError, ValueError, KeyError):
        return 6545.9, "fallback (SURVEY 0: 6545.9 GB/s)"


def kernel_source_hash():
    """hash of the chunk / dense kernel sources: an ncu capture under profiles/ is only quoted for the
    build it was taken from"""
    import hashlib
    h = hashlib.sha256()
    for f in ("dev_consts.h", "grp_dev.cuh", "chunk_dev.cuh", "chunk_kernels.cuh", "chunk_reg.cuh", "dense_kernels.cuh", "scan_host.cu"):
        try:
            h.update(open(os.path.join(ROOT, "paper_2601_02527_b200", "csrc", f), "rb").read())
        except OSError:
            pass
    return h.hexdigest()[:16]


def w_useful_flops(n):
    """dense flop count of the sequential algorithm per event (predict + update +
    smoother gain/update): 10.3 n^3 + 9 n^2."""
    return 10.3 * n ** 3 + 9.0 * n ** 2


def min_bytes(n):
    """inputs 24 B/event + outputs 8 B/event + one write and one read of the filtered
    (m, P) between the passes."""
    return 32 + 2 * 8 * (n + n * (n + 1) // 2)


def ncu_capture(kernel, cfg):
    """(dram bytes per launch, executed-DFMA fraction of the FP64 peak, source) of the dominant kernel from the
    committed ncu --set full capture of THIS build (profiles/r02_top_kernel_capture.json: config 3 only; the
    capture records the hash of the kernel sources it was taken from), else (None, None, why)"""
    path = os.path.join(ROOT, "profiles", "r02_top_kernel_capture.json")
    try:
        rec = json.load(open(path))
    except (OSError, ValueError):
        return None, None, "no capture file"
    if cfg != 3 or rec.get("kernel") != kernel:
        return None, None, "capture is of %s on config 3" % rec.get("kernel")
    if rec.get("source_hash") != kernel_source_hash():
        return None, None, "capture is stale (kernel sources changed since profiles/r02_top_kernel_capture.json)"
    return rec.get("traffic_bytes_per_launch"), rec.get("dfma_frac_of_peak"), "profiles/r02_top_kernel_capture.json"


def model_dim(w):
    d = 0
    for c in w["kernel"]:
        d += {W.MATERN32: 2, W.MATERN52: 3, W.SHO: 2}.get(c["family"], 2 + 4 * c["order"])
    return d + w["n_inst"]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference): the fp64 build of oracle/smolgp_oracle.c,
# as it stands, single thread (the recursion is sequential in k), on a bounded sample = the first
# `n_sample` exposures of the workload.
# ----------------------------------------------------------------------------------------------
def oracle_step(w, n_sample, series=0, split=False):
    """one pass of the fp64 oracle over the first n_sample exposures of series `series`; seconds (and, with
    split, the seconds of that pass spent in the discretisation: oracle instrumentation)"""
    import oracle
    sl = slice(0, n_sample)
    y = w["y"][series, sl] if w["y"].ndim == 2 else w["y"][sl]
    kern = w["kernel"]
    if w.get("amp") is not None:
        kern = [dict(k, sigma=k["sigma"] * float(w["amp"][series])) for k in kern]
    if w.get("instant"):
        t0 = time.perf_counter()
        oracle.ssm_instant(kern, w["n_inst"], w["t_start"][sl], w["instrument"][sl], y, w["sigma"][sl], prec="f64")
        dt = time.perf_counter() - t0
        return (dt, float("nan")) if split else dt
    t0 = time.perf_counter()
    r = oracle.ssm(kern, w["n_inst"], w["t_start"][sl], w["t_end"][sl], w["instrument"][sl], y, w["sigma"][sl],
                   flags=oracle.FLAG_IDLE_ZERO | oracle.FLAG_TWO_FILTER, prec="f64")
    dt = time.perf_counter() - t0
    return (dt, r["disc_seconds"]) if split else dt


def oracle_all_cores(w, n_series, n_sample):
    """batched workloads on all host cores, one series per thread (the C call releases the GIL).
    Returns (events/s, threads used, seconds)."""
    from concurrent.futures import ThreadPoolExecutor
    threads = min(os.cpu_count() or 1, n_series)
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(lambda s: oracle_step(w, n_sample, series=s), range(n_series)))
    dt = time.perf_counter() - t0
    return 2.0 * n_sample * n_series / dt, threads, dt


def oracle_sample_size(w, target_s):
    """exposures such that one oracle pass takes about target_s seconds (calibrated on 500)."""
    N = w["t_start"].size
    n0 = min(500, N)
    t = oracle_step(w, n0)
    return int(max(n0, min(N, n0 * target_s / max(t, 1e-6))))


def run_reference(args, w, cfgname):
    import oracle
    oracle.build()
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    ns = oracle_sample_size(w, 4.0)
    for _ in range(args.warmup):
        oracle_step(w, min(ns, 2000))
    ts = [oracle_step(w, ns) for _ in range(args.steps)]
    tot = sum(ts)
    epe = 1 if w.get("instant") else 2
    val = float(epe) * ns * args.steps / tot
    sample = "first %d of %d exposures (%d events) per step, oracle fp64 build, sequential filter + %s, 1 thread" % (
        ns, w["t_start"].size, epe * ns, "RTS smoother (section 2)" if w.get("instant") else "two-filter smoother")
    line = {"impl": "reference", "metric": "events/sec for loglik+RTS smoother at N=1e5", "value": val, "unit": "events/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfgname, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "events/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------
# multi-rank plumbing: replicas only -- no data-path collective; the only exchange is
# the max over ranks of the timed milliseconds
# ----------------------------------------------------------------------------------------------
def max_over_ranks(values, world, device):
    if world <= 1:
        return list(values)
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def aggregate_throughput(events_per_replica, steps, ms_max, world):
    """whole-job events/s: every rank processed the same number of events, in the slowest rank's time"""
    return world * events_per_replica * steps / (ms_max * 1e-3)


# ----------------------------------------------------------------------------------------------
# CUDA arm
# ----------------------------------------------------------------------------------------------
def run_cuda(args, w, cfgname):
    import torch
    import torch.distributed as dist
    from paper_2601_02527_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    ctx = B.Context(local)  # NULL stream = the legacy default stream = torch's current stream here
    if args.form == "sqrt":
        ctx.set_option("form", 1)  # square-root form of the chunk recursions: one chunk per series
    N = w["t_start"].size
    batch = w["batch"] or 1
    n = model_dim(w)
    K_events = 2 * N * batch
    h2d = lambda a: torch.tensor(a, device=dev)
    ts, te, ins, y, sg = (h2d(w[k]) for k in ("t_start", "t_end", "instrument", "y", "sigma"))
    amp = None if w["amp"] is None else h2d(w["amp"])
    out = dict(mean=torch.empty((batch, N), dtype=torch.float64, device=dev),
               var=torch.empty((batch, N), dtype=torch.float64, device=dev),
               loglik=torch.empty(batch, dtype=torch.float64, device=dev))
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)  # > the 126 MB L2

    instant = bool(w.get("instant"))
    ev_per_exp = 1 if instant else 2
    K_events = ev_per_exp * N * batch

    def step():
        ev = ctx.smolgp_build_events_instant(ts, ins, w["n_inst"]) if instant else ctx.smolgp_build_events(ts, te, ins, w["n_inst"])  # a1
        ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp, out=out)               # a2-a6
        ev.free()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()  # nvidia-smi needs a moment to come up: started before the warm-up, read after the timed loops
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # which kernel dominates: one untimed step with every launch bracketed by the library's CUDA events
    ctx.profile(True)
    step()
    prof1 = ctx.profile_read()
    top = max(prof1, key=lambda k: prof1[k][0])
    # timed region: only the dominant kernel is bracketed (two event records per step); bracketing every launch
    # costs ~0.25 ms per step of config 3 and would be charged to the headline
    ctx.profile(top)
    l0 = ctx.launch_count()
    evs = []
    barrier()
    for _ in range(args.steps):
        flush.fill_(1)  # evict L2 between timed iterations (not timed)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step(); b.record()
        evs.append((a, b))
    barrier()
    ms = sum(a.elapsed_time(b) for a, b in evs)
    launches = ctx.launch_count() - l0
    prof_top = ctx.profile_read()[top]
    # per-kernel table: a second pass of the same steps with every launch bracketed (not part of `value`)
    ctx.profile(True)
    evs_p = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step(); b.record()
        evs_p.append((a, b))
    prof = ctx.profile_read()
    ctx.profile(False)
    ms_bracketed = sum(a.elapsed_time(b) for a, b in evs_p)

    # ---- end to end: host buffers (pinned), copies inside the timed region, through the *_host C ABI ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hts, hte, hins, hy, hsg = (pin(w[k]) for k in ("t_start", "t_end", "instrument", "y", "sigma"))
    hamp = None if w["amp"] is None else pin(w["amp"])
    hout = dict(mean=pin(np.empty((batch, N))), var=pin(np.empty((batch, N))), loglik=pin(np.empty(batch)))

    def step_e2e():
        ev = ctx.smolgp_build_events_instant_host(hts, hins, w["n_inst"]) if instant else ctx.smolgp_build_events_host(hts, hte, hins, w["n_inst"])
        ctx.smolgp_condition_host(ev, w["kernel"], hy, hsg, amp=hamp, out=hout)
        ev.free()

    for _ in range(3):
        step_e2e()
    barrier()
    evs2 = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step_e2e(); b.record()
        evs2.append((a, b))
    barrier()
    ms_e2e = sum(a.elapsed_time(b) for a, b in evs2)
    clocks = sampler.stop() if rank == 0 else None
    peak = fp64_probe(local) if rank == 0 else None
    plan = ctx.plan_info()
    jit_log = ctx.jit_log()

    ms, ms_e2e = max_over_ranks([ms, ms_e2e], world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    value = aggregate_throughput(K_events, args.steps, ms, world)
    e2e_value = aggregate_throughput(K_events, args.steps, ms_e2e, world)
    # ---- roofline.  Three fractions, none to be mistaken for another:
    #   frac            : the dominant kernel credited with the whole path's USEFUL work, W_useful x the
    #                     events of one launch / its average duration (CUDA events on the ctx stream, timed region);
    #   frac_whole_step : SURVEY 8(d)'s headline fraction T_roof / t_measured over the WHOLE step;
    #   frac_executed_dfma : DFMA actually executed by that kernel (ncu capture of this build under profiles/).
    t_top_ms = prof_top[0] / prof_top[1]             # average launch duration over the timed region
    launches_per_step = prof_top[1] / args.steps
    flops_launch = K_events * w_useful_flops(n) / launches_per_step
    achieved = flops_launch / (t_top_ms * 1e-3) / 1e12
    hbm_gbs, hbm_src = hbm_peak_gbs()
    t_step = ms / args.steps * 1e-3
    t_roof = max(K_events * w_useful_flops(n) / (peak * 1e12), K_events * min_bytes(n) / (hbm_gbs * 1e9))
    traffic, dfma_frac, cap_src = ncu_capture(top, args.config) if args.form == "cov" else (None, None, "the capture is of the covariance form")
    roofline = {"bound": "alu", "kernel": top, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": traffic,
                "frac_whole_step": t_roof / t_step, "frac_executed_dfma": dfma_frac, "capture": cap_src,
                "peak_source": "measured in this run: register-only FP64 FMA probe (csrc/probe_fp64.cu), best of 5; "
                               "derived figure 148 SM x 64 FMA/clk x 2 x 1.965 GHz = %.1f TFLOP/s" % FP64_PEAK_DERIVED_TFLOPS,
                "work_model": "W_useful = 10.3 n^3 + 9 n^2 flop/event (SURVEY 8(d)), n = %d; `frac` credits the dominant kernel with "
                              "the whole path's useful work, `frac_whole_step` = T_roof / t_measured of the whole step, "
                              "`frac_executed_dfma` = executed DFMA of the dominant kernel (ncu)" % n,
                "kernel_share_of_step": prof_top[0] / ms,
                "timing": "dominant kernel: CUDA events on the ctx stream around its launches inside the timed region; "
                          "kernels_ms_per_step: a second pass of the same steps with every launch bracketed, %.3f ms/step "
                          "(the event records cost the difference to ms_per_step, so the headline loop does not carry them)" % (ms_bracketed / args.steps),
                "hbm": {"min_bytes_per_event": min_bytes(n), "achieved_gbs": K_events * min_bytes(n) * args.steps / (ms * 1e-3) / 1e9,
                        "peak_gbs": hbm_gbs, "peak_source": hbm_src},
                "kernels_ms_per_step": {k: v[0] / args.steps for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])}}
    # ---- CPU baseline: the oracle as it stands, bounded sample; discretisation and filter/smoother seconds apart
    #      (BASELINE.md 3); batched workloads also on all host cores, one series per thread ----
    import oracle
    oracle.build()
    ns = oracle_sample_size(w, 12.0)
    t_cpu, t_disc = oracle_step(w, ns, split=True)
    cpu = {"value": ev_per_exp * ns / t_cpu, "unit": "events/s", "cores": 1, "kind": "oracle",
           "seconds": {"total": t_cpu, "discretisation": t_disc, "filter_smoother": t_cpu - t_disc},
           "sample": "first %d of %d exposures (%d events), oracle fp64 build, sequential filter + %s, 1 thread, %.1f s" % (ns, N, ev_per_exp * ns, "RTS smoother (section 2)" if instant else "two-filter smoother", t_cpu)}
    if batch > 1:
        # a series of a batched workload is short: time enough of them for ~12 s on one core, then the same count per core on all cores
        n1 = int(max(1, min(batch, 12.0 / max(t_cpu, 1e-6))))
        t_one = sum(oracle_step(w, ns, series=s_) for s_ in range(n1))
        cpu.update(value=ev_per_exp * ns * n1 / t_one,
                   sample="%d series x first %d of %d exposures, oracle fp64 build, 1 thread, %.1f s" % (n1, ns, N, t_one))
        nser = int(min(batch, n1 * (os.cpu_count() or 1)))
        v_all, thr, t_all = oracle_all_cores(w, nser, ns)
        cpu["all_cores"] = {"value": v_all * ev_per_exp / 2.0, "unit": "events/s", "cores": thr,
                            "sample": "%d series x first %d exposures, one series per thread, %.1f s" % (nser, ns, t_all)}
    line = {"metric": "events/sec for loglik+RTS smoother at N=1e5", "value": value, "unit": "events/s",
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfgname, "N": N, "events": ev_per_exp * N, "batch": batch, "state_dim": n,
                       "path": "a1 build_events + a2 discretise + a3 filter scan + a4 smoother + a5 loglik + a6 posterior",
                       "l2": "flushed (512 MiB write) between timed iterations", "parallelism": "replicas x%d" % world,
                       "plan": plan, "form": args.form},
            "e2e": {"value": e2e_value, "unit": "events/s",
                    "h2d_bytes_per_step": int(hts.nbytes + hte.nbytes + hins.nbytes + hy.nbytes + hsg.nbytes + (0 if hamp is None else hamp.nbytes)),
                    "d2h_bytes_per_step": int(hout["mean"].nbytes + hout["var"].nbytes + hout["loglik"].nbytes),
                    "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": int(launches), "specialised": "jit=1" in plan, "jit_log": jit_log,
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
            "loglik": float(hout["loglik"][0])}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------------------------
# prediction workload (the paper's third benchmark column): condition + predict at
# M = mult x N query times
# ----------------------------------------------------------------------------------------------
def run_predict(args, w, cfgname):
    import torch
    from paper_2601_02527_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --workload predict: single GPU only")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    ctx = B.Context(0)
    if args.form == "sqrt":
        ctx.set_option("form", 1)  # query-time prediction from stored factors
    N = w["t_start"].size
    batch = w["batch"] or 1
    n = model_dim(w)
    M = int(args.predict_mult * N)
    t0, t1 = float(w["t_start"].min()), float(w["t_end"].max())
    tq_h = np.linspace(t0 - 0.001 * (t1 - t0), t1 + 0.001 * (t1 - t0), M)  # uniform grid over the data span (and a little beyond)
    h2d = lambda a: torch.tensor(a, device=dev)
    ts, te, ins, y, sg, tq = (h2d(a) for a in (w["t_start"], w["t_end"], w["instrument"], w["y"], w["sigma"], tq_h))
    amp = None if w["amp"] is None else h2d(w["amp"])
    out = dict(mean=torch.empty((batch, N), dtype=torch.float64, device=dev), var=torch.empty((batch, N), dtype=torch.float64, device=dev),
               loglik=torch.empty(batch, dtype=torch.float64, device=dev),
               mean_query=torch.empty((batch, M), dtype=torch.float64, device=dev), var_query=torch.empty((batch, M), dtype=torch.float64, device=dev))
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)

    def step():
        ev = ctx.smolgp_build_events(ts, te, ins, w["n_inst"])
        ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp, t_query=tq, query_instrument=0, out=out)
        ev.free()

    sampler = ClockSampler(0)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    ctx.memory_info(reset_peak=True)
    l0 = ctx.launch_count()
    evs = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step(); b.record()
        evs.append((a, b))
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / args.steps
    launches = (ctx.launch_count() - l0) // args.steps
    _, peak_bytes = ctx.memory_info()
    ctx.profile(True)
    step()
    prof = ctx.profile_read()
    ctx.profile(False)
    # end to end from pinned host buffers (queries and their outputs cross PCIe every step)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hts, hte, hins, hy, hsg, htq = (pin(a) for a in (w["t_start"], w["t_end"], w["instrument"], w["y"], w["sigma"], tq_h))
    hamp = None if w["amp"] is None else pin(w["amp"])
    hout = dict(mean=pin(np.empty((batch, N))), var=pin(np.empty((batch, N))), loglik=pin(np.empty(batch)),
                mean_query=pin(np.empty((batch, M))), var_query=pin(np.empty((batch, M))))

    def step_e2e():
        ev = ctx.smolgp_build_events_host(hts, hte, hins, w["n_inst"])
        ctx.smolgp_condition_host(ev, w["kernel"], hy, hsg, amp=hamp, t_query=htq, query_instrument=0, out=hout)
        ev.free()

    step_e2e()
    torch.cuda.synchronize()
    evs2 = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); step_e2e(); b.record()
        evs2.append((a, b))
    torch.cuda.synchronize()
    ms_e2e = sum(a.elapsed_time(b) for a, b in evs2) / args.steps
    clocks = sampler.stop()
    hbm_gbs, hbm_src = hbm_peak_gbs()
    # algorithmic bytes of the query kernel: per query the two stored states it combines (filtered state of the event
    # before, adjoint of the event after: "all 2N states"), its two step records, 8 B in, 16 B out
    stride_bytes = None
    qbytes = 2 * 8 * (n + n * n) + 16 + 8
    t_q = prof.get("k_query", (0.0, 1))[0]
    roofline = {"bound": "hbm", "kernel": "k_query", "achieved": batch * M * qbytes / (t_q * 1e-3) / 1e9 if t_q else None,
                "peak": hbm_gbs, "unit": "GB/s", "frac": (batch * M * qbytes / (t_q * 1e-3) / 1e9 / hbm_gbs) if t_q else None, "traffic": None,
                "peak_source": hbm_src,
                "work_model": "per query: two stored states of n + n^2 doubles + 24 B (neighbouring queries share the states through L2, so achieved can exceed the DRAM peak)",
                "kernels_ms_per_step": {k: v[0] for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])}}
    # CPU baseline: the oracle's Algorithm 1 on a bounded sample (first ns exposures, mult x ns queries inside their span)
    import oracle
    oracle.build()
    ns = min(N, 400)
    sl = slice(0, ns)
    yy = w["y"][0, sl] if w["y"].ndim == 2 else w["y"][sl]
    kern = w["kernel"] if w.get("amp") is None else [dict(k, sigma=k["sigma"] * float(w["amp"][0])) for k in w["kernel"]]
    tq_s = np.linspace(float(w["t_start"][sl].min()), float(w["t_end"][sl].max()), int(args.predict_mult * ns))
    tc = time.perf_counter()
    oracle.ssm(kern, w["n_inst"], w["t_start"][sl], w["t_end"][sl], w["instrument"][sl], yy, w["sigma"][sl],
               flags=oracle.FLAG_TWO_FILTER, tq=tq_s, query_inst=0, prec="f64")
    tc = time.perf_counter() - tc
    line = {"metric": "queries/sec for condition + predict at M = %g N (P:561)" % args.predict_mult, "value": batch * M / (ms * 1e-3), "unit": "queries/s",
            "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "predict: " + cfgname, "N": N, "events": 2 * N, "M": M, "batch": batch, "state_dim": n,
                       "path": "a1-a6 + a7 (Algorithm 1 at M uniform query times)", "l2": "flushed (512 MiB write) between timed iterations",
                       "plan": ctx.plan_info()},
            "events_per_s": batch * 2 * N / (ms * 1e-3),
            "peak_device_bytes": int(peak_bytes),
            "e2e": {"value": batch * M / (ms_e2e * 1e-3), "unit": "queries/s", "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": int(hts.nbytes + hte.nbytes + hins.nbytes + hy.nbytes + hsg.nbytes + htq.nbytes + (0 if hamp is None else hamp.nbytes)),
                    "d2h_bytes_per_step": int(sum(v.nbytes for v in hout.values()))},
            "gpu_launches": int(launches), "specialised": "jit=1" in ctx.plan_info(), "jit_log": ctx.jit_log(), "clocks": clocks, "roofline": roofline,
            "cpu_baseline": {"value": tq_s.size / tc, "unit": "queries/s", "cores": 1, "kind": "oracle",
                             "sample": "first %d exposures, %d queries, oracle fp64 build (filter + two-filter smoother + Algorithm 1), 1 thread, %.1f s" % (ns, tq_s.size, tc)}}
    print(json.dumps(line), flush=True)


CFG_NAMES = {"instant": "instantaneous samples (paper section 2), SHO + Matern-5/2 (Fig. 1 kernel), N=1e5 (K=1e5 events)",
             1: "cfg1 Matern-3/2 N=1e3", 2: "cfg2 SHO two instruments N=2e4",
             3: "cfg3 quasiperiodic Matern-3/2 x periodic(J=4), 3 overlapping instruments, n=21, N=1e5 (K=2e5 events)",
             4: "cfg4 joint multi-instrument n=17 N=1e6", 5: "cfg5 batched 4096 x N=2048, n=7"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", default="3", help="BASELINE.json config (1-5; 3 = the headline N=1e5) or `instant` (section-2 instantaneous data, SURVEY 8(f) item 3)")
    ap.add_argument("--workload", default="condition", choices=["condition", "predict"],
                    help="condition = the headline (rows a1-a6); predict = condition + prediction at --predict-mult x N query times (row a7)")
    ap.add_argument("--form", default="cov", choices=["cov", "sqrt"],
                    help="cov = covariance form (default, the headline); sqrt = square-root (Cholesky-factor) form of the chunk recursions, one chunk per series "
                         "(SURVEY 8(f) item 1; meant for the batched config 5)")
    ap.add_argument("--predict-mult", type=float, default=100.0, help="queries per exposure of the predict workload (the paper uses M = 100 N, P:561)")
    args = ap.parse_args()
    args.config = args.config if args.config == "instant" else int(args.config)
    w = W.make(args.config)
    if args.impl == "reference":
        run_reference(args, w, CFG_NAMES[args.config])
    elif args.workload == "predict":
        run_predict(args, w, CFG_NAMES[args.config])
    else:
        run_cuda(args, w, CFG_NAMES[args.config])


if __name__ == "__main__":
    main()
