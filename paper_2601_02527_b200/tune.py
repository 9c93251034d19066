"""Plan sweeps for one workload: times smolgp_condition (events pre-built, device pointers, CUDA events,
min of several runs) over the scan-plan knobs of smolgp_set_option, so that the automatic choices in
csrc/scan_host.cu can be checked against measurement on a given GPU.

    python -m paper_2601_02527_b200.tune --config 3 [--sweep group|top|chunks|jit|lanes|predict] [--reps 7]

Prints markdown table rows.  No oracle involved (accuracy sweeps: tests/accuracy_sweep.py)."""
import argparse

import numpy as np


def _timeit(torch, f, reps):
    f(); f(); torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); f(); b.record(); torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return min(ts)


def main():
    import torch
    from . import binding as B, workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--sweep", default="group", choices=["group", "top", "chunks", "jit", "lanes", "predict"])
    ap.add_argument("--reps", type=int, default=7)
    ap.add_argument("--predict-mult", type=int, default=10, help="queries per exposure for --sweep predict")
    args = ap.parse_args()
    dev = torch.device("cuda:0")
    ctx = B.Context(0)
    w = W.make(args.config)
    N, batch = w["t_start"].size, (w["batch"] or 1)
    K = 2 * N * batch
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    y, sg = torch.tensor(w["y"], device=dev), torch.tensor(w["sigma"], device=dev)
    amp = None if w["amp"] is None else torch.tensor(w["amp"], device=dev)
    out = ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp)
    sm = torch.cuda.get_device_properties(0).multi_processor_count

    def run(label):
        t = _timeit(torch, lambda: ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp, out=out), args.reps)
        ctx.profile(True)
        ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp, out=out)
        pr = ctx.profile_read()
        ctx.profile(False)
        ks = ", ".join("%s %.3f" % (k, v[0]) for k, v in sorted(pr.items(), key=lambda kv: -kv[1][0]) if v[0] >= 0.05)
        print("| %s | %.3f | %.3e | %s |" % (label, t, K / t * 1e3, ks), flush=True)

    print("config %d: N=%d batch=%d events=%d; columns: setting | ms (a2-a6) | events/s | kernels (ms)" % (args.config, N, batch, K))
    if args.sweep == "group":
        for g in (2, 3, 4, 6, 8, 16):
            ctx.set_option("group", g)
            run("group %d" % g)
    elif args.sweep == "top":
        for t in (2, 3, 4, 6, 8, 12, 16, 24):
            ctx.set_option("top", t)
            run("top %d" % t)
    elif args.sweep == "chunks":
        for per_sm in (0, 4, 6, 8, 10, 12, 16, 20):
            ctx.set_option("chunk", 0 if per_sm == 0 else -(-(2 * N) // (sm * per_sm)))
            run("automatic" if per_sm == 0 else "%d chunks/SM" % per_sm)
        ctx.set_option("chunk", 1 << 40)
        if batch > 1:
            run("one chunk per series")
    elif args.sweep == "jit":
        for j, name in ((-1, "generic kernels"), (1, "specialised kernels")):
            ctx.set_option("jit", j)
            run(name)
    elif args.sweep == "lanes":
        for lanes in (8, 16, 32):
            ctx.set_option("lanes", lanes)
            run("lanes %d (forced if >= needed)" % lanes)
    else:
        M = args.predict_mult * N
        tq = torch.tensor(np.sort(np.random.default_rng(1).uniform(w["t_start"].min(), w["t_end"].max(), M)), device=dev)
        o2 = ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp, t_query=tq)
        t = _timeit(torch, lambda: ctx.smolgp_condition(ev, w["kernel"], y, sg, amp=amp, t_query=tq, out=o2), 3)
        print("| condition + predict, M = %d x N = %d | %.3f | %.3e queries/s | |" % (args.predict_mult, M, t, M * batch / t * 1e3))
    if ctx.jit_log():
        print("jit log:", ctx.jit_log()[:500])


if __name__ == "__main__":
    main()
