"""Accuracy of the CUDA path on config 3 at full size (N = 1e5, n = 21) over scan plans, against the
values stored by tests/golden/make_golden.py (long-double oracle, 2000+ sampled exposures).

    python tests/accuracy_sweep.py

Prints markdown table rows: plan | ms | loglik rel | mean (scaled) | variance max rel | variance p99."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    from paper_2601_02527_b200 import binding as B, workloads as W
    rows = [l.split() for l in open(os.path.join(ROOT, "tests", "golden", "cfg3_full.txt")) if not l.startswith("#")]
    ll = float(rows[0][0])
    idx = np.array([int(r[0]) for r in rows[1:]])
    mean = np.array([float(r[1]) for r in rows[1:]])
    var = np.array([float(r[2]) for r in rows[1:]])
    w = W.make(3)
    dev = torch.device("cuda:0")
    ctx = B.Context(0)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    y, sg = torch.tensor(w["y"], device=dev), torch.tensor(w["sigma"], device=dev)
    plans = [(c, g) for c in (0, 68, 100, 200, 300) for g in (0, 2, 8)] + [(0, 64), (1 << 40, 0)]
    for chunk, group in plans:
        if chunk >= 1 << 40 and "--sequential" not in sys.argv:
            continue  # the one-chunk plan takes ~15 s on the GPU
        ctx.set_option("chunk", chunk)
        ctx.set_option("group", group)
        out = ctx.smolgp_condition(ev, w["kernel"], y, sg)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); ctx.smolgp_condition(ev, w["kernel"], y, sg, out=out); b.record(); torch.cuda.synchronize()
        m, v, l = out["mean"].cpu().numpy()[0][idx], out["var"].cpu().numpy()[0][idx], float(out["loglik"][0])
        rel = np.abs(v - var) / var
        em = np.max(np.abs(m - mean) / (np.abs(mean) + np.sqrt(var) + 1e-3))
        name = "%s, fan-in %s" % ("auto chunk" if chunk == 0 else ("one chunk" if chunk >= 1 << 40 else "chunk %d" % chunk),
                                  "auto" if group == 0 else group)
        print("| %s | %.2f | %.1e | %.1e | %.2e | %.2e |" % (name, a.elapsed_time(b), abs(l - ll) / abs(ll), em, rel.max(),
                                                          np.quantile(rel, 0.99)), flush=True)


if __name__ == "__main__":
    main()
