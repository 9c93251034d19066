"""Writes the stored expected values of the full-size parity tests.  Calls ONLY the CPU oracle
(oracle/, long-double build) on the seeded workloads of paper_2601_02527_b200/workloads.py:

    python tests/golden/make_golden.py [3] [4]

cfgN_full.txt: line 1 = log-likelihood; then `index mean var` for a fixed sample of exposures
(every exposure of the first and last 200, plus 2000 drawn with numpy default_rng(12345)).
Config 3 takes ~1 min, config 4 (N = 1e6) ~10 min of one core."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2601_02527_b200 import workloads as W  # noqa: E402


def sample_indices(N):
    rng = np.random.default_rng(12345)
    return np.unique(np.concatenate([np.arange(200), np.arange(N - 200, N), rng.integers(0, N, 2000)]))


def main():
    oracle.build()
    for cfg in [int(a) for a in sys.argv[1:]] or [3, 4]:
        w = W.make(cfg)
        ref = oracle.ssm(w["kernel"], w["n_inst"], w["t_start"], w["t_end"], w["instrument"], w["y"], w["sigma"],
                         flags=oracle.FLAG_IDLE_ZERO | oracle.FLAG_TWO_FILTER)
        idx = sample_indices(w["t_start"].size)
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg%d_full.txt" % cfg)
        with open(path, "w") as f:
            f.write("# oracle.ssm long double, two-filter smoother, workloads.make(%d); written by make_golden.py\n" % cfg)
            f.write("%.17g\n" % ref["loglik"])
            for i in idx:
                f.write("%d %.17g %.17g\n" % (i, ref["mean"][i], ref["var"][i]))
        print("wrote", path, flush=True)


if __name__ == "__main__":
    main()
