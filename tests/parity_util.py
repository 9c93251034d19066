"""Helpers shared by the GPU parity tests: tolerances (SURVEY reading c13)
and the oracle-side reference run.  Nothing here touches the CUDA path."""
import numpy as np

LL_RTOL = 1e-9    # north_star: relative 1e-9 on the log-likelihood
POST_RTOL = 1e-8  # north_star: relative 1e-8 on posterior mean and variance


def prior_sd(oracle, w, idx=None, series=None):
    """sqrt(k_FF,nn): prior standard deviation of each exposure average (of the exposures `idx`, default
    all) -- the floor of the mean's relative error (reading R13 / c13: a mean can be arbitrarily close to
    zero).  A per-series amplitude scales it (k_p = amp_p^2 k, reading R15)."""
    ts, te, inst = w["t_start"], w["t_end"], w["instrument"]
    idx = np.arange(ts.size) if idx is None else np.asarray(idx)
    out = np.empty(idx.size)
    # the diagonal of the dense kernel, one exposure at a time (O(N), uses the oracle's definition)
    for o, i in enumerate(idx):
        out[o] = oracle.kff(w["kernel"], ts[i:i + 1], te[i:i + 1], inst[i:i + 1])[0, 0]
    sd = np.sqrt(out)
    if series is not None and w.get("amp") is not None:
        sd = sd * float(w["amp"][series])
    return sd


def reference(oracle, w, series=None, want_post=True):
    """long-double sequential oracle (two-filter smoother, idle-z zeroing: readings R6, R7) on
    series `series` of workload w (None = the only series)."""
    y = w["y"] if series is None else w["y"][series]
    kern = w["kernel"]
    if series is not None and w.get("amp") is not None:
        a = float(w["amp"][series])
        kern = [dict(k, sigma=k["sigma"] * a) for k in kern]
    return oracle.ssm(kern, w["n_inst"], w["t_start"], w["t_end"], w["instrument"], y, w["sigma"],
                      flags=oracle.FLAG_IDLE_ZERO | oracle.FLAG_TWO_FILTER, want_post=want_post)


def errors(ref, got_ll, got_mean=None, got_var=None, floor=None):
    """returns dict of the scaled errors that the tolerances bound; floor = prior_sd(...) (reading R13),
    required whenever a mean is compared"""
    out = dict(ll=abs(got_ll - ref["loglik"]) / abs(ref["loglik"]))
    if got_mean is not None:
        assert floor is not None, "the mean's error is scaled by |ref| + prior sd of the exposure average (R13)"
        fl = floor
        out["mean"] = float(np.max(np.abs(got_mean - ref["mean"]) / (np.abs(ref["mean"]) + fl)))
        out["var"] = float(np.max(np.abs(got_var - ref["var"]) / ref["var"]))
    return out
