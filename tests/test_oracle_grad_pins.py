"""Pin of the oracle's log-likelihood gradient: central differences of the pinned
sequential likelihood against the dense route's ANALYTIC derivative  dL/dtheta = 1/2 tr((alpha alpha^T - C^-1) dC/dtheta),
with dC/dsigma in closed form (K_c is proportional to sigma_c^2) and dC/d(other) from the dense integrated kernel."""
import numpy as np

from paper_2601_02527_b200 import workloads as W


def _trace_formula(C, y, dC):
    alpha = np.linalg.solve(C, y)
    return 0.5 * (alpha @ dC @ alpha - np.trace(np.linalg.solve(C, dC)))


def test_gradient_matches_the_dense_analytic_derivative(oracle):
    for cfg in (2, 4, 3):
        w = W.make(cfg, N=60)
        kern = w["kernel"]
        ts, te, inst, y, sg = w["t_start"], w["t_end"], w["instrument"], w["y"], w["sigma"]
        fn = lambda k: oracle.ssm(k, w["n_inst"], ts, te, inst, y, sg, flags=oracle.FLAG_TWO_FILTER, want_post=False)["loglik"]
        g = oracle.loglik_grad(kern, fn)
        K = oracle.kff(kern, ts, te, inst)
        C = K + np.diag(sg ** 2)
        for c, comp in enumerate(kern):
            # amplitude: K = sum_c K_c, K_c = sigma_c^2 (...)  =>  dC/dsigma_c = 2 K_c / sigma_c, exactly
            Kc = oracle.kff([comp], ts, te, inst)
            exact = _trace_formula(C, y, 2 * Kc / comp["sigma"])
            assert abs(g[c, 0] - exact) <= 1e-7 * max(1.0, abs(exact)), (cfg, c, g[c, 0], exact)
            # the other parameters: dC/dtheta by differences of the dense integrated kernel (an independent route)
            for p in range(1, oracle.FAMILY_PARAMS[int(comp["family"])]):
                th, h = comp[oracle.PARAMS[p]], 1e-4
                Kp = oracle.kff([dict(comp, **{oracle.PARAMS[p]: th * (1 + h)})], ts, te, inst)
                Km = oracle.kff([dict(comp, **{oracle.PARAMS[p]: th * (1 - h)})], ts, te, inst)
                approx = _trace_formula(C, y, (Kp - Km) / (2 * h * th))
                assert abs(g[c, p] - approx) <= 1e-5 * max(1.0, abs(approx)), (cfg, c, p, g[c, p], approx)
