"""Pins of the oracle's dense integrated-GP solver and of its sequential state-space filter /
smoother / predictor to what the paper and the mathematics fix.  CPU only."""
import numpy as np
import pytest
from scipy import integrate

from paper_2601_02527_b200 import workloads as W
from test_oracle_model_pins import k_matern, k_sho


# ---------------------------------------------------------------------------------------------
# dense kernel (Eq. 3.1) against the printed celerite closed forms and 2-D quadrature
# ---------------------------------------------------------------------------------------------
def kff_celerite(a, b, c, d, delta, lag):
    """A3-A6, A8, A11, typed from the paper. lag >= 0."""
    C1 = a * c * c - a * d * d + 2 * b * c * d
    C2 = b * c * c - b * d * d - 2 * a * c * d
    den = (delta * (c * c + d * d)) ** 2
    ch, sh = np.cosh(c * delta), np.sinh(c * delta)
    A = (2 * C1 * (ch * np.cos(d * delta) - 1) - 2 * C2 * sh * np.sin(d * delta)) / den
    B = (2 * C2 * (ch * np.cos(d * delta) - 1) + 2 * C1 * sh * np.sin(d * delta)) / den
    if lag == 0:
        return 2 * ((a * c + b * d) * (c * c + d * d) * delta - C1
                    + np.exp(-c * delta) * (C1 * np.cos(d * delta) + C2 * np.sin(d * delta))) / den
    base = np.exp(-c * lag) * (A * np.cos(d * lag) + B * np.sin(d * lag))
    if lag >= delta:
        return base
    r = delta - lag
    return base + 2 * ((a * c + b * d) * (c * c + d * d) * r - C1 * np.sinh(c * r) * np.cos(d * r)
                       + C2 * np.cosh(c * r) * np.sin(d * r)) / den


def kff_real_term(a, c, delta, lag):
    """A12, the b = d = 0 case."""
    pre = 2 * a * np.exp(-c * lag) / (c * delta) ** 2
    if lag == 0:
        return pre * (np.exp(-c * delta) - 1 + c * delta)
    if lag <= delta:
        return pre * ((c * (delta - lag) - np.sinh(c * (delta - lag))) * np.exp(c * lag) + np.cosh(c * delta) - 1)
    return pre * (np.cosh(c * delta) - 1)


@pytest.mark.parametrize("w0,Q,s", [(2 * np.pi / 330.0, 10.0, 1.3), (0.02, 0.8, 0.7), (0.3, 3.0, 1.0)])
def test_kff_sho_matches_celerite_closed_forms(oracle, w0, Q, s):
    delta = 55.0
    eta = np.sqrt(1 - 1 / (4 * Q * Q))
    a, b, c, d = s * s, s * s / (2 * eta * Q), w0 / (2 * Q), eta * w0          # A1 vs (Kernel)
    lags = np.array([0.0, 10.0, 40.0, 55.0, 60.0, 200.0, 1000.0])
    ts = np.concatenate([[0.0], lags[1:]])
    K = oracle.kff([W.comp(W.SHO, s, w0, Q)], ts, ts + delta, np.zeros(ts.size, np.int32))
    for j, lag in enumerate(lags):
        ref = kff_celerite(a, b, c, d, delta, lag)
        assert K[0, j] == pytest.approx(ref, rel=1e-9, abs=1e-11 * s * s), (lag, K[0, j], ref)


def test_kff_real_term_A12(oracle):
    """an overdamped SHO is the sum of two real terms (Kernel, Q < 1/2)."""
    w0, Q, s, delta = 0.05, 0.3, 0.9, 30.0
    eta = np.sqrt(1 / (4 * Q * Q) - 1)
    A = 1 / (2 * eta * Q)
    terms = [(s * s * (1 + A) / 2, w0 / (2 * Q) - eta * w0), (s * s * (1 - A) / 2, w0 / (2 * Q) + eta * w0)]
    lags = np.array([0.0, 12.0, 30.0, 45.0, 300.0])
    ts = np.concatenate([[0.0], lags[1:]])
    K = oracle.kff([W.comp(W.SHO, s, w0, Q)], ts, ts + delta, np.zeros(ts.size, np.int32))
    for j, lag in enumerate(lags):
        ref = sum(kff_real_term(a, c, delta, lag) for a, c in terms)
        assert K[0, j] == pytest.approx(ref, rel=1e-10)


def test_kff_quadrature_unequal_overlapping_exposures(oracle):
    """Eq. 3.1 by brute-force 2-D quadrature, exposures of different lengths, nested,
    partially overlapping, touching and disjoint; two instruments with a private component."""
    kern = [W.comp(W.MATERN52, 1.0, 400.0), W.comp(W.MATERN32, 0.6, 150.0, inst_mask=0b10)]
    ts = np.array([0.0, 20.0, 100.0, 130.0, 160.0, 900.0])
    te = np.array([100.0, 60.0, 160.0, 300.0, 200.0, 1000.0])
    inst = np.array([0, 1, 0, 1, 0, 1], np.int32)
    K = oracle.kff(kern, ts, te, inst)

    def k(tau, i, j):
        v = k_matern(tau, 400.0, 1.0, 2.5)
        if inst[i] == 1 and inst[j] == 1:
            v = v + k_matern(tau, 150.0, 0.6, 1.5)
        return v
    for i, j in [(0, 1), (0, 2), (1, 3), (3, 4), (2, 4), (0, 5), (3, 3), (1, 1), (3, 5)]:
        # split at the kink |t - t'| = 0 by integrating the inner variable piecewise
        def inner(t):
            pts = [p for p in (t,) if ts[j] < p < te[j]]
            return integrate.quad(lambda u: k(abs(t - u), i, j), ts[j], te[j], points=pts or None,
                                  epsabs=0, epsrel=1e-12)[0]
        brk = [p for p in (ts[j], te[j]) if ts[i] < p < te[i]]
        val = integrate.quad(inner, ts[i], te[i], points=brk or None, epsabs=0, epsrel=1e-11)[0]
        ref = val / ((te[i] - ts[i]) * (te[j] - ts[j]))
        assert K[i, j] == pytest.approx(ref, rel=2e-10), (i, j)
    assert np.all(K == K.T) and np.linalg.eigvalsh(K).min() > 0


# ---------------------------------------------------------------------------------------------
# tiny workloads with the structure of every config
# ---------------------------------------------------------------------------------------------
def tiny(cfg, N, seed=None):
    w = W.make(cfg, N=N, batch=2 if cfg == 5 else None, seed=seed)
    kern, y = w["kernel"], w["y"]
    if w["batch"] is not None:
        kern = [dict(k, sigma=k["sigma"] * w["amp"][1]) for k in kern]
        y = y[1]
    return kern, w["n_inst"], w["t_start"], w["t_end"], w["instrument"], y, w["sigma"]


CASES = [(1, 120), (2, 90), (3, 70), (4, 80), (5, 100), ("fig2", 60), ("fig3", 90)]


@pytest.mark.parametrize("cfg,N", CASES)
def test_dense_solver_matches_numpy_linear_algebra(oracle, cfg, N):
    """Eq. 2.4 and the Gaussian log density (P:258 via the chain rule 2.24) with numpy's
    LAPACK on the oracle's own K: pins the Cholesky / substitution / loglik code."""
    kern, ni, ts, te, inst, y, sig = tiny(cfg, N)
    K = oracle.kff(kern, ts, te, inst)
    Cm = K + np.diag(sig ** 2)
    alpha = np.linalg.solve(Cm, y)
    ll = -0.5 * (y @ alpha + np.linalg.slogdet(Cm)[1] + N * np.log(2 * np.pi))
    mean = K @ alpha
    var = np.diag(K - K @ np.linalg.solve(Cm, K))
    d = oracle.dense(kern, ts, te, inst, y, sig)
    assert d["loglik"] == pytest.approx(ll, rel=1e-10)
    np.testing.assert_allclose(d["mean"], mean, rtol=0, atol=1e-8 * np.abs(y).max())
    np.testing.assert_allclose(d["var"], var, rtol=1e-5, atol=1e-10)   # numpy's fp64 is the loose side here


@pytest.mark.parametrize("cfg,N", CASES)
@pytest.mark.parametrize("flags", [0, 2, 3])
def test_ssm_equals_dense_gp(oracle, cfg, N, flags):
    """The paper's central claim: the augmented SSM gives exactly the dense
    integrated GP's likelihood and posterior.  flags: 0 = textbook RTS (Eq. 3.16), 2 = two-filter
    backward pass, 3 = two-filter + zeroing of idle integral states (reading R6)."""
    kern, ni, ts, te, inst, y, sig = tiny(cfg, N)
    d = oracle.dense(kern, ts, te, inst, y, sig)
    s = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=flags)
    prior_sd = np.sqrt(np.diag(oracle.kff(kern, ts, te, inst)))
    assert s["loglik"] == pytest.approx(d["loglik"], rel=1e-13)
    vtol = 1e-9 if flags == 0 else 1e-12     # textbook RTS inverts a near-singular P^- after resets
    assert np.max(np.abs(s["mean"] - d["mean"]) / (np.abs(d["mean"]) + prior_sd)) < vtol
    assert np.max(np.abs(s["var"] / d["var"] - 1)) < vtol


def test_f64_oracle_close_to_f80(oracle):
    kern, ni, ts, te, inst, y, sig = tiny(2, 200)
    a = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=2, prec="f80")
    b = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=2, prec="f64")
    assert b["loglik"] == pytest.approx(a["loglik"], rel=1e-11)
    assert np.max(np.abs(b["var"] / a["var"] - 1)) < 1e-7
    assert np.max(np.abs(b["mean"] - a["mean"])) < 1e-9


def test_invariance_to_z_prior_and_idle_zeroing(oracle):
    """the integral-state block of P0 'will not matter'."""
    kern, ni, ts, te, inst, y, sig = tiny(4, 80)
    ref = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=2, zprior=1.0)
    for zp, fl in [(0.0, 2), (1e6, 2), (1.0, 3), (1e6, 0)]:
        s = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=fl, zprior=zp)
        assert s["loglik"] == pytest.approx(ref["loglik"], rel=1e-13)
        np.testing.assert_allclose(s["mean"], ref["mean"], rtol=0, atol=1e-10)
        np.testing.assert_allclose(s["var"], ref["var"], rtol=1e-9)


def test_exact_ties_and_input_order(oracle):
    """simultaneous events of different instruments (start/start, end/start, end/end) and a
    permuted input order give the dense GP's answer (reading R5: ends sort before starts)."""
    kern = [W.comp(W.SHO, 1.0, 2 * np.pi / 330.0, 10.0)]
    ts = np.array([0.0, 0.0, 60.0, 100.0, 120.0, 200.0, 260.0])
    te = np.array([55.0, 100.0, 120.0, 180.0, 180.0, 260.0, 300.0])
    inst = np.array([0, 1, 0, 1, 0, 1, 0], np.int32)
    rng = np.random.default_rng(5)
    y, sig = rng.standard_normal(7), np.full(7, 0.25)
    d = oracle.dense(kern, ts, te, inst, y, sig)
    s = oracle.ssm(kern, 2, ts, te, inst, y, sig, flags=3)
    assert s["loglik"] == pytest.approx(d["loglik"], rel=1e-13)
    np.testing.assert_allclose(s["mean"], d["mean"], atol=1e-13)
    np.testing.assert_allclose(s["var"], d["var"], rtol=1e-12)
    p = rng.permutation(7)
    s2 = oracle.ssm(kern, 2, ts[p], te[p], inst[p], y[p], sig[p], flags=3)
    assert s2["loglik"] == pytest.approx(s["loglik"], rel=1e-14)
    np.testing.assert_allclose(s2["mean"], s["mean"][p], atol=1e-14)


def test_same_instrument_overlap_rejected(oracle):
    kern = [W.comp(W.MATERN32, 1.0, 100.0)]
    ts, te = np.array([0.0, 40.0]), np.array([50.0, 90.0])
    with pytest.raises(RuntimeError, match="rc=-2"):
        oracle.ssm(kern, 1, ts, te, np.zeros(2, np.int32), np.zeros(2), np.ones(2))


def test_reduction_to_ordinary_gp_as_exposures_shrink(oracle):
    """delta -> 0: the integrated model tends to the ordinary GP K_ij = k(t_i - t_j) (P:19-23,
    Fig. 1), at second order in delta/ell."""
    rng = np.random.default_rng(3)
    N, ell = 40, 100.0
    t = np.cumsum(rng.uniform(12.0, 60.0, N))
    y, sig = rng.standard_normal(N), np.full(N, 0.1)
    Cm = k_matern(t[:, None] - t[None, :], ell, 1.0, 1.5) + np.diag(sig ** 2)
    ll0 = -0.5 * (y @ np.linalg.solve(Cm, y) + np.linalg.slogdet(Cm)[1] + N * np.log(2 * np.pi))
    kern = [W.comp(W.MATERN32, 1.0, ell)]
    gaps = []
    for delta in (10.0, 1.0, 0.1):
        s = oracle.ssm(kern, 1, t - delta / 2, t + delta / 2, np.zeros(N, np.int32), y, sig, flags=2)
        gaps.append(abs(s["loglik"] - ll0) / abs(ll0))
    assert gaps[0] > 50 * gaps[1] > 2500 * gaps[2] and gaps[2] < 1e-5
    assert 60 < gaps[0] / gaps[1] < 160 and 60 < gaps[1] / gaps[2] < 160


def test_instantaneous_sho_equals_ordinary_gp_limit(oracle):
    """the same reduction for the SHO kernel the paper works out (App. B)."""
    rng = np.random.default_rng(4)
    N, w0, Q = 30, 2 * np.pi / 330.0, 10.0
    t = np.cumsum(rng.uniform(5.0, 200.0, N))
    y, sig = rng.standard_normal(N), np.full(N, 0.2)
    Cm = k_sho(t[:, None] - t[None, :], w0, Q, 1.0) + np.diag(sig ** 2)
    ll0 = -0.5 * (y @ np.linalg.solve(Cm, y) + np.linalg.slogdet(Cm)[1] + N * np.log(2 * np.pi))
    d = 1e-2
    s = oracle.ssm([W.comp(W.SHO, 1.0, w0, Q)], 1, t - d / 2, t + d / 2, np.zeros(N, np.int32), y, sig, flags=2)
    assert s["loglik"] == pytest.approx(ll0, rel=1e-8)


@pytest.mark.parametrize("cfg,N", [(1, 60), (2, 60), (4, 60)])
@pytest.mark.parametrize("flags", [0, 2])
def test_query_prediction_matches_dense(oracle, cfg, N, flags):
    """Algorithm 1 (readings R8/R9): retrodiction, interpolation (inside exposures and in
    gaps, at event times) and extrapolation of the instantaneous latent equal the dense GP's."""
    kern, ni, ts, te, inst, y, sig = tiny(cfg, N)
    t0, t1 = ts.min(), te.max()
    rng = np.random.default_rng(9)
    tq = np.concatenate([[t0 - 500.0, t0 - 1.0], rng.uniform(t0, t1, 25), [ts[3], te[5]], [t1 + 1.0, t1 + 800.0]])
    for qi in range(ni):
        d = oracle.dense(kern, ts, te, inst, y, sig, tq=tq, query_inst=qi)
        s = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=flags, tq=tq, query_inst=qi)
        np.testing.assert_allclose(s["mq"], d["mq"], rtol=0, atol=1e-11)
        np.testing.assert_allclose(s["vq"], d["vq"], rtol=1e-10, atol=1e-13)


# ---------------------------------------------------------------------------------------------
# component-wise prediction (App. C.3, Eq. C10-C14): a VIRTUAL instrument (a mask bit
# >= n_inst that takes no data) selects H^m
# ---------------------------------------------------------------------------------------------
def test_component_wise_prediction(oracle):
    rng = np.random.default_rng(4)
    N = 40
    ts = np.sort(rng.uniform(0, 6000.0, N))
    te = ts + rng.uniform(20.0, 100.0, N)
    te[:-1] = np.minimum(te[:-1], ts[1:] - 1.0)
    inst = np.zeros(N, np.int32)
    w0, Q, s0, ell, s1 = 2 * np.pi / 330.0, 4.0, 1.1, 900.0, 0.7
    # both components are seen by instrument 0; bit 1 marks the SHO alone, bit 2 the Matern alone
    kern = [W.comp(W.SHO, s0, w0, Q, inst_mask=0b011), W.comp(W.MATERN52, s1, ell, inst_mask=0b101)]
    y, sig = rng.standard_normal(N), np.full(N, 0.25)
    tq = np.concatenate([[ts[0] - 200.0], rng.uniform(ts[0], te[-1], 12), [te[-1] + 300.0]])
    tot = oracle.dense(kern, ts, te, inst, y, sig, tq=tq, query_inst=0)
    parts = [oracle.dense(kern, ts, te, inst, y, sig, tq=tq, query_inst=v) for v in (1, 2)]
    # C12: the component means add up to the mean of the sum; the data likelihood is untouched
    np.testing.assert_allclose(parts[0]["mq"] + parts[1]["mq"], tot["mq"], rtol=0, atol=1e-12)
    assert parts[0]["loglik"] == tot["loglik"] == parts[1]["loglik"]
    # C13-C14 typed out independently: mu_m = k_m*^T C^-1 y, var_m = k_m(0) - k_m*^T C^-1 k_m*, with the
    # exposure average of the component's kernel by quadrature
    C = oracle.kff(kern, ts, te, inst) + np.diag(sig ** 2)
    a = np.linalg.solve(C, y)
    ks = [lambda tau: k_sho(tau, w0, Q, s0), lambda tau: k_matern(tau, ell, s1, 2.5)]
    for m in range(2):
        for qi in (0, 5, len(tq) - 1):
            col = np.array([integrate.quad(lambda u: ks[m](tq[qi] - u), ts[j], te[j], epsabs=0, epsrel=1e-12,
                                           points=[tq[qi]] if ts[j] < tq[qi] < te[j] else None)[0] / (te[j] - ts[j])
                            for j in range(N)])
            assert parts[m]["mq"][qi] == pytest.approx(col @ a, rel=1e-9, abs=1e-11)
            assert parts[m]["vq"][qi] == pytest.approx(ks[m](0.0) - col @ np.linalg.solve(C, col), rel=1e-8)
    # the sequential algorithm with H^m (C13-C14) agrees with the dense definition
    for v in (1, 2):
        s = oracle.ssm(kern, 1, ts, te, inst, y, sig, flags=2, tq=tq, query_inst=v)
        np.testing.assert_allclose(s["mq"], parts[v - 1]["mq"], rtol=0, atol=1e-11)
        np.testing.assert_allclose(s["vq"], parts[v - 1]["vq"], rtol=1e-10, atol=1e-13)
