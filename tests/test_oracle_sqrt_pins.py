"""Pins of the oracle's square-root (Cholesky-factor) sequential pass, oracle_ssm_sqrt (the
paper's remedy for the conditioning of the covariance recursions).  The paper prints no algorithm for
it: what it must compute is the posterior the dense definition (Eq. 2.4; Eq. 2.26) and the
covariance-form sequential passes give, so those are the pins.  CPU only."""
import numpy as np
import pytest

from test_oracle_inference_pins import CASES, tiny


@pytest.mark.parametrize("cfg,N", CASES)
def test_sqrt_form_equals_dense_gp(oracle, cfg, N):
    """every model structure of the five configs + the Fig. 2 (back-to-back, exact ties) and Fig. 3 (overlapping
    instruments) layouts: likelihood and posterior of the dense integrated GP"""
    kern, ni, ts, te, inst, y, sig = tiny(cfg, N)
    d = oracle.dense(kern, ts, te, inst, y, sig)
    s = oracle.ssm_sqrt(kern, ni, ts, te, inst, y, sig)
    prior_sd = np.sqrt(np.diag(oracle.kff(kern, ts, te, inst)))
    assert s["loglik"] == pytest.approx(d["loglik"], rel=1e-13)
    assert np.max(np.abs(s["mean"] - d["mean"]) / (np.abs(d["mean"]) + prior_sd)) < 1e-12
    assert np.max(np.abs(s["var"] / d["var"] - 1)) < 1e-12


@pytest.mark.parametrize("cfg,N", [(3, 1500), (4, 1500), (5, 1024)])
def test_sqrt_form_equals_covariance_form_beyond_dense_sizes(oracle, cfg, N):
    """against the covariance-form passes (two-filter backward pass, idle integral states zeroed: readings R6, R7),
    both in 80-bit arithmetic, at sizes where the recursions have run for thousands of events"""
    kern, ni, ts, te, inst, y, sig = tiny(cfg, N)
    a = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=3)
    s = oracle.ssm_sqrt(kern, ni, ts, te, inst, y, sig)
    assert s["loglik"] == pytest.approx(a["loglik"], rel=1e-14)
    assert np.max(np.abs(s["mean"] - a["mean"])) < 1e-11 * np.abs(y).max()
    assert np.max(np.abs(s["var"] / a["var"] - 1)) < 1e-11


def test_sqrt_form_does_not_depend_on_the_z_prior(oracle):
    """the integral-state block of P0 'will not matter'"""
    kern, ni, ts, te, inst, y, sig = tiny(4, 80)
    ref = oracle.ssm_sqrt(kern, ni, ts, te, inst, y, sig, zprior=1.0)
    for zp in (0.0, 1e6):
        s = oracle.ssm_sqrt(kern, ni, ts, te, inst, y, sig, zprior=zp)
        assert s["loglik"] == pytest.approx(ref["loglik"], rel=1e-13)
        np.testing.assert_allclose(s["mean"], ref["mean"], rtol=0, atol=1e-10)
        np.testing.assert_allclose(s["var"], ref["var"], rtol=1e-9)


def test_sqrt_form_is_the_better_conditioned_one_in_double_precision(oracle):
    """the reason the paper names it: in plain fp64 the factor form loses fewer digits than the covariance
    form against the 80-bit reference -- the joint 4-instrument model (config 4) by orders of magnitude, the
    quasi-periodic model (config 3) by a smaller factor"""
    for cfg, N, gain in ((4, 3000, 100.0), (3, 3000, 2.0)):
        kern, ni, ts, te, inst, y, sig = tiny(cfg, N)
        ref = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=3, prec="f80")
        cov = oracle.ssm(kern, ni, ts, te, inst, y, sig, flags=3, prec="f64")
        fac = oracle.ssm_sqrt(kern, ni, ts, te, inst, y, sig, prec="f64")
        e_cov = np.max(np.abs(cov["var"] / ref["var"] - 1))
        e_fac = np.max(np.abs(fac["var"] / ref["var"] - 1))
        assert e_fac < 1e-10 and e_fac * gain < e_cov, (cfg, e_fac, e_cov)
        assert fac["loglik"] == pytest.approx(ref["loglik"], rel=1e-12)


def test_sqrt_form_rejects_what_the_covariance_form_rejects(oracle):
    ts = np.array([0.0, 5.0]); te = np.array([8.0, 9.0])
    kern, ni, *_ = tiny(1, 10)
    with pytest.raises(RuntimeError, match="rc=-2"):   # one instrument overlapping itself
        oracle.ssm_sqrt(kern, 1, ts, te, np.zeros(2, np.int32), np.zeros(2), np.ones(2))
