"""Pins of the oracle's instantaneous-data routes (paper section 2): the dense
definition against numpy on the (already pinned) scalar kernel, the section-2 sequential algorithm against the
dense definition (the paper's Fig. 1 claim: the state-space model equals the GP on instantaneous data to
machine precision), and the exposure-integrated oracle converging to it as the exposures shrink."""
import numpy as np
import pytest

from paper_2601_02527_b200 import workloads as W

KERNELS = {
    "fig1": [W.comp(W.SHO, 1.0, 2 * np.pi / 300.0, 2.0), W.comp(W.MATERN52, 0.7, 900.0)],   # Fig. 1: SHO + Matern-5/2
    "m32": [W.comp(W.MATERN32, 1.3, 600.0)],
    "masked": [W.comp(W.SHO, 1.0, 2 * np.pi / 330.0, 10.0), W.comp(W.MATERN32, 0.5, 900.0, inst_mask=2)],
    "qp": [W.comp(W.MATERN32_X_PERIODIC, 1.0, 4000.0, 9000.0, 1.0, order=2)],
}


def _data(rng, kern, N, ninst, span=20000.0, ties=False):
    t = np.sort(rng.uniform(0, span, N))
    if ties:
        t[1::7] = t[0::7][: t[1::7].size]      # exact ties, also between instruments
    inst = rng.integers(0, ninst, N).astype(np.int32)
    sigma = rng.uniform(0.1, 0.4, N)
    y = W.synth_y(rng, kern, t, t + 1e-9, inst, sigma)   # spectral synthesis at (essentially) instantaneous samples
    return t, inst, y, sigma


@pytest.mark.parametrize("name", sorted(KERNELS))
def test_dense_instant_against_numpy_on_the_pinned_kernel(oracle, name):
    rng = np.random.default_rng(3)
    kern = KERNELS[name]
    ninst = 2 if name == "masked" else 1
    t, inst, y, sigma = _data(rng, kern, 70, ninst)
    tq = np.concatenate([rng.uniform(-500, 20500, 15), t[:3]])
    got = oracle.dense_instant(kern, t, inst, y, sigma, tq=tq, query_inst=ninst - 1)
    K = np.empty((70, 70))
    for a in range(ninst):
        for b in range(ninst):
            ia, ib = np.nonzero(inst == a)[0], np.nonzero(inst == b)[0]
            K[np.ix_(ia, ib)] = oracle.kernel(kern, a, b, np.abs(t[ia][:, None] - t[ib][None, :]).ravel()).reshape(ia.size, ib.size)
    Cm = K + np.diag(sigma ** 2)
    alpha = np.linalg.solve(Cm, y)
    ll = -0.5 * (y @ alpha + np.linalg.slogdet(Cm)[1] + 70 * np.log(2 * np.pi))
    assert abs(got["loglik"] - ll) <= 1e-11 * abs(ll)
    np.testing.assert_allclose(got["mean"], K @ alpha, rtol=1e-9, atol=1e-11)
    np.testing.assert_allclose(got["var"], np.diag(K - K @ np.linalg.solve(Cm, K)), rtol=1e-7, atol=1e-10)
    Ks = np.stack([oracle.kernel(kern, ninst - 1, int(q), np.abs(tq - t[i:i + 1])) for i, q in enumerate(inst)], axis=1)
    np.testing.assert_allclose(got["mq"], Ks @ alpha, rtol=1e-9, atol=1e-11)
    k0 = oracle.kernel(kern, ninst - 1, ninst - 1, np.zeros(1))[0]
    np.testing.assert_allclose(got["vq"], k0 - np.einsum("qi,iq->q", Ks, np.linalg.solve(Cm, Ks.T)), rtol=1e-7, atol=1e-10)


@pytest.mark.parametrize("ties", [False, True])
@pytest.mark.parametrize("name", sorted(KERNELS))
def test_ssm_instant_equals_the_dense_definition(oracle, name, ties):
    """Fig. 1's claim: the section-2 state-space algorithm reproduces the GP on instantaneous data"""
    rng = np.random.default_rng(5)
    kern = KERNELS[name]
    ninst = 2 if name == "masked" else 1
    t, inst, y, sigma = _data(rng, kern, 90, ninst, ties=ties)
    tq = np.concatenate([rng.uniform(-800, 20800, 25), t[:2], [t.min() - 1.0, t.max() + 1.0]])
    for qi in range(ninst):
        a = oracle.dense_instant(kern, t, inst, y, sigma, tq=tq, query_inst=qi)
        b = oracle.ssm_instant(kern, ninst, t, inst, y, sigma, tq=tq, query_inst=qi)
        assert abs(a["loglik"] - b["loglik"]) <= 1e-12 * abs(a["loglik"])
        np.testing.assert_allclose(b["mean"], a["mean"], rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(b["var"], a["var"], rtol=1e-8, atol=1e-12)
        np.testing.assert_allclose(b["mq"], a["mq"], rtol=1e-9, atol=1e-11)
        np.testing.assert_allclose(b["vq"], a["vq"], rtol=1e-8, atol=1e-11)


def test_integrated_oracle_converges_to_the_instantaneous_one(oracle):
    """exposures of length delta centred on the sample times: the integrated model tends to the instantaneous
    one with second order in delta / ell (reduction test)"""
    rng = np.random.default_rng(8)
    kern = KERNELS["m32"]
    t, inst, y, sigma = _data(rng, kern, 60, 1, span=40000.0)
    t = 600.0 * np.arange(60) + 300.0 * rng.uniform(0, 1, 60)   # well separated: no self-overlap for delta up to 60 s
    ref = oracle.ssm_instant(kern, 1, t, inst, y, sigma)
    gaps = []
    for delta in (60.0, 6.0, 0.6):
        got = oracle.ssm(kern, 1, t - delta / 2, t + delta / 2, inst, y, sigma, flags=oracle.FLAG_TWO_FILTER)
        gaps.append(abs(got["loglik"] - ref["loglik"]) / abs(ref["loglik"]))
    assert gaps[0] < 1e-2 and gaps[1] < 2e-2 * gaps[0] and gaps[2] < 2e-2 * gaps[1], gaps


def test_float64_build_agrees_with_long_double(oracle):
    rng = np.random.default_rng(9)
    kern = KERNELS["fig1"]
    t, inst, y, sigma = _data(rng, kern, 200, 1)
    a = oracle.ssm_instant(kern, 1, t, inst, y, sigma)
    b = oracle.ssm_instant(kern, 1, t, inst, y, sigma, prec="f64")
    assert abs(a["loglik"] - b["loglik"]) <= 1e-10 * abs(a["loglik"])
    np.testing.assert_allclose(b["mean"], a["mean"], rtol=1e-7, atol=1e-9)
