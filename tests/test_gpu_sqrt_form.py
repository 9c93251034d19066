"""GPU parity of the square-root (Cholesky-factor) form of the whole scan (option "form" = 1; SURVEY 8(f) item 1, P:535,
P:557; csrc/chunk_sqrt.cuh, csrc/dense_sqrt.cuh) against the long-double oracle: same bars as the covariance form
(loglik 1e-9, posterior 1e-8), on every model structure and every scan plan (chunk lengths, fan-ins, the sequential
plan); plus what the form is for -- fewer digits lost, with no compensated product anywhere on its path."""
import numpy as np
import pytest

from paper_2601_02527_b200 import workloads as W
import parity_util as PU

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2601_02527_b200 import binding as B
    c = B.Context(0)
    yield c
    c.close()


def _golden(cfg):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg%d_full.txt" % cfg)
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    return float(rows[0][0]), np.array([int(r[0]) for r in rows[1:]]), np.array([float(r[1]) for r in rows[1:]]), \
        np.array([float(r[2]) for r in rows[1:]])


SCAN_OPTS = {
    "auto": (),
    "sequential": (("chunk", 1 << 40),),                       # one chunk per series (row a8): no dense level on the path
    "deep": (("chunk", 16), ("group", 2), ("top", 2)),         # many dense levels, tree up to the root
    "walk": (("chunk", 16), ("group", 2), ("top", 13)),        # long sequential walk at the top level
    "ragged": (("chunk", 37), ("group", 3), ("lanes", 32)),    # chunk / group sizes dividing nothing
}


def _run(ctx, w, form, opts=(), **kw):
    ctx.set_option("form", form)
    for k, v in opts:
        ctx.set_option(k, v)
    try:
        ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
        out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"], **kw)
        plan = ctx.plan_info()
        ll = ctx.smolgp_loglik_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
    finally:
        for k in ("form", "chunk", "group", "top", "lanes"):
            ctx.set_option(k, 0)
    return out, ll, plan


CASES = [(1, 1000, None), (2, 3001, None), ("fig2", 400, None), ("fig3", 600, None), (3, 1500, None), (4, 1203, None), (5, 300, 6)]


@pytest.mark.parametrize("opt", sorted(SCAN_OPTS))
@pytest.mark.parametrize("cfg,N,batch", CASES)
def test_sqrt_form_matches_oracle(ctx, oracle, cfg, N, batch, opt):
    w = W.make(cfg, N=N, batch=batch)
    out, ll, plan = _run(ctx, w, 1, SCAN_OPTS[opt])
    assert "form=sqrt" in plan and ("levels=0" in plan) == (opt == "sequential")
    for s in ([None] if batch is None else range(batch)):
        ref = PU.reference(oracle, w, series=s)
        i = 0 if s is None else s
        e = PU.errors(ref, out["loglik"][i], out["mean"][i], out["var"][i], floor=PU.prior_sd(oracle, w, series=s))
        assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, e
        assert abs(ll[i] - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])


def test_sqrt_form_loses_fewer_digits_than_the_covariance_form(ctx, oracle):
    """the quasi-periodic model (config 3: time scales from minutes to weeks in one state) is where the covariance
    recursions lose the most; the factor form, with plain FMAs only, stays two orders below it"""
    w = W.make(3, N=3000)
    ref = PU.reference(oracle, w)
    floor = PU.prior_sd(oracle, w)
    cov, _, pc = _run(ctx, w, 0)
    fac, _, pf = _run(ctx, w, 1)
    assert "form=cov" in pc and "form=sqrt" in pf
    ec = PU.errors(ref, cov["loglik"][0], cov["mean"][0], cov["var"][0], floor=floor)
    ef = PU.errors(ref, fac["loglik"][0], fac["mean"][0], fac["var"][0], floor=floor)
    assert ec["var"] <= PU.POST_RTOL and ef["var"] <= 1e-10 and ef["var"] * 10 <= ec["var"], (ec, ef)
    assert ef["mean"] <= 1e-11 and ef["ll"] <= 1e-12, ef


def test_sqrt_form_instantaneous_data(ctx, oracle):
    """paper section 2 (K = N observe events): the record's extra row is then a copy of x_0, its factor row 0 of L_xx"""
    kern = [W.comp(W.SHO, 1.1, 2 * np.pi / 300.0, 2.0), W.comp(W.MATERN52, 0.6, 900.0)]
    rng = np.random.default_rng(8)
    t = np.cumsum(rng.uniform(5.0, 60.0, 1500))
    inst = np.zeros(1500, np.int32)
    sigma = rng.uniform(0.1, 0.4, 1500)
    y = W.synth_y(rng, kern, t, t + 1e-9, inst, sigma)
    ctx.set_option("form", 1)
    try:
        ev = ctx.smolgp_build_events_instant_host(t, inst, 1)
        out = ctx.smolgp_condition_host(ev, kern, y, sigma)
    finally:
        ctx.set_option("form", 0)
    ref = oracle.ssm_instant(kern, 1, t, inst, y, sigma)
    psd = np.sqrt(oracle.kernel(kern, 0, 0, np.zeros(1))[0])
    assert abs(out["loglik"][0] - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])
    assert np.max(np.abs(out["mean"][0] - ref["mean"]) / (np.abs(ref["mean"]) + psd)) <= PU.POST_RTOL
    assert np.max(np.abs(out["var"][0] - ref["var"]) / ref["var"]) <= PU.POST_RTOL


def test_sqrt_form_full_size_cfg5_sampled_series(ctx, oracle):
    """config 5 (8192 series x 2048 exposures) runs one chunk per series in either form: the batched sequential
    variant (row a8) is the factor form's production plan"""
    w = W.make(5)
    out, _, plan = _run(ctx, w, 1)
    assert "form=sqrt" in plan
    base_sd = PU.prior_sd(oracle, w)
    lo, hi = int(np.argmin(w["amp"])), int(np.argmax(w["amp"]))
    for s in sorted({0, 4095, lo, hi} | set(int(x) for x in np.random.default_rng(51).choice(4096, 12, replace=False))):
        ref = PU.reference(oracle, w, series=s)
        e = PU.errors(ref, out["loglik"][s], out["mean"][s], out["var"][s], floor=base_sd * float(w["amp"][s]))
        assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, (s, e)
    assert np.all(np.isfinite(out["loglik"])) and np.all(out["var"] > 0)


@pytest.mark.parametrize("cfg", [3, 4])
def test_sqrt_form_full_size_golden(ctx, oracle, cfg):
    """N = 1e5 (n = 21) and N = 1e6 (n = 17) in the automatic plan (chunked scan, ten dense levels in factor form):
    with no compensated product anywhere the variance stays within 1e-10 of the long-double oracle (the covariance
    form: 1e-9 on config 3 WITH compensated products in its dense levels)"""
    ll, idx, mean, var = _golden(cfg)
    w = W.make(cfg)
    out, _, plan = _run(ctx, w, 1)
    assert "form=sqrt" in plan and "levels=10" in plan
    assert abs(out["loglik"][0] - ll) <= 1e-11 * abs(ll)
    floor = PU.prior_sd(oracle, w, idx=idx)
    assert np.max(np.abs(out["mean"][0][idx] - mean) / (np.abs(mean) + floor)) <= 1e-10
    rel = np.abs(out["var"][0][idx] - var) / var
    assert rel.max() <= 1e-10, (rel.max(), np.quantile(rel, [0.5, 0.9, 0.99]))


def test_sqrt_form_gradient_and_unsupported_queries(ctx, oracle):
    from paper_2601_02527_b200 import binding as B
    w = W.make(2, N=400)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    ll0, g0 = ctx.smolgp_loglik_grad_host(ev, w["kernel"], w["y"], w["sigma"])
    ctx.set_option("form", 1)
    try:
        ll1, g1 = ctx.smolgp_loglik_grad_host(ev, w["kernel"], w["y"], w["sigma"])
        with pytest.raises(B.SmolgpError) as e:   # the state store of row a7 is kept in covariance form only
            ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], t_query=np.array([10.0, 20.0]))
        assert e.value.rc == -3 and "square-root" in str(e.value)
    finally:
        ctx.set_option("form", 0)
    assert abs(ll1[0] - ll0[0]) <= 1e-11 * abs(ll0[0])
    assert np.max(np.abs(g1 - g0)) <= 1e-6 * np.max(np.abs(g0))
    with pytest.raises(B.SmolgpError):
        ctx.set_option("form", 2)
