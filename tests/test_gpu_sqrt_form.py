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


@pytest.mark.parametrize("opt", ["auto", "sequential", "ragged"])
def test_sqrt_form_instantaneous_data(ctx, oracle, opt):
    """paper section 2 (K = N observe events; two instruments sampling different sums of the components, simultaneous
    samples): the record's extra row is then a copy of x_0, its factor row 0 of L_xx; with query times"""
    kern = [W.comp(W.SHO, 1.1, 2 * np.pi / 300.0, 2.0), W.comp(W.MATERN52, 0.6, 900.0, inst_mask=2)]
    rng = np.random.default_rng(8)
    N = 1500
    t = np.round(np.cumsum(rng.uniform(5.0, 60.0, N)))          # whole seconds: some samples of the two instruments coincide
    inst = rng.integers(0, 2, N).astype(np.int32)
    sigma = rng.uniform(0.1, 0.4, N)
    y = W.synth_y(rng, kern, t, t + 1e-9, inst, sigma)
    tq = np.concatenate([rng.uniform(t.min() - 200.0, t.max() + 200.0, 60), t[:3]])
    ctx.set_option("form", 1)
    for k, v in SCAN_OPTS[opt]:
        ctx.set_option(k, v)
    try:
        ev = ctx.smolgp_build_events_instant_host(t, inst, 2)
        out = ctx.smolgp_condition_host(ev, kern, y, sigma, t_query=tq, query_instrument=1)
        assert "form=sqrt" in ctx.plan_info()
    finally:
        for k in ("form", "chunk", "group", "top", "lanes"):
            ctx.set_option(k, 0)
    ref = oracle.ssm_instant(kern, 2, t, inst, y, sigma, tq=tq, query_inst=1)
    psd = np.sqrt(np.array([oracle.kernel(kern, int(q), int(q), np.zeros(1))[0] for q in inst]))
    assert abs(out["loglik"][0] - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])
    assert np.max(np.abs(out["mean"][0] - ref["mean"]) / (np.abs(ref["mean"]) + psd)) <= PU.POST_RTOL
    assert np.max(np.abs(out["var"][0] - ref["var"]) / ref["var"]) <= PU.POST_RTOL
    k0 = float(oracle.kernel(kern, 1, 1, np.zeros(1))[0])
    assert np.max(np.abs(out["mean_query"][0] - ref["mq"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mq"])))
    assert np.max(np.abs(out["var_query"][0] - ref["vq"]) / ref["vq"]) <= 1e-8


def test_sqrt_form_full_size_cfg5_sampled_series(ctx, oracle):
    """config 5 (4096 series x 2048 exposures) runs one chunk per series in either form: the batched sequential
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
    floor = PU.prior_sd(oracle, w, idx=idx)
    err = {}
    for form in (0, 1):
        out, _, plan = _run(ctx, w, form)
        assert ("form=sqrt" if form else "form=cov") in plan and "levels=10" in plan
        err[form] = (abs(out["loglik"][0] - ll) / abs(ll), np.max(np.abs(out["mean"][0][idx] - mean) / (np.abs(mean) + floor)),
                     np.max(np.abs(out["var"][0][idx] - var) / var))
        # (pytest -s: the figures quoted in profiles/r02_sqrt_form.md)
        print("\nconfig %d, %s form: loglik %.2e  mean %.2e  variance %.2e  [%s]" % ((cfg, "square-root" if form else "covariance") + err[form] + (plan,)))
    assert err[1][0] <= 1e-11 and err[1][1] <= 1e-10 and err[1][2] <= 1e-10, err
    assert err[0][2] <= PU.POST_RTOL and err[1][2] <= 1.01 * err[0][2], err


def test_sqrt_form_gradient(ctx, oracle):
    from paper_2601_02527_b200 import binding as B
    w = W.make(2, N=400)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    ll0, g0 = ctx.smolgp_loglik_grad_host(ev, w["kernel"], w["y"], w["sigma"])
    ctx.set_option("form", 1)
    try:
        ll1, g1 = ctx.smolgp_loglik_grad_host(ev, w["kernel"], w["y"], w["sigma"])
    finally:
        ctx.set_option("form", 0)
    assert abs(ll1[0] - ll0[0]) <= 1e-11 * abs(ll0[0])
    assert np.max(np.abs(g1 - g0)) <= 1e-6 * np.max(np.abs(g0))
    with pytest.raises(B.SmolgpError):
        ctx.set_option("form", 2)


@pytest.mark.parametrize("cfg,N,batch,qi", [(2, 800, None, 0), ("fig3", 500, None, 1), (3, 700, None, 2), (4, 600, None, 3), (5, 200, 3, 0)])
@pytest.mark.parametrize("opt", ["auto", "sequential", "ragged"])
def test_sqrt_form_query_prediction_matches_oracle(ctx, oracle, cfg, N, batch, qi, opt):
    """row a7 (Algorithm 1) from the stored FACTORS: before the first event, between events, at event
    times, after the last event"""
    w = W.make(cfg, N=N, batch=batch)
    rng = np.random.default_rng(4)
    t0, t1 = w["t_start"].min(), w["t_end"].max()
    tq = np.concatenate([rng.uniform(t0 - 0.05 * (t1 - t0), t1 + 0.05 * (t1 - t0), 150), w["t_start"][:3], w["t_end"][-3:], [t0 - 1000.0, t1 + 1000.0]])
    out, _, plan = _run(ctx, w, 1, SCAN_OPTS[opt], t_query=tq, query_instrument=qi)
    assert "form=sqrt" in plan
    for s in ([None] if batch is None else range(batch)):
        i = 0 if s is None else s
        kern = w["kernel"] if s is None else [dict(k, sigma=k["sigma"] * w["amp"][s]) for k in w["kernel"]]
        y = w["y"] if s is None else w["y"][s]
        # (the oracle's Algorithm 1 inverts P^-_next as printed, which idle-z zeroing makes exactly singular: run without
        # it -- output-equivalent, pinned in tests/test_oracle_inference_pins.py)
        ref = oracle.ssm(kern, w["n_inst"], w["t_start"], w["t_end"], w["instrument"], y, w["sigma"],
                         flags=oracle.FLAG_TWO_FILTER, tq=tq, query_inst=qi)
        k0 = float(oracle.kernel(kern, qi, qi, np.zeros(1))[0])  # prior variance of the latent
        assert np.max(np.abs(out["mean_query"][i] - ref["mq"])) <= 1e-8 * np.sqrt(k0) + 1e-8 * np.max(np.abs(ref["mq"]))
        assert np.max(np.abs(out["var_query"][i] - ref["vq"]) / ref["vq"]) <= 1e-8
        assert abs(out["loglik"][i] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"])
        assert np.max(np.abs(out["var"][i] - ref["var"]) / ref["var"]) <= 1e-8


def test_sqrt_form_degenerate_inputs(ctx, oracle):
    """N = 1, N = 2, exact ties between instruments (start/start, end/start, end/end), one query; against the dense
    definition"""
    kern = [W.comp(W.SHO, 1.0, 2 * np.pi / 330.0, 10.0), W.comp(W.MATERN32, 0.5, 900.0, inst_mask=2)]
    cases = [
        (np.array([5.0]), np.array([60.0]), np.array([0], np.int32), 1),
        (np.array([5.0, 100.0]), np.array([60.0, 130.0]), np.array([0, 0], np.int32), 1),
        (np.array([0.0, 0.0, 50.0, 80.0, 120.0]), np.array([50.0, 80.0, 120.0, 120.0, 200.0]), np.array([0, 1, 0, 1, 0], np.int32), 2),
    ]
    rng = np.random.default_rng(2)
    for ts, te, inst, ninst in cases:
        y = rng.standard_normal(ts.size)
        sigma = np.full(ts.size, 0.3)
        tq = np.array([0.5 * (ts[0] + te[-1])])
        w = dict(t_start=ts, t_end=te, instrument=inst, n_inst=ninst, kernel=kern, y=y, sigma=sigma, amp=None)
        for opts in ((), (("chunk", 2), ("group", 2))):
            out, _, plan = _run(ctx, w, 1, opts, t_query=tq, query_instrument=ninst - 1)
            assert "form=sqrt" in plan
            ref = oracle.dense(kern, ts, te, inst, y, sigma, tq=tq, query_inst=ninst - 1)
            assert abs(out["loglik"][0] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"])
            np.testing.assert_allclose(out["mean"][0], ref["mean"], rtol=1e-8, atol=1e-9)
            np.testing.assert_allclose(out["var"][0], ref["var"], rtol=1e-8, atol=1e-10)
            np.testing.assert_allclose(out["mean_query"][0], ref["mq"], rtol=1e-8, atol=1e-9)
            np.testing.assert_allclose(out["var_query"][0], ref["vq"], rtol=1e-8, atol=1e-10)


def test_sqrt_form_largest_state_dimension(ctx, oracle):
    """n = SMOLGP_MAX_DIM = 31 (periodic product of order 6, d = 26, five overlapping instruments): 64 columns in the
    stacked matrix of a predict step, 143 KB of shared memory per dense combine"""
    rng = np.random.default_rng(21)
    N, ninst = 240, 5
    ts = np.sort(rng.uniform(0, 40000.0, N))
    inst = np.arange(N, dtype=np.int32) % ninst
    te = ts + rng.uniform(20.0, 120.0, N)
    for q in range(ninst):
        idx = np.nonzero(inst == q)[0]
        te[idx[:-1]] = np.minimum(te[idx[:-1]], ts[idx[1:]] - 1.0)
    kern = [W.comp(W.MATERN32_X_PERIODIC, 1.2, 5000.0, 9000.0, 0.8, order=6)]
    sigma = np.full(N, 0.2)
    y = W.synth_y(rng, kern, ts, te, inst, sigma)
    w = dict(kernel=kern, n_inst=ninst, t_start=ts, t_end=te, instrument=inst, y=y, sigma=sigma, amp=None)
    ref = PU.reference(oracle, w)
    for opts in ((), (("chunk", 48),)):
        out, _, plan = _run(ctx, w, 1, opts)
        assert "form=sqrt" in plan and "n=31" in plan
        e = PU.errors(ref, out["loglik"][0], out["mean"][0], out["var"][0], floor=PU.prior_sd(oracle, w))
        assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, e
