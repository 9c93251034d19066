"""Randomly drawn model structures and exposure layouts, both forms of the scan, against the dense definition (Eq. 2.4
P:72-76, Eq. 2.26): sums of 1-4 components of every family (App. C.1; under-, critically and over-damped
SHO; products with the periodic series, App. C.2), each entering a random subset of 1-4 instruments (Eq. 3.2),
exposures that overlap across instruments, with back-to-back exposures and exact cross-instrument ties.  The shipped
configs fix five structures; this sweeps what they do not (block orders, masks, block dimensions 2-3-4 mixed, ...)."""
import numpy as np
import pytest

from paper_2601_02527_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2601_02527_b200 import binding as B
    c = B.Context(0)
    yield c
    c.close()


def _draw(seed):
    rng = np.random.default_rng(1000 + seed)
    ninst = int(rng.integers(1, 5))
    ncomp = int(rng.integers(1, 5))
    kern = []
    for c in range(ncomp):
        fam = int(rng.choice([W.MATERN32, W.MATERN52, W.SHO, W.SHO, W.MATERN32_X_PERIODIC]))
        mask = int(rng.integers(1, 1 << ninst))
        sig = float(rng.uniform(0.3, 1.5))
        if fam == W.SHO:
            q = float(rng.choice([0.3, 0.5, 0.8, 4.0, 30.0]))          # over-, critically, under-damped
            kern.append(W.comp(W.SHO, sig, 2 * np.pi / float(rng.uniform(100.0, 3000.0)), q, inst_mask=mask))
        elif fam == W.MATERN32_X_PERIODIC:
            kern.append(W.comp(fam, sig, float(rng.uniform(2000.0, 20000.0)), float(rng.uniform(500.0, 5000.0)), float(rng.uniform(0.6, 1.5)),
                               order=int(rng.integers(1, 3)), inst_mask=mask))
        else:
            kern.append(W.comp(fam, sig, float(rng.uniform(100.0, 5000.0)), inst_mask=mask))
    seen = 0
    for k in kern:
        seen |= k["inst_mask"]
    for q in range(ninst):                                             # every instrument sees something
        if not (seen >> q) & 1:
            kern[int(rng.integers(0, ncomp))]["inst_mask"] |= 1 << q
    # exposures: per instrument a sequence on a 10 s grid (so that instruments tie exactly), some back to back
    N = 260
    ts, te, inst = [], [], []
    per = [N // ninst + (1 if q < N % ninst else 0) for q in range(ninst)]
    for q in range(ninst):
        t = float(rng.integers(0, 20)) * 10.0
        for _ in range(per[q]):
            length = float(rng.integers(2, 30)) * 10.0
            ts.append(t); te.append(t + length); inst.append(q)
            t += length + (0.0 if rng.random() < 0.3 else float(rng.integers(1, 40)) * 10.0)
    ts, te, inst = np.array(ts), np.array(te), np.array(inst, np.int32)
    p = rng.permutation(N)                                             # arbitrary input order
    ts, te, inst = ts[p], te[p], inst[p]
    sigma = rng.uniform(0.05, 0.5, N)
    y = W.synth_y(rng, kern, ts, te, inst, sigma, n_features=32)
    return kern, ninst, ts, te, inst, y, sigma


@pytest.mark.parametrize("seed", range(12))
def test_random_structure_matches_dense_definition(ctx, oracle, seed):
    kern, ninst, ts, te, inst, y, sigma = _draw(seed)
    n = oracle.model_dim(kern, ninst)
    if n > 31:
        pytest.skip("augmented dimension above SMOLGP_MAX_DIM")
    tq = np.linspace(ts.min() - 50.0, te.max() + 50.0, 40)
    qi = int(seed % ninst)
    ref = oracle.dense(kern, ts, te, inst, y, sigma, tq=tq, query_inst=qi)
    prior_sd = np.sqrt(np.diag(oracle.kff(kern, ts, te, inst)))
    k0 = float(oracle.kernel(kern, qi, qi, np.zeros(1))[0])
    # (form, scan options): covariance and square-root form; automatic plan, short chunks with a deep tree, the
    # specialised kernels (compiled at run time for a structure nobody has seen)
    for form, opts in ((0, ()), (1, ()), (0, (("chunk", 16), ("group", 2))), (1, (("chunk", 16), ("group", 3))), (0, (("jit", 1), ("chunk", 24)))):
        ctx.set_option("form", form)
        for k, v in opts:
            ctx.set_option(k, v)
        try:
            ev = ctx.smolgp_build_events_host(ts, te, inst, ninst)
            out = ctx.smolgp_condition_host(ev, kern, y, sigma, t_query=tq, query_instrument=qi)
            plan = ctx.plan_info()
        finally:
            for k in ("form", "chunk", "group", "jit"):
                ctx.set_option(k, 0)
        tag = (seed, form, opts, plan)
        assert abs(out["loglik"][0] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"]), tag
        assert np.max(np.abs(out["mean"][0] - ref["mean"]) / (np.abs(ref["mean"]) + prior_sd)) <= 1e-8, tag
        assert np.max(np.abs(out["var"][0] - ref["var"]) / ref["var"]) <= 1e-8, tag
        assert np.max(np.abs(out["mean_query"][0] - ref["mq"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mq"]))), tag
        assert np.max(np.abs(out["var_query"][0] - ref["vq"]) / np.maximum(ref["vq"], 1e-12 * k0)) <= 1e-8, tag
