"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (ctypes binding), against the
CPU oracle on the same seeded inputs.  Bars (north_star): event stream
bit-exact; log-likelihood relative 1e-9; posterior mean and variance relative 1e-8 (the mean's
error is scaled by |mean| + prior sd of the exposure average, reading c13)."""
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


def _reset(ctx):
    ctx.set_option("chunk", 0)
    ctx.set_option("group", 0)
    ctx.set_option("top", 0)
    ctx.set_option("lanes", 0)
    ctx.set_option("jit", 0)


SCAN_OPTS = {
    "auto": (),
    "sequential": (("chunk", 1 << 40),),                       # one chunk per series (row a8)
    "deep": (("chunk", 16), ("group", 2), ("top", 2)),         # many dense levels, tree up to the root
    "walk": (("chunk", 16), ("group", 2), ("top", 13)),        # long sequential walk at the top level
    "ragged": (("chunk", 37), ("group", 3), ("lanes", 32)),    # chunk/group sizes dividing nothing
    "jit": (("chunk", 29), ("jit", 1)),                        # specialised chunk kernels (ahead-of-time module or NVRTC)
    "generic": (("chunk", 23), ("jit", -1)),                   # the statically compiled shared-memory kernels
}


# ---------------------------------------------------------------------------------------------
# a1: event build, bit-exact against the oracle's sort
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,N", [(1, 1000), (2, 20000), (3, 5000), (4, 4097), (5, 2048), ("fig2", 400), ("fig3", 600)])
def test_events_bit_exact(ctx, oracle, cfg, N):
    w = W.make(cfg, N=N, batch=(2 if cfg == 5 else None), n_features=4)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    t, kind, inst, idx = ev.export()
    ot, ok, oi, ox = oracle.events(w["t_start"], w["t_end"], w["instrument"])
    assert np.array_equal(t, ot)
    assert np.array_equal(kind, ok)
    assert np.array_equal(inst, oi)
    assert np.array_equal(idx, ox)
    ev.free()


def test_events_device_pointers_and_shuffled_input(ctx, oracle):
    """device-pointer entry point; exposures given in random order; negative and tied times"""
    import torch
    rng = np.random.default_rng(5)
    w = W.make("fig2", N=300, n_features=4)            # back-to-back: every end ties with a start
    ts, te = w["t_start"] - 20000.0, w["t_end"] - 20000.0  # times straddle zero
    p = rng.permutation(ts.size)
    ts, te, inst = ts[p], te[p], w["instrument"][p]
    dev = torch.device("cuda:0")
    ev = ctx.smolgp_build_events(torch.tensor(ts, device=dev), torch.tensor(te, device=dev),
                                 torch.tensor(inst, device=dev), 1)
    t, kind, ins, idx = ev.export()
    ot, ok, oi, ox = oracle.events(ts, te, inst)
    assert np.array_equal(t, ot) and np.array_equal(kind, ok) and np.array_equal(idx, ox)
    # ties: the end comes first (reading R5)
    tie = np.nonzero(t[1:] == t[:-1])[0]
    assert tie.size > 100 and np.all(kind[tie] == 0) and np.all(kind[tie + 1] == 1)


def test_events_tie_order_is_time_kind_instrument_index(ctx, oracle):
    """simultaneous same-kind events of several instruments, given in REVERSE instrument order and with
    repeated exposures of one instrument out of index order: the stream is ordered by (time, end before
    start, instrument, exposure index) whatever the input order (include/smolgp.h; SURVEY reading c5)"""
    ts = np.array([100.0, 100.0, 100.0, 0.0, 0.0, 0.0, 250.0, 160.0, 160.0])
    te = np.array([160.0, 160.0, 150.0, 100.0, 100.0, 90.0, 300.0, 250.0, 250.0])
    inst = np.array([2, 1, 0, 2, 1, 0, 1, 2, 1], np.int32)  # starts tie at 0 / 100 / 160, ends tie at 100 / 160 / 250, all in reverse order
    ev = ctx.smolgp_build_events_host(ts, te, inst, 3)
    t, kind, ins, idx = ev.export()
    ot, ok, oi, ox = oracle.events(ts, te, inst)
    assert np.array_equal(t, ot) and np.array_equal(kind, ok) and np.array_equal(ins, oi) and np.array_equal(idx, ox)
    # the rule, spelled out (not only "equal to the oracle"): lexicographic in (t, kind, instrument, index)
    keys = list(zip(t.tolist(), kind.tolist(), ins.tolist(), idx.tolist()))
    assert keys == sorted(keys)
    # a shuffled copy of a larger overlapping case gives the same stream up to the exposure renumbering
    rng = np.random.default_rng(11)
    w = W.make("fig3", N=500, n_features=4)
    ts2 = np.round(w["t_start"] / 30.0) * 30.0   # coarse grid: many cross-instrument ties of both kinds
    te2 = ts2 + np.maximum(30.0, np.round((w["t_end"] - w["t_start"]) / 30.0) * 30.0)
    for q in range(2):  # keep each instrument free of self-overlap after the rounding
        m = np.nonzero(w["instrument"] == q)[0]
        for a, b in zip(m[:-1], m[1:]):
            ts2[b] = max(ts2[b], te2[a]); te2[b] = max(te2[b], ts2[b] + 30.0)
    p = rng.permutation(ts2.size)
    ev2 = ctx.smolgp_build_events_host(ts2[p], te2[p], w["instrument"][p], 2)
    t, kind, ins, idx = ev2.export()
    ot, ok, oi, ox = oracle.events(ts2[p], te2[p], w["instrument"][p])
    assert np.array_equal(t, ot) and np.array_equal(kind, ok) and np.array_equal(ins, oi) and np.array_equal(idx, ox)
    assert np.sum(t[1:] == t[:-1]) > 100


def test_events_validation(ctx):
    from paper_2601_02527_b200.binding import SmolgpError
    ts, te, ins = np.array([0.0, 10.0, 30.0]), np.array([5.0, 20.0, 40.0]), np.zeros(3, np.int32)
    with pytest.raises(SmolgpError) as e:   # same-instrument overlap
        ctx.smolgp_build_events_host(ts, np.array([5.0, 31.0, 40.0]), ins, 1)
    assert e.value.rc == -2
    ctx.smolgp_build_events_host(ts, np.array([10.0, 30.0, 40.0]), ins, 1).free()  # back-to-back is legal
    ctx.smolgp_build_events_host(ts, np.array([5.0, 31.0, 40.0]), np.array([0, 1, 0], np.int32), 2).free()
    for bad_te in (np.array([5.0, 10.0, 40.0]), np.array([5.0, np.nan, 40.0]), np.array([5.0, np.inf, 40.0])):
        with pytest.raises(SmolgpError) as e:
            ctx.smolgp_build_events_host(ts, bad_te, ins, 1)
        assert e.value.rc == -1
    with pytest.raises(SmolgpError) as e:
        ctx.smolgp_build_events_host(ts, te, np.array([0, 2, 0], np.int32), 2)
    assert e.value.rc == -1
    with pytest.raises(SmolgpError) as e:
        ctx.smolgp_build_events_host(ts, te, ins, 17)
    assert e.value.rc == -3


# ---------------------------------------------------------------------------------------------
# a2: discretisation against the oracle's long-double Taylor + doubling
# ---------------------------------------------------------------------------------------------
KERNELS = {
    "m32": [W.comp(W.MATERN32, 1.3, 600.0)],
    "m52": [W.comp(W.MATERN52, 0.7, 86400.0)],
    "sho": [W.comp(W.SHO, 1.0, 2 * np.pi / 330.0, 10.0)],
    "sho_crit": [W.comp(W.SHO, 1.1, 0.02, 0.5)],
    "sho_over": [W.comp(W.SHO, 0.9, 0.05, 0.3)],
    "qp": [W.comp(W.MATERN32_X_PERIODIC, 1.0, 20 * W.DAY, 25 * W.DAY, 1.0, order=4)],
    "cfg4": W.make(4, N=8, n_features=2)["kernel"],
}


@pytest.mark.parametrize("name", sorted(KERNELS))
@pytest.mark.parametrize("dt", [0.0, 1e-3, 12.0, 55.0, 300.0, 5000.0, 57600.0, 3e6])
def test_discretise_matches_oracle(ctx, oracle, name, dt):
    kern = KERNELS[name]
    ninst = 4 if name == "cfg4" else 2
    A, Q = ctx.smolgp_discretise_host(kern, ninst, dt)
    Ao, Qo = oracle.discretise(kern, ninst, dt)
    n = A.shape[0]
    d = n - ninst
    # compare in equilibrated units: x rows by sqrt(Pinf_ii), z rows by dt * sd (so every entry is O(1))
    _, _, Pinf, _ = oracle.ssm_matrices(kern, ninst)
    s = np.concatenate([np.sqrt(np.diag(Pinf)), np.full(ninst, (dt if dt > 0 else 1.0) * np.sqrt(np.trace(Pinf)))])
    As, Aos = A / s[:, None] * s[None, :], Ao / s[:, None] * s[None, :]
    Qs, Qos = Q / np.outer(s, s), Qo / np.outer(s, s)
    assert np.max(np.abs(As - Aos)) <= 5e-13 * max(1.0, np.max(np.abs(Aos)))
    # Q entries span many orders of magnitude inside one matrix (q22 ~ dt^5 for short steps): each
    # entry is compared relative to the geometric mean of its diagonal entries (Cauchy-Schwarz scale)
    dg = np.sqrt(np.abs(np.diag(Qos)))
    scale = np.outer(dg, dg) + 1e-300
    assert np.max(np.abs(Qs - Qos) / scale) <= 2e-12


# ---------------------------------------------------------------------------------------------
# a3-a6: log-likelihood and posterior at the observations, reduced-size versions of every config
# (sizes the long-double oracle finishes in seconds; several chunks, several dense levels, ragged tails)
# ---------------------------------------------------------------------------------------------
CASES = [(1, 1000, None), (2, 3001, None), ("fig2", 400, None), ("fig3", 600, None), (3, 1500, None),
         (4, 1203, None), (5, 300, 6)]


@pytest.mark.parametrize("opt", sorted(SCAN_OPTS))
@pytest.mark.parametrize("cfg,N,batch", CASES)
def test_condition_matches_oracle(ctx, oracle, cfg, N, batch, opt):
    w = W.make(cfg, N=N, batch=batch)
    for k, v in SCAN_OPTS[opt]:
        ctx.set_option(k, v)
    try:
        ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
        out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
        ll = ctx.smolgp_loglik_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
    finally:
        _reset(ctx)
    for s in ([None] if batch is None else range(batch)):
        ref = PU.reference(oracle, w, series=s)
        i = 0 if s is None else s
        floor = PU.prior_sd(oracle, w, series=s)
        e = PU.errors(ref, out["loglik"][i], out["mean"][i], out["var"][i], floor=floor)
        assert e["ll"] <= PU.LL_RTOL, e
        assert abs(ll[i] - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])
        assert e["mean"] <= PU.POST_RTOL, e
        assert e["var"] <= PU.POST_RTOL, e


def test_device_pointer_entry_points_match_host_ones(ctx):
    import torch
    w = W.make(2, N=2000)
    dev = torch.device("cuda:0")
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    h = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
    y, sg = torch.tensor(w["y"], device=dev), torch.tensor(w["sigma"], device=dev)
    d = ctx.smolgp_condition(ev, w["kernel"], y, sg)
    ll = ctx.smolgp_loglik(ev, w["kernel"], y, sg)
    torch.cuda.synchronize()
    assert np.array_equal(d["mean"].cpu().numpy()[0], h["mean"][0])
    assert np.array_equal(d["var"].cpu().numpy()[0], h["var"][0])
    assert d["loglik"].cpu().numpy()[0] == h["loglik"][0] == ll.cpu().numpy()[0]


def test_dense_definition_parity_tiny(ctx, oracle):
    """the GPU path against the DEFINITION (dense integrated GP, Eq. 2.4 + 3.1) directly, N = 150"""
    for cfg, batch in [(2, None), (3, None), (4, None), (5, 2)]:
        w = W.make(cfg, N=150, batch=batch)
        ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
        out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
        for s in ([None] if batch is None else range(batch)):
            i = 0 if s is None else s
            kern = w["kernel"] if s is None else [dict(k, sigma=k["sigma"] * w["amp"][s]) for k in w["kernel"]]
            y = w["y"] if s is None else w["y"][s]
            ref = oracle.dense(kern, w["t_start"], w["t_end"], w["instrument"], y, w["sigma"])
            assert abs(out["loglik"][i] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"])
            floor = PU.prior_sd(oracle, dict(w, kernel=kern))
            assert np.max(np.abs(out["mean"][i] - ref["mean"]) / (np.abs(ref["mean"]) + floor)) <= 1e-8
            # the dense solver's own variance (K - K C^-1 K, cancellation) is good to ~1e-10 of the prior
            assert np.max(np.abs(out["var"][i] - ref["var"]) / floor ** 2) <= 1e-8


def test_numeric_errors_are_reported(ctx):
    from paper_2601_02527_b200.binding import SmolgpError
    w = W.make(1, N=64)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    y = w["y"].copy()
    y[10] = np.nan
    with pytest.raises(SmolgpError) as e:
        ctx.smolgp_loglik_host(ev, w["kernel"], y, w["sigma"])
    assert e.value.rc == -6
    with pytest.raises(SmolgpError) as e:
        ctx.smolgp_loglik_host(ev, [W.comp(7, 1.0, 1.0)], w["y"], w["sigma"])
    assert e.value.rc == -3
    sg = w["sigma"].copy()
    sg[5] = 0.0
    with pytest.raises(SmolgpError) as e:   # sigma_n <= 0 is an invalid argument
        ctx.smolgp_loglik_host(ev, w["kernel"], w["y"], sg)
    assert e.value.rc == -1
    # the context stays usable after an error
    ll = ctx.smolgp_loglik_host(ev, w["kernel"], w["y"], w["sigma"])
    assert np.isfinite(ll[0])


# ---------------------------------------------------------------------------------------------
# a7: prediction at arbitrary times (Algorithm 1) against the oracle's Algorithm 1 and
# against the dense definition
# ---------------------------------------------------------------------------------------------
def _queries(w, rng, M):
    ts, te = w["t_start"], w["t_end"]
    t0, t1 = ts.min(), te.max()
    span = t1 - t0
    tq = np.concatenate([
        rng.uniform(t0, t1, M),                       # interpolation (inside exposures and gaps)
        t0 - rng.uniform(0, 0.05 * span, 5),          # retrodiction (reading R8)
        t1 + rng.uniform(0, 0.05 * span, 5),          # extrapolation
        ts[:3], te[-3:], [t0, t1],                    # exactly at event times
    ])
    return tq


@pytest.mark.parametrize("cfg,N,batch,qi", [(1, 400, None, 0), (2, 900, None, 1), ("fig2", 300, None, 0),
                                            (4, 700, None, 3), (5, 200, 3, 0)])
def test_query_prediction_matches_oracle(ctx, oracle, cfg, N, batch, qi):
    rng = np.random.default_rng(17)
    w = W.make(cfg, N=N, batch=batch)
    tq = _queries(w, rng, 60)
    ctx.set_option("chunk", 24)
    try:
        ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
        out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"], t_query=tq, query_instrument=qi)
    finally:
        _reset(ctx)
    for s in ([None] if batch is None else range(batch)):
        i = 0 if s is None else s
        kern = w["kernel"] if s is None else [dict(k, sigma=k["sigma"] * w["amp"][s]) for k in w["kernel"]]
        y = w["y"] if s is None else w["y"][s]
        # the oracle's Algorithm 1 inverts P^-_next (as printed), which idle-z zeroing makes exactly singular:
        # run it without that (output-equivalent, pinned in tests/test_oracle_inference_pins.py)
        ref = oracle.ssm(kern, w["n_inst"], w["t_start"], w["t_end"], w["instrument"], y, w["sigma"],
                         flags=oracle.FLAG_TWO_FILTER, tq=tq, query_inst=qi)
        k0 = float(oracle.kernel(kern, qi, qi, np.zeros(1))[0])  # prior variance of the latent
        assert np.max(np.abs(out["mean_query"][i] - ref["mq"])) <= 1e-8 * np.sqrt(k0) + 1e-8 * np.max(np.abs(ref["mq"]))
        assert np.max(np.abs(out["var_query"][i] - ref["vq"]) / ref["vq"]) <= 1e-8
        # the observation-time outputs are unchanged by asking for queries
        assert abs(out["loglik"][i] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"])
        assert np.max(np.abs(out["var"][i] - ref["var"]) / ref["var"]) <= 1e-8


def test_query_prediction_matches_dense_definition(ctx, oracle):
    rng = np.random.default_rng(3)
    for cfg, qi in [(2, 0), (4, 2), (3, 1)]:  # config 3: Algorithm 1's printed RTS step is too ill-conditioned to serve as a reference
        w = W.make(cfg, N=150 if cfg != 3 else 300)
        tq = _queries(w, rng, 40)
        ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
        out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], t_query=tq, query_instrument=qi)
        ref = oracle.dense(w["kernel"], w["t_start"], w["t_end"], w["instrument"], w["y"], w["sigma"], tq=tq, query_inst=qi)
        k0 = float(oracle.kernel(w["kernel"], qi, qi, np.zeros(1))[0])
        assert np.max(np.abs(out["mean_query"][0] - ref["mq"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mq"])))
        assert np.max(np.abs(out["var_query"][0] - ref["vq"])) <= 1e-8 * k0


def test_query_prediction_specialised_kernels_match_generic(ctx):
    """the NVRTC-specialised query kernel against the statically compiled one (bitwise: same source)"""
    rng = np.random.default_rng(9)
    w = W.make(4, N=400)
    tq = _queries(w, rng, 50)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    outs = []
    try:
        for jit in (-1, 1):
            ctx.set_option("jit", jit)
            ctx.set_option("chunk", 40)
            outs.append(ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], t_query=tq, query_instrument=1))
    finally:
        _reset(ctx)
    assert ctx.jit_log() == "", ctx.jit_log()
    for k in ("mean_query", "var_query", "mean", "var", "loglik"):
        np.testing.assert_allclose(outs[0][k], outs[1][k], rtol=1e-11, atol=1e-13)


def test_query_device_pointers(ctx):
    import torch
    w = W.make(2, N=500)
    dev = torch.device("cuda:0")
    tq = np.linspace(w["t_start"].min() - 100, w["t_end"].max() + 100, 257)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    h = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], t_query=tq, query_instrument=1)
    d = ctx.smolgp_condition(ev, w["kernel"], torch.tensor(w["y"], device=dev), torch.tensor(w["sigma"], device=dev),
                             t_query=torch.tensor(tq, device=dev), query_instrument=1)
    torch.cuda.synchronize()
    assert np.array_equal(d["mean_query"].cpu().numpy(), h["mean_query"])
    assert np.array_equal(d["var_query"].cpu().numpy(), h["var_query"])


# ---------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times (automatic scan plan)
# ---------------------------------------------------------------------------------------------
def _golden(cfg):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg%d_full.txt" % cfg)
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    ll = float(rows[0][0])
    idx = np.array([int(r[0]) for r in rows[1:]])
    mean = np.array([float(r[1]) for r in rows[1:]])
    var = np.array([float(r[2]) for r in rows[1:]])
    return ll, idx, mean, var


def test_full_size_cfg2(ctx, oracle):
    w = W.make(2)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
    ref = PU.reference(oracle, w)
    e = PU.errors(ref, out["loglik"][0], out["mean"][0], out["var"][0], floor=PU.prior_sd(oracle, w))
    assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, e


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_golden(ctx, oracle, cfg):
    """N = 1e5 (n = 21) and N = 1e6 (n = 17) against values stored by tests/golden/make_golden.py
    (long-double oracle, sampled exposures)."""
    ll, idx, mean, var = _golden(cfg)
    w = W.make(cfg)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
    assert abs(out["loglik"][0] - ll) <= PU.LL_RTOL * abs(ll)
    floor = PU.prior_sd(oracle, w, idx=idx)  # reading R13: prior sd of the exposure average
    assert np.max(np.abs(out["mean"][0][idx] - mean) / (np.abs(mean) + floor)) <= PU.POST_RTOL
    rel = np.abs(out["var"][0][idx] - var) / var
    assert rel.max() <= PU.POST_RTOL, (rel.max(), np.quantile(rel, [0.5, 0.9, 0.99]))


def test_full_size_cfg5_sampled_series(ctx, oracle):
    w = W.make(5)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    out = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
    lo, hi = int(np.argmin(w["amp"])), int(np.argmax(w["amp"]))
    base_sd = PU.prior_sd(oracle, w)  # prior sd of the exposure averages at amp = 1; scales with the series' amplitude
    picks = sorted({0, 1, 4095, lo, hi} | set(int(x) for x in np.random.default_rng(50).choice(4096, 60, replace=False)))
    assert len(picks) >= 60
    for s in picks:
        ref = PU.reference(oracle, w, series=s)
        e = PU.errors(ref, out["loglik"][s], out["mean"][s], out["var"][s], floor=base_sd * float(w["amp"][s]))
        assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, (s, e)
    assert np.all(np.isfinite(out["loglik"])) and np.all(out["var"] > 0)


def test_largest_state_dimension(ctx, oracle):
    """n = SMOLGP_MAX_DIM = 31: periodic product of order 6 (d = 26) seen by 5 overlapping instruments;
    n = 32 is refused"""
    from paper_2601_02527_b200.binding import SmolgpError
    rng = np.random.default_rng(21)
    N, ninst = 240, 5
    ts = np.sort(rng.uniform(0, 40000.0, N))
    inst = np.arange(N, dtype=np.int32) % ninst
    te = ts + rng.uniform(20.0, 120.0, N)
    for q in range(ninst):  # no self-overlap: clip each exposure at the instrument's next start
        idx = np.nonzero(inst == q)[0]
        te[idx[:-1]] = np.minimum(te[idx[:-1]], ts[idx[1:]] - 1.0)
    kern = [W.comp(W.MATERN32_X_PERIODIC, 1.2, 5000.0, 9000.0, 0.8, order=6)]
    sigma = np.full(N, 0.2)
    y = W.synth_y(rng, kern, ts, te, inst, sigma)
    w = dict(kernel=kern, n_inst=ninst, t_start=ts, t_end=te, instrument=inst, y=y, sigma=sigma, amp=None)
    ev = ctx.smolgp_build_events_host(ts, te, inst, ninst)
    for jit in (-1, 1):
        ctx.set_option("jit", jit)
        ctx.set_option("chunk", 48)
        try:
            out = ctx.smolgp_condition_host(ev, kern, y, sigma)
        finally:
            _reset(ctx)
        ref = PU.reference(oracle, w)
        e = PU.errors(ref, out["loglik"][0], out["mean"][0], out["var"][0], floor=PU.prior_sd(oracle, w))
        assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, (jit, e)
    ev6 = ctx.smolgp_build_events_host(ts, te, np.arange(N, dtype=np.int32) % 6, 6)  # n would be 32
    with pytest.raises(SmolgpError) as ex:
        ctx.smolgp_loglik_host(ev6, kern, y, sigma)
    assert ex.value.rc == -3


def test_degenerate_inputs(ctx, oracle):
    """N = 1, N = 2, exact ties between instruments (start/start, end/start, end/end), one query"""
    kern = [W.comp(W.SHO, 1.0, 2 * np.pi / 330.0, 10.0), W.comp(W.MATERN32, 0.5, 900.0, inst_mask=2)]
    cases = [
        (np.array([5.0]), np.array([60.0]), np.array([0], np.int32), 1),
        (np.array([5.0, 100.0]), np.array([60.0, 130.0]), np.array([0, 0], np.int32), 1),
        # two instruments: equal starts, an end tied with a start, equal ends
        (np.array([0.0, 0.0, 50.0, 80.0, 120.0]), np.array([50.0, 80.0, 120.0, 120.0, 200.0]),
         np.array([0, 1, 0, 1, 0], np.int32), 2),
    ]
    rng = np.random.default_rng(2)
    for ts, te, inst, ninst in cases:
        y = rng.standard_normal(ts.size)
        sigma = np.full(ts.size, 0.3)
        tq = np.array([0.5 * (ts[0] + te[-1])])
        for opts in ((), (("chunk", 2), ("group", 2))):
            for k, v in opts:
                ctx.set_option(k, v)
            try:
                ev = ctx.smolgp_build_events_host(ts, te, inst, ninst)
                out = ctx.smolgp_condition_host(ev, kern, y, sigma, t_query=tq, query_instrument=ninst - 1)
            finally:
                _reset(ctx)
            ref = oracle.dense(kern, ts, te, inst, y, sigma, tq=tq, query_inst=ninst - 1)
            assert abs(out["loglik"][0] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"])
            np.testing.assert_allclose(out["mean"][0], ref["mean"], rtol=1e-8, atol=1e-9)
            np.testing.assert_allclose(out["var"][0], ref["var"], rtol=1e-8, atol=1e-10)
            np.testing.assert_allclose(out["mean_query"][0], ref["mq"], rtol=1e-8, atol=1e-9)
            np.testing.assert_allclose(out["var_query"][0], ref["vq"], rtol=1e-8, atol=1e-10)


def test_component_wise_prediction(ctx, oracle):
    """App. C.3 (C13-C14): a virtual instrument (mask bit >= n_inst) selects the component(s)
    whose latent is predicted; GPU against the oracle's dense definition and sequential algorithm"""
    rng = np.random.default_rng(8)
    w = W.make(2, N=400)                                   # two overlapping instruments
    w0 = 2 * np.pi / 330.0
    kern = [W.comp(W.SHO, 1.0, w0, 10.0, inst_mask=0b0111),            # seen by both; bit 2: the SHO alone
            W.comp(W.MATERN52, 0.6, 3000.0, inst_mask=0b1011),          # seen by both; bit 3: the Matern alone
            W.comp(W.MATERN32, 0.4, 900.0, inst_mask=0b0010)]           # systematic of instrument 1 only
    ts, te, inst, sig = w["t_start"], w["t_end"], w["instrument"], w["sigma"]
    y = W.synth_y(rng, kern, ts, te, inst, sig)
    tq = _queries(w, rng, 40)
    ev = ctx.smolgp_build_events_host(ts, te, inst, 2)
    got = {}
    for v in (0, 1, 2, 3):
        ctx.set_option("chunk", 40)
        try:
            got[v] = ctx.smolgp_condition_host(ev, kern, y, sig, t_query=tq, query_instrument=v)
        finally:
            _reset(ctx)
        ref = oracle.ssm(kern, 2, ts, te, inst, y, sig, flags=oracle.FLAG_TWO_FILTER, tq=tq, query_inst=v)
        k0 = float(oracle.kernel(kern, v, v, np.zeros(1))[0])
        assert np.max(np.abs(got[v]["mean_query"][0] - ref["mq"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mq"])))
        assert np.max(np.abs(got[v]["var_query"][0] - ref["vq"]) / ref["vq"]) <= 1e-8
    # C12: instrument 1's latent = SHO + Matern-5/2 + its own systematic
    sub = W.make(2, N=120)
    y2 = W.synth_y(rng, kern, sub["t_start"], sub["t_end"], sub["instrument"], sub["sigma"])
    tq2 = _queries(sub, rng, 20)
    ev2 = ctx.smolgp_build_events_host(sub["t_start"], sub["t_end"], sub["instrument"], 2)
    for v in (2, 3):
        out = ctx.smolgp_condition_host(ev2, kern, y2, sub["sigma"], t_query=tq2, query_instrument=v)
        ref = oracle.dense(kern, sub["t_start"], sub["t_end"], sub["instrument"], y2, sub["sigma"], tq=tq2, query_inst=v)
        np.testing.assert_allclose(out["mean_query"][0], ref["mq"], rtol=1e-8, atol=1e-9)
        np.testing.assert_allclose(out["var_query"][0], ref["vq"], rtol=1e-8, atol=1e-11)


def test_specialised_kernels_are_reused_across_hyperparameters(ctx, oracle):
    """the run-time specialisation depends on the kernel STRUCTURE only: new hyper-parameter values reuse
    the compiled module (no second compilation) and still match the oracle"""
    import time
    w = W.make(4, N=500)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    ctx.set_option("jit", 1)
    ctx.set_option("chunk", 50)
    try:
        ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])          # compiles (or finds) the structure
        kern2 = [dict(k, sigma=k["sigma"] * 1.7, p0=k["p0"] * 0.6) for k in w["kernel"]]
        t0 = time.perf_counter()
        out = ctx.smolgp_condition_host(ev, kern2, w["y"], w["sigma"])
        dt = time.perf_counter() - t0
    finally:
        _reset(ctx)
    assert ctx.jit_log() == ""
    assert dt < 0.5, "second call with new hyper-parameters took %.2f s: recompiled?" % dt
    ref = PU.reference(oracle, dict(w, kernel=kern2))
    e = PU.errors(ref, out["loglik"][0], out["mean"][0], out["var"][0], floor=PU.prior_sd(oracle, dict(w, kernel=kern2)))
    assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, e


def test_tiered_specialisation_keeps_results(ctx, oracle):
    """automatic mode: after 32 calls with one kernel structure the specialised kernels take over
    (include/smolgp.h, option "jit"); results before and after agree and match the oracle"""
    w = W.make("fig3", N=300)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    first = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
    for i in range(40):
        kern = [dict(k, sigma=k["sigma"] * (1.0 + 0.01 * i)) for k in w["kernel"]]
        ctx.smolgp_loglik_host(ev, kern, w["y"], w["sigma"])
    last = ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
    assert ctx.jit_log() == ""
    for k in ("loglik", "mean", "var"):
        np.testing.assert_allclose(first[k], last[k], rtol=1e-11, atol=1e-13)
    ref = PU.reference(oracle, w)
    e = PU.errors(ref, last["loglik"][0], last["mean"][0], last["var"][0], floor=PU.prior_sd(oracle, w))
    assert e["ll"] <= PU.LL_RTOL and e["mean"] <= PU.POST_RTOL and e["var"] <= PU.POST_RTOL, e


def test_profile_modes(ctx):
    """smolgp_profile (include/smolgp.h): 1 brackets every launch, 2 + id only the launches of kernel id (what
    bench.py uses inside its timed region), 0 none; the launch counter counts in every mode"""
    w = W.make(2, N=2000)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    try:
        ctx.set_option("chunk", 32)
        ctx.profile(True)
        l0 = ctx.launch_count()
        ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
        n_launch = ctx.launch_count() - l0
        every = ctx.profile_read()
        assert {"k_disc", "k_fold0", "k_foldD", "k_downD", "k_down0"} <= set(every)
        assert sum(c for _, c in every.values()) == n_launch
        ctx.profile("k_down0")
        ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
        one = ctx.profile_read()
        assert set(one) == {"k_down0"} and one["k_down0"][1] == every["k_down0"][1] and one["k_down0"][0] > 0.0
        ctx.profile(False)
        ctx.smolgp_condition_host(ev, w["kernel"], w["y"], w["sigma"])
        assert ctx.profile_read() == {}
        with pytest.raises(Exception):
            ctx.profile(2 + 1000)
    finally:
        ctx.profile(False)
        _reset(ctx)


# ---------------------------------------------------------------------------------------------
# instantaneous data (the paper's section 2, K = N events) against the oracle's section-2
# sequential algorithm and the dense definition
# ---------------------------------------------------------------------------------------------
INSTANT_KERNELS = {
    "fig1": ([W.comp(W.SHO, 1.0, 2 * np.pi / 300.0, 2.0), W.comp(W.MATERN52, 0.7, 900.0)], 1),   # Fig. 1: SHO + Matern-5/2
    "masked": ([W.comp(W.SHO, 1.0, 2 * np.pi / 330.0, 10.0), W.comp(W.MATERN32, 0.5, 900.0, inst_mask=2)], 2),
    "qp": ([W.comp(W.MATERN32_X_PERIODIC, 1.0, 4000.0, 9000.0, 1.0, order=2)], 1),
}


def _instant_data(rng, kern, N, ninst, span, ties=False):
    t = np.sort(rng.uniform(0, span, N))
    if ties:
        t[1::9] = t[0::9][: t[1::9].size]
    inst = rng.integers(0, ninst, N).astype(np.int32)
    sigma = rng.uniform(0.1, 0.4, N)
    y = W.synth_y(rng, kern, t, t + 1e-9, inst, sigma)
    return t, inst, y, sigma


@pytest.mark.parametrize("opt", ["auto", "deep", "ragged", "jit", "sequential"])
@pytest.mark.parametrize("name", sorted(INSTANT_KERNELS))
def test_instantaneous_data_matches_oracle(ctx, oracle, name, opt):
    kern, ninst = INSTANT_KERNELS[name]
    rng = np.random.default_rng(31)
    t, inst, y, sigma = _instant_data(rng, kern, 1500, ninst, 1500 * 40.0, ties=(name == "masked"))
    p = rng.permutation(t.size)   # samples in arbitrary order
    t, inst, y, sigma = t[p], inst[p], y[p], sigma[p]
    tq = np.concatenate([rng.uniform(t.min() - 300, t.max() + 300, 50), t[:3]])
    for k, v in SCAN_OPTS[opt]:
        ctx.set_option(k, v)
    try:
        ev = ctx.smolgp_build_events_instant_host(t, inst, ninst)
        et, kind, ei, ex = ev.export()
        out = ctx.smolgp_condition_host(ev, kern, y, sigma, t_query=tq, query_instrument=ninst - 1)
        ll = ctx.smolgp_loglik_host(ev, kern, y, sigma)
    finally:
        _reset(ctx)
    # the stream: K = N observe events by (time, instrument, index)
    order = np.lexsort((np.arange(t.size), inst, t))
    assert et.size == t.size and np.array_equal(et, t[order]) and np.array_equal(ex, order) and np.all(kind == 0) and np.array_equal(ei, inst[order])
    ref = oracle.ssm_instant(kern, ninst, t, inst, y, sigma, tq=tq, query_inst=ninst - 1)
    assert abs(out["loglik"][0] - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])
    assert abs(ll[0] - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])
    psd = np.sqrt(np.array([oracle.kernel(kern, int(q), int(q), np.zeros(1))[0] for q in inst]))   # prior sd of the sampled latent
    assert np.max(np.abs(out["mean"][0] - ref["mean"]) / (np.abs(ref["mean"]) + psd)) <= PU.POST_RTOL
    assert np.max(np.abs(out["var"][0] - ref["var"]) / ref["var"]) <= PU.POST_RTOL
    k0 = float(oracle.kernel(kern, ninst - 1, ninst - 1, np.zeros(1))[0])
    assert np.max(np.abs(out["mean_query"][0] - ref["mq"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mq"])))
    assert np.max(np.abs(out["var_query"][0] - ref["vq"]) / ref["vq"]) <= 1e-8


def test_instantaneous_data_matches_dense_definition(ctx, oracle):
    rng = np.random.default_rng(32)
    for name in sorted(INSTANT_KERNELS):
        kern, ninst = INSTANT_KERNELS[name]
        t, inst, y, sigma = _instant_data(rng, kern, 160, ninst, 160 * 60.0, ties=True)
        tq = rng.uniform(t.min() - 200, t.max() + 200, 30)
        ev = ctx.smolgp_build_events_instant_host(t, inst, ninst)
        out = ctx.smolgp_condition_host(ev, kern, y, sigma, t_query=tq, query_instrument=0)
        ref = oracle.dense_instant(kern, t, inst, y, sigma, tq=tq, query_inst=0)
        assert abs(out["loglik"][0] - ref["loglik"]) <= 1e-9 * abs(ref["loglik"])
        k0 = float(oracle.kernel(kern, 0, 0, np.zeros(1))[0])
        assert np.max(np.abs(out["mean"][0] - ref["mean"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mean"])))
        assert np.max(np.abs(out["var"][0] - ref["var"])) <= 1e-8 * k0
        assert np.max(np.abs(out["mean_query"][0] - ref["mq"])) <= 1e-8 * (np.sqrt(k0) + np.max(np.abs(ref["mq"])))
        assert np.max(np.abs(out["var_query"][0] - ref["vq"])) <= 1e-8 * k0


def test_instantaneous_data_full_size_fig1_kernel(ctx, oracle):
    """N = 1e5 samples, SHO + Matern-5/2 (the Fig. 1 kernel): device-pointer entry point, automatic plan; loglik
    against the long-double section-2 oracle, posterior on the whole series"""
    import torch
    kern, ninst = INSTANT_KERNELS["fig1"]
    rng = np.random.default_rng(33)
    N = 100000
    t = np.cumsum(rng.uniform(5.0, 60.0, N))
    inst = np.zeros(N, np.int32)
    sigma = np.full(N, 0.3)
    sub = np.random.default_rng(34)
    y = np.concatenate([W.synth_y(np.random.default_rng(35), kern, t[a:a + 20000], t[a:a + 20000] + 1e-9, inst[a:a + 20000], np.zeros(min(20000, N - a)))
                        for a in range(0, N, 20000)]) + sigma * sub.standard_normal(N)
    dev = torch.device("cuda:0")
    ev = ctx.smolgp_build_events_instant(torch.tensor(t, device=dev), torch.tensor(inst, device=dev), 1)
    out = ctx.smolgp_condition(ev, kern, torch.tensor(y, device=dev), torch.tensor(sigma, device=dev))
    torch.cuda.synchronize()
    ref = oracle.ssm_instant(kern, 1, t, inst, y, sigma)
    assert abs(float(out["loglik"][0]) - ref["loglik"]) <= PU.LL_RTOL * abs(ref["loglik"])
    k0 = float(oracle.kernel(kern, 0, 0, np.zeros(1))[0])
    assert np.max(np.abs(out["mean"][0].cpu().numpy() - ref["mean"]) / (np.abs(ref["mean"]) + np.sqrt(k0))) <= PU.POST_RTOL
    assert np.max(np.abs(out["var"][0].cpu().numpy() - ref["var"]) / ref["var"]) <= PU.POST_RTOL


def test_instantaneous_events_validation(ctx):
    from paper_2601_02527_b200.binding import SmolgpError
    t, ins = np.array([3.0, 1.0, 2.0]), np.zeros(3, np.int32)
    ctx.smolgp_build_events_instant_host(t, ins, 1).free()
    with pytest.raises(SmolgpError) as e:
        ctx.smolgp_build_events_instant_host(np.array([3.0, np.nan, 2.0]), ins, 1)
    assert e.value.rc == -1
    with pytest.raises(SmolgpError) as e:
        ctx.smolgp_build_events_instant_host(t, np.array([0, 1, 0], np.int32), 1)
    assert e.value.rc == -1


# ---------------------------------------------------------------------------------------------
# gradient of the log-likelihood w.r.t. every hyper-parameter against the oracle's
# (central differences of the long-double sequential likelihood, pinned to the dense analytic derivative)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,N,batch", [(1, 600, None), (2, 900, None), (3, 500, None), (4, 500, None), (5, 200, 3)])
def test_loglik_gradient_matches_oracle(ctx, oracle, cfg, N, batch):
    w = W.make(cfg, N=N, batch=batch)
    ev = ctx.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
    ll, g = ctx.smolgp_loglik_grad_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
    for s in ([None] if batch is None else range(batch)):
        i = 0 if s is None else s
        y = w["y"] if s is None else w["y"][s]
        a = 1.0 if s is None else float(w["amp"][s])
        fn = lambda k: oracle.ssm([dict(c, sigma=c["sigma"] * a) for c in k], w["n_inst"], w["t_start"], w["t_end"], w["instrument"], y, w["sigma"],
                                  flags=oracle.FLAG_IDLE_ZERO | oracle.FLAG_TWO_FILTER, want_post=False)["loglik"]
        ref = oracle.loglik_grad(w["kernel"], fn)
        assert abs(ll[i] - fn(w["kernel"])) <= PU.LL_RTOL * abs(ll[i])
        scale = np.max(np.abs(ref * np.array([[c["sigma"], c["p0"], max(c["p1"], 1e-300), max(c["p2"], 1e-300)] for c in w["kernel"]])))  # largest |dL/dlog theta|
        for c, comp in enumerate(w["kernel"]):
            for p in range(oracle.FAMILY_PARAMS[int(comp["family"])]):
                th = comp[oracle.PARAMS[p]]
                assert abs(g[i, c, p] - ref[c, p]) * th <= 1e-6 * scale, (cfg, s, c, p, g[i, c, p], ref[c, p])
            assert np.all(g[i, c, oracle.FAMILY_PARAMS[int(comp["family"])]:] == 0.0)


def test_loglik_gradient_device_pointers_and_instant(ctx, oracle):
    import torch
    kern, ninst = INSTANT_KERNELS["fig1"]
    rng = np.random.default_rng(41)
    t, inst, y, sigma = _instant_data(rng, kern, 800, ninst, 800 * 40.0)
    dev = torch.device("cuda:0")
    ev = ctx.smolgp_build_events_instant_host(t, inst, ninst)
    ll, g = ctx.smolgp_loglik_grad(ev, kern, torch.tensor(y, device=dev), torch.tensor(sigma, device=dev))
    fn = lambda k: oracle.ssm_instant(k, ninst, t, inst, y, sigma, want_post=False)["loglik"]
    ref = oracle.loglik_grad(kern, fn)
    scale = np.max(np.abs(ref * np.array([[c["sigma"], c["p0"], max(c["p1"], 1e-300), 1e-300] for c in kern])))
    for c, comp in enumerate(kern):
        for p in range(oracle.FAMILY_PARAMS[int(comp["family"])]):
            assert abs(g[0, c, p] - ref[c, p]) * comp[oracle.PARAMS[p]] <= 1e-6 * scale


def test_shipped_structures_use_the_ahead_of_time_modules(ctx):
    """the structures of BASELINE.json's configs (and fig2 / fig3 / the instantaneous Fig. 1 kernel) are compiled when the
    library is built (_build.py: PREBUILT) and used from the first call, without NVRTC"""
    from paper_2601_02527_b200 import binding as B
    c2 = B.Context(0)   # a fresh ctx: nothing is "hot" yet
    try:
        for cfg, N, batch in [(1, 200, None), (2, 300, None), (3, 300, None), (4, 300, None), (5, 100, 2), ("fig2", 100, None), ("fig3", 150, None)]:
            w = W.make(cfg, N=N, batch=batch, n_features=4)
            ev = c2.smolgp_build_events_host(w["t_start"], w["t_end"], w["instrument"], w["n_inst"])
            c2.smolgp_loglik_host(ev, w["kernel"], w["y"], w["sigma"], amp=w["amp"])
            assert "prebuilt=1" in c2.plan_info() and "kernels=reg" in c2.plan_info(), (cfg, c2.plan_info())
            ev.free()
        w = W.make("instant", N=300, n_features=4)
        ev = c2.smolgp_build_events_instant_host(w["t_start"], w["instrument"], 1)
        c2.smolgp_loglik_host(ev, w["kernel"], w["y"], w["sigma"])
        assert "prebuilt=1" in c2.plan_info(), c2.plan_info()
        assert c2.jit_log() == ""
    finally:
        c2.close()
