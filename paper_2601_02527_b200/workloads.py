"""Seeded synthetic workload generators shaped like the paper's (arXiv:2601.02527, P:541-549:
all of the paper's experiments use synthetic draws from GP priors) and like BASELINE.json's five
configs.  This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle:
it produces plain numpy input arrays (exposure starts/ends, instrument labels, data, noise) and
the kernel description.  It holds none of the method's arithmetic (no state-space model, no
discretisation, no filter, no covariance matrix): the data y are synthesised spectrally, as a
sum of random sinusoids whose frequencies are drawn from each kernel component's normalised
power spectral density, averaged in closed form over each exposure, plus white noise.  In the
limit of many sinusoids that is a draw from the GP prior with that kernel (Bochner), which is
what BASELINE.json's "y drawn from the dense integrated GP" / "sequential-SSM draw" produce; see
DESIGN.md, "Input recipe".

Kernel description: list of dicts {family, order, inst_mask, sigma, p0, p1, p2} with
  MATERN32 / MATERN52 : p0 = ell [s]
  SHO                 : p0 = omega0 [rad/s], p1 = Q
  MATERN32_X_PERIODIC : p0 = ell, p1 = period, p2 = ell_periodic, order = J
All times in seconds (SURVEY reading c14).
"""
import numpy as np

MATERN32, MATERN52, SHO, MATERN32_X_PERIODIC = 0, 1, 2, 3
DAY = 86400.0


def comp(family, sigma, p0, p1=0.0, p2=0.0, order=0, inst_mask=0xFFFFFFFF):
    return dict(family=family, order=order, inst_mask=inst_mask, sigma=sigma, p0=p0, p1=p1, p2=p2)


# ------------------------------------------------------------------------------------------
# exposure time tables
# ------------------------------------------------------------------------------------------
def _sequential(rng, N, first, length, gap):
    """one instrument, back-to-back-with-gaps: s_{n+1} = e_n + gap()."""
    ts, te = np.empty(N), np.empty(N)
    t = first
    for i in range(N):
        ts[i] = t
        te[i] = t + length()
        t = te[i] + gap()
    return ts, te


def _daily(rng, n_target, specs, window=28800.0, day=DAY):
    """several instruments observing in daily windows (config 3/4 shape).  specs: list of
    (length_fn, dead_fn or None, cadence_fn or None).  Returns exposures sorted by start."""
    ts, te, inst = [], [], []
    total, d = 0, 0
    while total < n_target:
        for q, (length, dead, cadence) in enumerate(specs):
            t = d * day + rng.uniform(0.0, 60.0)
            while True:
                L = length()
                if t + L > d * day + window:
                    break
                ts.append(t); te.append(t + L); inst.append(q)
                total += 1
                t = t + cadence() if cadence is not None else t + L + dead()
        d += 1
    ts, te, inst = np.array(ts), np.array(te), np.array(inst, dtype=np.int32)
    o = np.argsort(ts, kind="stable")[:n_target]
    return ts[o], te[o], inst[o]


# ------------------------------------------------------------------------------------------
# spectral synthesis of y
# ------------------------------------------------------------------------------------------
def _sho_freqs(rng, w0, Q, J):
    """frequencies ~ normalised SHO PSD  S(w) ~ 1/((w^2-w0^2)^2 + w0^2 w^2/Q^2)  by rejection from a
    Cauchy proposal centred on the resonance."""
    a = w0 / (2 * Q)
    b = w0 * np.sqrt(max(1 - 1 / (4 * Q * Q), 0.0)) if Q > 0.5 else 0.0
    S = lambda w: 1.0 / ((w * w - w0 * w0) ** 2 + (w0 * w / Q) ** 2)
    g = lambda w: 0.5 * (a / np.pi) * (1 / ((w - b) ** 2 + a * a) + 1 / ((w + b) ** 2 + a * a))
    grid = np.linspace(-6 * w0, 6 * w0, 20001)
    Mb = 1.05 * np.max(S(grid) / g(grid))
    out = np.empty(0)
    while out.size < J:
        w = b * rng.choice([-1.0, 1.0], size=4 * J) + a * rng.standard_cauchy(4 * J)
        keep = rng.uniform(size=4 * J) * Mb * g(w) < S(w)
        out = np.concatenate([out, w[keep]])
    return out[:J]


def _periodic_q2(order, ell_p):
    from scipy.special import ive
    a = 1.0 / (ell_p * ell_p)
    q2 = np.array([(1.0 if j == 0 else 2.0) * ive(j, a) for j in range(order + 1)])
    return q2


def _component_freqs(rng, c, J):
    """(frequencies [J], total variance k(0)) of one component."""
    f = c["family"]
    if f == MATERN32:
        return rng.standard_t(3, J) / c["p0"], c["sigma"] ** 2
    if f == MATERN52:
        return rng.standard_t(5, J) / c["p0"], c["sigma"] ** 2
    if f == SHO:
        return _sho_freqs(rng, c["p0"], c["p1"], J), c["sigma"] ** 2
    if f == MATERN32_X_PERIODIC:
        q2 = _periodic_q2(c["order"], c["p2"])
        j = rng.choice(len(q2), size=J, p=q2 / q2.sum())
        w = rng.standard_t(3, J) / c["p0"] + rng.choice([-1.0, 1.0], J) * j * (2 * np.pi / c["p1"])
        return w, c["sigma"] ** 2 * q2.sum()
    raise ValueError(f)


def synth_y(rng, kernel, ts, te, inst, sigma, batch=None, amp=None, n_features=256):
    """y[n] = sum_c [c in inst_n] sqrt(2 k_c(0)/J) sum_j <cos(w_j t + phi_j)>_n + sigma_n eps_n,
    <.>_n the average over exposure n: cos(w t_mid + phi) sinc(w delta / 2)."""
    N = ts.size
    tm, half = 0.5 * (ts + te), 0.5 * (te - ts)
    B = 1 if batch is None else batch
    y = np.zeros((B, N))
    for c in kernel:
        w, var = _component_freqs(rng, c, n_features)
        sel = ((c["inst_mask"] >> inst.astype(np.int64)) & 1).astype(np.float64)  # [N]
        arg = np.outer(tm, w)                                                      # [N, J]
        sinc = np.sinc(np.outer(half, w) / np.pi) * sel[:, None]
        Cm, Sm = np.cos(arg) * sinc, np.sin(arg) * sinc
        phi = rng.uniform(0, 2 * np.pi, size=(n_features, B))
        y += (np.sqrt(2 * var / n_features) * (Cm @ np.cos(phi) - Sm @ np.sin(phi))).T
    if amp is not None:
        y *= amp[:, None]
    y += sigma[None, :] * rng.standard_normal((B, N))
    return y if batch is not None else y[0]


# ------------------------------------------------------------------------------------------
# the five BASELINE.json configs, plus the paper's Fig. 2 / Fig. 3 shapes
# ------------------------------------------------------------------------------------------
FULL_N = {1: 1000, 2: 20000, 3: 100000, 4: 1000000, 5: 2048, "fig2": 400, "fig3": 600, "instant": 100000}
FULL_BATCH = {5: 4096}


def make(cfg, N=None, batch=None, seed=None, n_features=None):
    """Returns dict(name, kernel, n_inst, t_start, t_end, instrument, y, sigma, amp, batch)."""
    N = FULL_N[cfg] if N is None else int(N)
    default_seed = {1: 0, 2: 1, 3: 2, 4: 3, 5: 4, "fig2": 12, "fig3": 13, "instant": 14}[cfg]
    rng = np.random.default_rng(default_seed if seed is None else seed)
    U = rng.uniform
    amp = None
    if cfg == 1:
        name = "cfg1: single series, Matern-3/2 (ell=600 s), non-overlapping exposures"
        kernel = [comp(MATERN32, 1.0, 600.0)]
        ts, te = _sequential(rng, N, U(10, 600), lambda: U(50, 300), lambda: U(10, 600))
        inst = np.zeros(N, dtype=np.int32)
        noise = np.array([0.1])
    elif cfg == 2:
        name = "cfg2: two overlapping instruments, SHO (330 s, Q=10)"
        kernel = [comp(SHO, 1.0, 2 * np.pi / 330.0, 10.0)]
        NA = (3 * N) // 4
        NB = N - NA
        tsA = 60.0 * np.arange(NA)
        teA = tsA + 55.0
        tsB, teB = _sequential(rng, NB, U(0, 60), lambda: U(140, 178), lambda: U(2, 40))
        ts, te = np.concatenate([tsA, tsB]), np.concatenate([teA, teB])
        inst = np.concatenate([np.zeros(NA, np.int32), np.ones(NB, np.int32)])
        noise = np.array([0.2, 0.3])
    elif cfg in (3, 4):
        specs = [(lambda: 12.0, None, lambda: 40 + U(0, 1)),
                 (lambda: 55.0, None, lambda: 82 + U(0, 1)),
                 (lambda: U(140, 178), lambda: 25 + U(0, 1), None)]
        if cfg == 3:
            name = "cfg3: quasiperiodic Matern-3/2(20 d) x periodic(25 d, order 4), 3 instruments"
            kernel = [comp(MATERN32_X_PERIODIC, 1.0, 20 * DAY, 25 * DAY, 1.0, order=4)]
            noise = np.array([0.1, 0.2, 0.3])
        else:
            name = "cfg4: shared SHO(330 s)+Matern-5/2(1 d) + per-instrument Matern-3/2, 4 instruments"
            specs.append((lambda: 300.0, None, lambda: 330 + U(0, 1)))
            kernel = [comp(SHO, 1.0, 2 * np.pi / 330.0, 10.0), comp(MATERN52, 1.0, DAY)] + \
                     [comp(MATERN32, 0.5, 3600.0, inst_mask=1 << q) for q in range(4)]
            noise = np.array([0.2, 0.3, 0.3, 0.25])
        ts, te, inst = _daily(rng, N, specs)
    elif cfg == 5:
        name = "cfg5: batched spectral pixels, Matern-5/2(1 d)+SHO(330 s), shared grid, 2 instruments"
        kernel = [comp(MATERN52, 1.0, DAY), comp(SHO, 1.0, 2 * np.pi / 330.0, 10.0)]
        NA = int(round(N * 1734 / 2048))
        NB = N - NA
        tsA = 60.0 * np.arange(NA); teA = tsA + 55.0
        tsB = 17.5 + 330.0 * np.arange(NB); teB = tsB + 300.0
        ts, te = np.concatenate([tsA, tsB]), np.concatenate([teA, teB])
        inst = np.concatenate([np.zeros(NA, np.int32), np.ones(NB, np.int32)])
        noise = np.array([0.2, 0.3])
        batch = FULL_BATCH[5] if batch is None else int(batch)
        amp = np.exp(rng.uniform(np.log(0.1), np.log(10.0), size=batch))
    elif cfg == "fig2":
        name = "fig2 shape (P:531,543): one instrument, SHO ~300 s, 180 s exposures, no dead time"
        kernel = [comp(SHO, 1.0, 2 * np.pi / 300.0, 2.0)]
        ts = 180.0 * np.arange(N); te = ts + 180.0
        inst = np.zeros(N, dtype=np.int32)
        noise = np.array([0.3])
    elif cfg == "fig3":
        name = "fig3 shape (P:535,545): 55 s fixed + N(180,30) s exposures, frequent overlap"
        kernel = [comp(SHO, 1.0, 2 * np.pi / 300.0, 2.0)]
        NA = (2 * N) // 3
        NB = N - NA
        tsA = 60.0 * np.arange(NA); teA = tsA + 55.0
        tsB, teB = _sequential(rng, NB, U(0, 30), lambda: max(60.0, rng.normal(180, 30)), lambda: U(5, 25))
        ts, te = np.concatenate([tsA, tsB]), np.concatenate([teA, teB])
        inst = np.concatenate([np.zeros(NA, np.int32), np.ones(NB, np.int32)])
        noise = np.array([0.3, 0.3])
    elif cfg == "instant":
        name = "instantaneous samples (paper section 2; Fig. 1 kernel P:334: SHO + Matern-5/2), one instrument, gaps U[5,60] s"
        kernel = [comp(SHO, 1.0, 2 * np.pi / 300.0, 2.0), comp(MATERN52, 0.7, 900.0)]
        ts = np.cumsum(U(5.0, 60.0, N))
        te = ts + 1e-9   # only used by the spectral synthesis of y (sinc(w 1e-9 / 2) = 1): the samples are instantaneous
        inst = np.zeros(N, dtype=np.int32)
        noise = np.array([0.3])
    else:
        raise ValueError(cfg)
    n_inst = int(noise.size)
    sigma = noise[inst]
    J = n_features if n_features is not None else (64 if batch else (32 if N > 200000 else 256))
    # y synthesis costs O(N J) sincos: chunk it for the large configs
    if batch is None and N > 50000:
        y = np.empty(N)
        sub = np.random.default_rng(rng.integers(1 << 62))
        # same frequencies/phases for every chunk: re-seed identically and slice exposures
        seed_y = int(sub.integers(1 << 62))
        for a in range(0, N, 20000):
            sl = slice(a, min(N, a + 20000))
            r2 = np.random.default_rng(seed_y)
            y[sl] = synth_y(r2, kernel, ts[sl], te[sl], inst[sl], np.zeros(sl.stop - sl.start), n_features=J)
        y += sigma * np.random.default_rng(seed_y + 1).standard_normal(N)
    else:
        y = synth_y(rng, kernel, ts, te, inst, sigma, batch=batch, amp=amp, n_features=J)
    return dict(name=name, cfg=cfg, kernel=kernel, n_inst=n_inst, t_start=ts, t_end=te, instrument=inst,
                y=y, sigma=sigma, amp=amp, batch=batch, instant=(cfg == "instant"))
