"""ctypes loader for the CPU oracle (oracle/smolgp_oracle.c) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares nothing with paper_2601_02527_b200/ (the CUDA product path).

Two builds of the same C file (see its header): ``f80`` = x87 long double (the parity
reference) and ``f64`` = plain double, -O3 (the timed CPU baseline).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "smolgp_oracle.c")

FAM_MATERN32, FAM_MATERN52, FAM_SHO, FAM_MATERN32_X_PERIODIC = 0, 1, 2, 3
FLAG_IDLE_ZERO, FLAG_TWO_FILTER = 1, 2


class OComp(C.Structure):
    _fields_ = [("family", C.c_int32), ("order", C.c_int32), ("inst_mask", C.c_uint32),
                ("sigma", C.c_double), ("p0", C.c_double), ("p1", C.c_double), ("p2", C.c_double)]


def build(force=False):
    """Compile the two shared objects with gcc if missing or stale."""
    out = {}
    for tag, flags in (("f80", ["-O2", "-DREAL_IS_LONG_DOUBLE"]), ("f64", ["-O3", "-march=native"])):
        so = os.path.join(_HERE, "liboracle_%s.so" % tag)
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", "-fPIC", "-shared", *flags, "-o", so, _SRC, "-lquadmath", "-lm"])
        out[tag] = so
    return out


_libs = {}


def _lib(tag):
    if tag not in _libs:
        so = build()[tag]
        _libs[tag] = C.CDLL(so)
    return _libs[tag]


def _comps(kernel):
    """kernel: list of dicts {family, order, inst_mask, sigma, p0, p1, p2}."""
    arr = (OComp * len(kernel))()
    for i, k in enumerate(kernel):
        arr[i] = OComp(int(k["family"]), int(k.get("order", 0)), int(k["inst_mask"]), float(k["sigma"]),
                       float(k.get("p0", 0.0)), float(k.get("p1", 0.0)), float(k.get("p2", 0.0)))
    return arr


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def kernel(kern, ia, ib, tau):
    tau = _d(tau)
    out = np.empty_like(tau)
    rc = _lib("f80").oracle_kernel(len(kern), _comps(kern), ia, ib, tau.size, _p(tau), _p(out))
    assert rc == 0, rc
    return out


def kff(kern, ts, te, inst):
    ts, te = _d(ts), _d(te)
    inst = np.ascontiguousarray(inst, dtype=np.int32)
    N = ts.size
    K = np.empty((N, N))
    rc = _lib("f80").oracle_kff(len(kern), _comps(kern), N, _p(ts), _p(te), _p(inst, C.c_int32), _p(K))
    assert rc == 0, rc
    return K


def model_dim(kern, ninst):
    return _lib("f80").oracle_model_dim(len(kern), _comps(kern), ninst)


def ssm_matrices(kern, ninst):
    n = model_dim(kern, ninst)
    d = n - ninst
    Ft, Wt, Pinf, H = np.empty((n, n)), np.empty((n, n)), np.empty((d, d)), np.empty((ninst, d))
    rc = _lib("f80").oracle_ssm_matrices(len(kern), _comps(kern), ninst, _p(Ft), _p(Wt), _p(Pinf), _p(H))
    assert rc == 0, rc
    return Ft, Wt, Pinf, H


def discretise(kern, ninst, dt, prec="f80"):
    n = model_dim(kern, ninst)
    A, Q = np.empty((n, n)), np.empty((n, n))
    f = _lib(prec).oracle_discretise
    f.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
    rc = f(len(kern), C.cast(_comps(kern), C.c_void_p), ninst, float(dt), A.ctypes.data, Q.ctypes.data)
    assert rc == 0, rc
    return A, Q


def events(ts, te, inst):
    ts, te = _d(ts), _d(te)
    inst = np.ascontiguousarray(inst, dtype=np.int32)
    N = ts.size
    t = np.empty(2 * N)
    kind, io, idx = (np.empty(2 * N, dtype=np.int32) for _ in range(3))
    rc = _lib("f80").oracle_events(N, _p(ts), _p(te), _p(inst, C.c_int32), _p(t), _p(kind, C.c_int32),
                                   _p(io, C.c_int32), _p(idx, C.c_int32))
    assert rc == 0, rc
    return t, kind, io, idx


def dense(kern, ts, te, inst, y, sigma, tq=None, query_inst=0, want_post=True):
    """The definition: dense integrated-GP solve. Returns dict(loglik, mean, var, mq, vq)."""
    ts, te, y, sigma = _d(ts), _d(te), _d(y), _d(sigma)
    inst = np.ascontiguousarray(inst, dtype=np.int32)
    N = ts.size
    M = 0 if tq is None else len(tq)
    tq = _d(tq) if M else None
    ll = C.c_double()
    mean = np.empty(N) if want_post else None
    var = np.empty(N) if want_post else None
    mq = np.empty(M) if M else None
    vq = np.empty(M) if M else None
    rc = _lib("f80").oracle_dense(len(kern), _comps(kern), N, _p(ts), _p(te), _p(inst, C.c_int32), _p(y),
                                  _p(sigma), M, _p(tq), query_inst, C.byref(ll), _p(mean), _p(var),
                                  _p(mq), _p(vq))
    if rc != 0:
        raise RuntimeError("oracle_dense rc=%d" % rc)
    return dict(loglik=ll.value, mean=mean, var=var, mq=mq, vq=vq)


def ssm(kern, ninst, ts, te, inst, y, sigma, flags=FLAG_TWO_FILTER, zprior=1.0, tq=None, query_inst=0,
        want_post=True, prec="f80"):
    """The paper's sequential algorithm. Returns dict(loglik, mean, var, mq, vq, rc)."""
    ts, te, y, sigma = _d(ts), _d(te), _d(y), _d(sigma)
    inst = np.ascontiguousarray(inst, dtype=np.int32)
    N = ts.size
    M = 0 if tq is None else len(tq)
    tq = _d(tq) if M else None
    ll = C.c_double()
    mean = np.empty(N) if want_post else None
    var = np.empty(N) if want_post else None
    mq = np.empty(M) if M else None
    vq = np.empty(M) if M else None
    f = _lib(prec).oracle_ssm
    f.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int] + [C.c_void_p] * 5 + \
                 [C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_int] + [C.c_void_p] * 5
    ptr = lambda a: None if a is None else a.ctypes.data
    rc = f(len(kern), C.cast(_comps(kern), C.c_void_p), ninst, N, ptr(ts), ptr(te), ptr(inst), ptr(y),
           ptr(sigma), int(flags), float(zprior), M, ptr(tq), query_inst, C.addressof(ll), ptr(mean),
           ptr(var), ptr(mq), ptr(vq))
    if rc != 0:
        raise RuntimeError("oracle_ssm rc=%d" % rc)
    g = _lib(prec).oracle_ssm_disc_seconds  # instrumentation: seconds of this call spent in the discretisation
    g.restype = C.c_double
    return dict(loglik=ll.value, mean=mean, var=var, mq=mq, vq=vq, disc_seconds=float(g()))


def ssm_sqrt(kern, ninst, ts, te, inst, y, sigma, zprior=1.0, want_post=True, prec="f80"):
    """The sequential passes in square-root (Cholesky-factor) array form (oracle_ssm_sqrt): same
    posterior as ssm(flags=IDLE_ZERO | TWO_FILTER).  Returns dict(loglik, mean, var)."""
    ts, te, y, sigma = _d(ts), _d(te), _d(y), _d(sigma)
    inst = np.ascontiguousarray(inst, dtype=np.int32)
    N = ts.size
    ll = C.c_double()
    mean = np.empty(N) if want_post else None
    var = np.empty(N) if want_post else None
    f = _lib(prec).oracle_ssm_sqrt
    f.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int] + [C.c_void_p] * 5 + [C.c_double] + [C.c_void_p] * 3
    ptr = lambda a: None if a is None else a.ctypes.data
    rc = f(len(kern), C.cast(_comps(kern), C.c_void_p), ninst, N, ptr(ts), ptr(te), ptr(inst), ptr(y), ptr(sigma),
           float(zprior), C.addressof(ll), ptr(mean), ptr(var))
    if rc != 0:
        raise RuntimeError("oracle_ssm_sqrt rc=%d" % rc)
    return dict(loglik=ll.value, mean=mean, var=var)


def _instant(fn, kern, ninst, t, inst, y, sigma, tq, query_inst, want_post, prec):
    t, y, sigma = _d(t), _d(y), _d(sigma)
    inst = np.ascontiguousarray(inst, dtype=np.int32)
    N = t.size
    M = 0 if tq is None else len(tq)
    tq = _d(tq) if M else None
    ll = C.c_double()
    mean = np.empty(N) if want_post else None
    var = np.empty(N) if want_post else None
    mq = np.empty(M) if M else None
    vq = np.empty(M) if M else None
    f = getattr(_lib(prec), fn)
    ptr = lambda a: None if a is None else a.ctypes.data
    head = [len(kern), C.cast(_comps(kern), C.c_void_p)] + ([int(ninst)] if ninst is not None else [])
    f.argtypes = [C.c_int, C.c_void_p] + ([C.c_int] if ninst is not None else []) + [C.c_int] + [C.c_void_p] * 4 + \
                 [C.c_int, C.c_void_p, C.c_int] + [C.c_void_p] * 5
    rc = f(*head, N, ptr(t), ptr(inst), ptr(y), ptr(sigma), M, ptr(tq), int(query_inst), C.addressof(ll), ptr(mean),
           ptr(var), ptr(mq), ptr(vq))
    if rc != 0:
        raise RuntimeError("%s rc=%d" % (fn, rc))
    return dict(loglik=ll.value, mean=mean, var=var, mq=mq, vq=vq)


def dense_instant(kern, t, inst, y, sigma, tq=None, query_inst=0, want_post=True):
    """The definition for instantaneous data (paper section 2): K_ij = k(|t_i - t_j|), Eq. 2.4 / 2.26."""
    return _instant("oracle_dense_instant", kern, None, t, inst, y, sigma, tq, query_inst, want_post, "f80")


def ssm_instant(kern, ninst, t, inst, y, sigma, tq=None, query_inst=0, want_post=True, prec="f80"):
    """The paper's section-2 sequential algorithm (Kalman filter, RTS smoother, Algorithm 1) on instantaneous data."""
    return _instant("oracle_ssm_instant", kern, ninst, t, inst, y, sigma, tq, query_inst, want_post, prec)


PARAMS = ("sigma", "p0", "p1", "p2")
FAMILY_PARAMS = {FAM_MATERN32: 2, FAM_MATERN52: 2, FAM_SHO: 3, FAM_MATERN32_X_PERIODIC: 4}


def loglik_grad(kern, loglik_fn, h=1e-3):
    """d loglik / d (sigma, p0, p1, p2) of every component: the derivative's definition evaluated numerically on
    `loglik_fn(kernel) -> float` (the long-double sequential or dense oracle), by Richardson-extrapolated central
    differences in log theta.  Returns an array [n_comp][4] (0 for parameters the family does not use).  Pinned
    against the dense route's analytic 1/2 tr((alpha alpha^T - C^-1) dC/dtheta) in tests/test_oracle_grad_pins.py."""
    g = np.zeros((len(kern), 4))
    for c, comp in enumerate(kern):
        for p in range(FAMILY_PARAMS[int(comp["family"])]):
            th = float(comp[PARAMS[p]])
            f = []
            for mult in (np.exp(h), np.exp(-h), np.exp(2 * h), np.exp(-2 * h)):
                k2 = [dict(x) for x in kern]
                k2[c][PARAMS[p]] = th * mult
                f.append(loglik_fn(k2))
            d1, d2 = (f[0] - f[1]) / (2 * h), (f[2] - f[3]) / (4 * h)
            g[c, p] = (4 * d1 - d2) / 3 / th
    return g
