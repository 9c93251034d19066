"""Thin ctypes binding of libsmolgp_b200.so (include/smolgp.h).  Argument marshalling only: every
step of the path runs inside the CUDA library.  Device entry points take torch CUDA tensors (torch
is used for device memory and streams, nothing else); *_host entry points take numpy arrays.
There is no CPU fallback: loading fails loudly when the library is missing or cannot be built."""
import ctypes as C
import os

import numpy as np

from . import _build

MATERN32, MATERN52, SHO, MATERN32_X_PERIODIC = 0, 1, 2, 3
STATUS = {0: "OK", -1: "EINVAL", -2: "EOVERLAP", -3: "EUNSUPPORTED", -4: "ENOMEM", -5: "ECUDA", -6: "ENUMERIC"}
EXPORTS = ["smolgp_create", "smolgp_destroy", "smolgp_last_error", "smolgp_set_option", "smolgp_build_events",
           "smolgp_build_events_host", "smolgp_build_events_instant", "smolgp_build_events_instant_host", "smolgp_free_events", "smolgp_events_export", "smolgp_loglik",
           "smolgp_loglik_host", "smolgp_loglik_grad", "smolgp_loglik_grad_host", "smolgp_condition", "smolgp_condition_host", "smolgp_discretise_host",
           "smolgp_launch_count", "smolgp_profile", "smolgp_profile_read", "smolgp_kernel_name", "smolgp_jit_log", "smolgp_plan_info", "smolgp_memory_info",
           "smolgp_build_events_noalloc", "smolgp_noalloc_setup", "smolgp_noalloc_max_events", "smolgp_noalloc_scratch_bytes", "smolgp_noalloc_last_error"]
NKERNELS = 11  # SMOLGP_NKERNELS


class SmolgpError(RuntimeError):
    def __init__(self, rc, msg):
        super().__init__("smolgp: %s (%d): %s" % (STATUS.get(rc, "?"), rc, msg))
        self.rc = rc


class _Comp(C.Structure):
    _fields_ = [("family", C.c_int32), ("order", C.c_int32), ("inst_mask", C.c_uint32), ("sigma", C.c_double),
                ("p0", C.c_double), ("p1", C.c_double), ("p2", C.c_double)]


class _Kernel(C.Structure):
    _fields_ = [("n_comp", C.c_int32), ("comp", C.POINTER(_Comp))]


_lib = None


def lib():
    """Loads (building if stale) the shared library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        so = _build.build()
        L = C.CDLL(so)
        vp, i64, i32, dp = C.c_void_p, C.c_int64, C.c_int32, C.c_void_p
        L.smolgp_create.argtypes = [C.POINTER(vp), C.c_int, vp]
        L.smolgp_destroy.argtypes = [vp]
        L.smolgp_destroy.restype = None
        L.smolgp_last_error.argtypes = [vp]
        L.smolgp_last_error.restype = C.c_char_p
        L.smolgp_set_option.argtypes = [vp, C.c_char_p, i64]
        for f in (L.smolgp_build_events, L.smolgp_build_events_host):
            f.argtypes = [vp, i64, dp, dp, dp, i32, C.POINTER(vp)]
        for f in (L.smolgp_build_events_instant, L.smolgp_build_events_instant_host):
            f.argtypes = [vp, i64, dp, dp, i32, C.POINTER(vp)]
        L.smolgp_free_events.argtypes = [vp]
        L.smolgp_free_events.restype = None
        L.smolgp_events_export.argtypes = [vp, vp, dp, dp, dp, dp]
        for f in (L.smolgp_loglik, L.smolgp_loglik_host):
            f.argtypes = [vp, vp, C.POINTER(_Kernel), i64, dp, dp, dp, dp]
        for f in (L.smolgp_loglik_grad, L.smolgp_loglik_grad_host):
            f.argtypes = [vp, vp, C.POINTER(_Kernel), i64, dp, dp, dp, C.c_double, dp, dp]
        for f in (L.smolgp_condition, L.smolgp_condition_host):
            f.argtypes = [vp, vp, C.POINTER(_Kernel), i64, dp, dp, dp, i64, dp, i32, dp, dp, dp, dp, dp]
        L.smolgp_discretise_host.argtypes = [vp, C.POINTER(_Kernel), i32, C.c_double, dp, dp, C.POINTER(i32)]
        L.smolgp_launch_count.argtypes = [vp]
        L.smolgp_launch_count.restype = i64
        L.smolgp_profile.argtypes = [vp, i32]
        L.smolgp_profile_read.argtypes = [vp, dp, dp]
        L.smolgp_kernel_name.argtypes = [i32]
        L.smolgp_kernel_name.restype = C.c_char_p
        L.smolgp_jit_log.argtypes = [vp]
        L.smolgp_jit_log.restype = C.c_char_p
        L.smolgp_plan_info.argtypes = [vp]
        L.smolgp_plan_info.restype = C.c_char_p
        L.smolgp_memory_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), i32]
        L.smolgp_build_events_noalloc.argtypes = [i32, vp, i64, dp, dp, dp, i32, dp, dp, dp, dp, dp, dp]
        L.smolgp_noalloc_setup.argtypes = [i32]
        L.smolgp_noalloc_max_events.restype = i64
        L.smolgp_noalloc_scratch_bytes.restype = i64
        L.smolgp_noalloc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _kernel(kernel):
    arr = (_Comp * len(kernel))()
    for i, k in enumerate(kernel):
        arr[i] = _Comp(int(k["family"]), int(k.get("order", 0)), int(k["inst_mask"]) & 0xFFFFFFFF, float(k["sigma"]),
                       float(k.get("p0", 0.0)), float(k.get("p1", 0.0)), float(k.get("p2", 0.0)))
    return _Kernel(len(kernel), arr), arr


def _dptr(t, dtype="float64", numel=None, name="argument"):
    """device pointer of a contiguous torch CUDA tensor (None -> NULL).  The C ABI sees plain pointers: dtype
    and element count are checked here, where they are still known."""
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous()):
        raise TypeError("%s: expected a contiguous CUDA tensor" % name)
    if str(t.dtype) != "torch." + dtype:
        raise TypeError("%s: expected dtype %s, got %s" % (name, dtype, t.dtype))
    if numel is not None and t.numel() != numel:
        raise ValueError("%s: expected %d elements, got %d" % (name, numel, t.numel()))
    return t.data_ptr()


def _hptr(a, numel=None, name="argument"):
    """host pointer of a C-contiguous numpy array (None -> NULL); float64 / int32 arrays only"""
    if a is None:
        return None
    if not a.flags["C_CONTIGUOUS"] or a.dtype not in (np.float64, np.int32, np.int64):
        raise TypeError("%s: expected a C-contiguous float64 / int32 array" % name)
    if numel is not None and a.size != numel:
        raise ValueError("%s: expected %d elements, got %d" % (name, numel, a.size))
    return a.ctypes.data


class Events:
    def __init__(self, ctx, handle, N, n_inst, instant=False):
        self.ctx, self.handle, self.N, self.n_inst, self.instant = ctx, handle, N, n_inst, instant
        self.K = N if instant else 2 * N

    def export(self):
        K = self.K
        t = np.empty(K)
        kind, inst, idx = (np.empty(K, dtype=np.int32) for _ in range(3))
        self.ctx._check(lib().smolgp_events_export(self.ctx.handle, self.handle, _hptr(t), _hptr(kind), _hptr(inst), _hptr(idx)))
        return t, kind, inst, idx

    def free(self):
        if self.handle:
            lib().smolgp_free_events(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """smolgp_ctx.  stream: a torch.cuda.Stream or None (default stream)."""

    def __init__(self, device=0, stream=None):
        h = C.c_void_p()
        sp = None if stream is None else C.c_void_p(stream.cuda_stream)
        rc = lib().smolgp_create(C.byref(h), int(device), sp)
        if rc != 0:
            raise SmolgpError(rc, "smolgp_create failed (no CUDA device?)")
        self.handle = h
        self.device = device

    def _check(self, rc):
        if rc != 0:
            raise SmolgpError(rc, lib().smolgp_last_error(self.handle).decode())

    def set_option(self, name, value):
        self._check(lib().smolgp_set_option(self.handle, name.encode(), int(value)))

    def launch_count(self):
        return int(lib().smolgp_launch_count(self.handle))

    def profile(self, enable):
        """False/0: off; True/1: every kernel; a kernel name: only that kernel's launches"""
        if isinstance(enable, str):
            enable = 2 + [lib().smolgp_kernel_name(i).decode() for i in range(NKERNELS)].index(enable)
        self._check(lib().smolgp_profile(self.handle, int(enable)))

    def profile_read(self):
        """{kernel name: (milliseconds, launches)} of the window since profile(True) / the last read"""
        ms, cnt = np.zeros(NKERNELS), np.zeros(NKERNELS, dtype=np.int64)
        self._check(lib().smolgp_profile_read(self.handle, _hptr(ms), _hptr(cnt)))
        return {lib().smolgp_kernel_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(NKERNELS) if cnt[i]}

    def jit_log(self):
        return lib().smolgp_jit_log(self.handle).decode()

    def memory_info(self, reset_peak=False):
        """(bytes held now, high-water mark) of this ctx's device memory"""
        cur, peak = C.c_int64(), C.c_int64()
        self._check(lib().smolgp_memory_info(self.handle, C.byref(cur), C.byref(peak), int(bool(reset_peak))))
        return cur.value, peak.value

    def plan_info(self):
        return lib().smolgp_plan_info(self.handle).decode()

    # ---- a1 ----
    def smolgp_build_events(self, t_start, t_end, instrument, n_inst):
        """device tensors: t_start, t_end float64 [N]; instrument int32 [N]"""
        N = t_start.numel()
        h = C.c_void_p()
        self._check(lib().smolgp_build_events(self.handle, N, _dptr(t_start, name="t_start"), _dptr(t_end, numel=N, name="t_end"),
                                              _dptr(instrument, "int32", N, "instrument"), int(n_inst), C.byref(h)))
        return Events(self, h, N, n_inst)

    def smolgp_build_events_host(self, t_start, t_end, instrument, n_inst):
        ts, te = np.ascontiguousarray(t_start, np.float64), np.ascontiguousarray(t_end, np.float64)
        ins = np.ascontiguousarray(instrument, np.int32)
        h = C.c_void_p()
        self._check(lib().smolgp_build_events_host(self.handle, ts.size, _hptr(ts), _hptr(te, ts.size, "t_end"), _hptr(ins, ts.size, "instrument"),
                                                   int(n_inst), C.byref(h)))
        return Events(self, h, ts.size, n_inst)

    # ---- instantaneous data (paper section 2) ----
    def smolgp_build_events_instant(self, t, instrument, n_inst):
        """device tensors: t float64 [N], instrument int32 [N]"""
        N = t.numel()
        h = C.c_void_p()
        self._check(lib().smolgp_build_events_instant(self.handle, N, _dptr(t, name="t"), _dptr(instrument, "int32", N, "instrument"),
                                                      int(n_inst), C.byref(h)))
        return Events(self, h, N, n_inst, instant=True)

    def smolgp_build_events_instant_host(self, t, instrument, n_inst):
        tt = np.ascontiguousarray(t, np.float64)
        ins = np.ascontiguousarray(instrument, np.int32)
        h = C.c_void_p()
        self._check(lib().smolgp_build_events_instant_host(self.handle, tt.size, _hptr(tt), _hptr(ins, tt.size, "instrument"), int(n_inst), C.byref(h)))
        return Events(self, h, tt.size, n_inst, instant=True)

    # ---- a2-a5 ----
    def smolgp_loglik(self, ev, kernel, y, noise_sigma, amp=None, out=None):
        import torch
        batch = 1 if y.dim() == 1 else y.shape[0]
        if out is None:
            out = torch.empty(batch, dtype=torch.float64, device=y.device)
        k, keep = _kernel(kernel)
        self._check(lib().smolgp_loglik(self.handle, ev.handle, C.byref(k), batch, _dptr(y, numel=batch * ev.N, name="y"),
                                        _dptr(noise_sigma, numel=ev.N, name="noise_sigma"), _dptr(amp, numel=batch, name="amp"),
                                        _dptr(out, numel=batch, name="out")))
        return out

    def smolgp_loglik_host(self, ev, kernel, y, noise_sigma, amp=None):
        y = np.ascontiguousarray(y, np.float64)
        batch = 1 if y.ndim == 1 else y.shape[0]
        sg = np.ascontiguousarray(noise_sigma, np.float64)
        am = None if amp is None else np.ascontiguousarray(amp, np.float64)
        out = np.empty(batch)
        k, keep = _kernel(kernel)
        self._check(lib().smolgp_loglik_host(self.handle, ev.handle, C.byref(k), batch, _hptr(y, batch * ev.N, "y"), _hptr(sg, ev.N, "noise_sigma"),
                                             _hptr(am, batch, "amp"), _hptr(out)))
        return out

    # ---- gradient of the log-likelihood ----
    def smolgp_loglik_grad(self, ev, kernel, y, noise_sigma, amp=None, rel_step=0.0):
        """device tensors in; returns (loglik [batch], grad [batch, n_comp, 4]) as numpy arrays: d loglik / d (sigma, p0, p1, p2)"""
        batch = 1 if y.dim() == 1 else y.shape[0]
        ll, g = np.empty(batch), np.zeros((batch, len(kernel), 4))
        k, keep = _kernel(kernel)
        self._check(lib().smolgp_loglik_grad(self.handle, ev.handle, C.byref(k), batch, _dptr(y, numel=batch * ev.N, name="y"),
                                             _dptr(noise_sigma, numel=ev.N, name="noise_sigma"), _dptr(amp, numel=batch, name="amp"),
                                             float(rel_step), _hptr(ll), _hptr(g)))
        return ll, g

    def smolgp_loglik_grad_host(self, ev, kernel, y, noise_sigma, amp=None, rel_step=0.0):
        y = np.ascontiguousarray(y, np.float64)
        batch = 1 if y.ndim == 1 else y.shape[0]
        sg = np.ascontiguousarray(noise_sigma, np.float64)
        am = None if amp is None else np.ascontiguousarray(amp, np.float64)
        ll, g = np.empty(batch), np.zeros((batch, len(kernel), 4))
        k, keep = _kernel(kernel)
        self._check(lib().smolgp_loglik_grad_host(self.handle, ev.handle, C.byref(k), batch, _hptr(y, batch * ev.N, "y"), _hptr(sg, ev.N, "noise_sigma"),
                                                  _hptr(am, batch, "amp"), float(rel_step), _hptr(ll), _hptr(g)))
        return ll, g

    # ---- a2-a7 ----
    def smolgp_condition(self, ev, kernel, y, noise_sigma, amp=None, t_query=None, query_instrument=0, out=None):
        """returns dict(mean, var, loglik[, mean_query, var_query]) of device tensors"""
        import torch
        batch = 1 if y.dim() == 1 else y.shape[0]
        N = ev.N
        if out is None:
            out = dict(mean=torch.empty((batch, N), dtype=torch.float64, device=y.device),
                       var=torch.empty((batch, N), dtype=torch.float64, device=y.device),
                       loglik=torch.empty(batch, dtype=torch.float64, device=y.device))
        M = 0 if t_query is None else t_query.numel()
        if M and "mean_query" not in out:
            out["mean_query"] = torch.empty((batch, M), dtype=torch.float64, device=y.device)
            out["var_query"] = torch.empty((batch, M), dtype=torch.float64, device=y.device)
        k, keep = _kernel(kernel)
        bn, bm = batch * N, batch * M
        self._check(lib().smolgp_condition(self.handle, ev.handle, C.byref(k), batch, _dptr(y, numel=bn, name="y"),
                                           _dptr(noise_sigma, numel=N, name="noise_sigma"), _dptr(amp, numel=batch, name="amp"),
                                           M, _dptr(t_query, name="t_query"), int(query_instrument),
                                           _dptr(out["mean"], numel=bn, name="out[mean]"), _dptr(out["var"], numel=bn, name="out[var]"),
                                           _dptr(out.get("mean_query"), numel=bm, name="out[mean_query]"),
                                           _dptr(out.get("var_query"), numel=bm, name="out[var_query]"),
                                           _dptr(out["loglik"], numel=batch, name="out[loglik]")))
        return out

    def smolgp_condition_host(self, ev, kernel, y, noise_sigma, amp=None, t_query=None, query_instrument=0, out=None):
        y = np.ascontiguousarray(y, np.float64)
        batch = 1 if y.ndim == 1 else y.shape[0]
        N = ev.N
        sg = np.ascontiguousarray(noise_sigma, np.float64)
        am = None if amp is None else np.ascontiguousarray(amp, np.float64)
        tq = None if t_query is None else np.ascontiguousarray(t_query, np.float64)
        M = 0 if tq is None else tq.size
        if out is None:
            out = dict(mean=np.empty((batch, N)), var=np.empty((batch, N)), loglik=np.empty(batch))
            if M:
                out["mean_query"], out["var_query"] = np.empty((batch, M)), np.empty((batch, M))
        k, keep = _kernel(kernel)
        bn, bm = batch * N, batch * M
        self._check(lib().smolgp_condition_host(self.handle, ev.handle, C.byref(k), batch, _hptr(y, bn, "y"), _hptr(sg, N, "noise_sigma"),
                                                _hptr(am, batch, "amp"), M, _hptr(tq), int(query_instrument),
                                                _hptr(out["mean"], bn, "out[mean]"), _hptr(out["var"], bn, "out[var]"),
                                                _hptr(out.get("mean_query"), bm, "out[mean_query]"),
                                                _hptr(out.get("var_query"), bm, "out[var_query]"), _hptr(out["loglik"], batch, "out[loglik]")))
        return out

    def smolgp_discretise_host(self, kernel, n_inst, dt):
        k, keep = _kernel(kernel)
        n = C.c_int32()
        A = np.zeros((32, 32))
        Q = np.zeros((32, 32))
        self._check(lib().smolgp_discretise_host(self.handle, C.byref(k), int(n_inst), float(dt), _hptr(A), _hptr(Q), C.byref(n)))
        nn = n.value
        return A.ravel()[:nn * nn].reshape(nn, nn).copy(), Q.ravel()[:nn * nn].reshape(nn, nn).copy()

    def close(self):
        if self.handle:
            lib().smolgp_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- event build that allocates nothing (include/smolgp.h: smolgp_build_events_noalloc) ----
def smolgp_noalloc_setup(device=0):
    rc = lib().smolgp_noalloc_setup(int(device))
    if rc:
        raise SmolgpError(rc, lib().smolgp_noalloc_last_error().decode())


def smolgp_noalloc_max_events():
    return int(lib().smolgp_noalloc_max_events())


def smolgp_noalloc_scratch_bytes():
    return int(lib().smolgp_noalloc_scratch_bytes())


def smolgp_build_events_noalloc(device, stream, t_start, t_end, instrument, n_inst, t, dt, delta, meta, exposure, flags):
    """All tensors are the caller's CUDA tensors: t_start, t_end (None = instantaneous samples) float64 [N], instrument
    int32 [N]; outputs t, dt, delta float64 [K], meta, exposure int32 [K] (meta holds the packed uint32 bits), flags
    int32 [1]; K = 2N, or N for instantaneous samples.  stream: a cudaStream_t as an integer (0 / None = default)."""
    N = t_start.numel()
    K = N if t_end is None else 2 * N
    rc = lib().smolgp_build_events_noalloc(int(device), C.c_void_p(stream or None), N, _dptr(t_start, name="t_start"),
                                           _dptr(t_end, numel=N, name="t_end"), _dptr(instrument, "int32", N, "instrument"), int(n_inst),
                                           _dptr(t, numel=K, name="t"), _dptr(dt, numel=K, name="dt"), _dptr(delta, numel=K, name="delta"),
                                           _dptr(meta, "int32", K, "meta"), _dptr(exposure, "int32", K, "exposure"),
                                           _dptr(flags, "int32", 1, "flags"))
    if rc:
        raise SmolgpError(rc, lib().smolgp_noalloc_last_error().decode())
