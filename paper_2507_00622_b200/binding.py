"""Thin Python binding of libchaoticus.so (include/chaoticus.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch supplies device
memory and the stream.  Arrays are torch.float64 CUDA tensors in the library's layout
(y [n, n_ic], w [k, n, n_ic], contiguous) and y / w are advanced IN PLACE.  The *_host
functions take numpy arrays (host memory) and go through the library's host-buffer entry
points.  There is no CPU fallback: if the shared library is missing, import of this module
raises, and without a CUDA device every call raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchaoticus.so")

SYS_HENON_HEILES, SYS_COUPLED3, SYS_FPUT, SYS_DOUBLE_PENDULUM = 0, 1, 2, 3
WHAT_INTEGRATE, WHAT_SALI, WHAT_GALI, WHAT_LD, WHAT_LYAP = 0, 1, 2, 3, 4
ST_OK, ST_NONFINITE, ST_UNDERFLOW, ST_MAXSTEPS = 0, 1, 2, 3

EXPORTS = [
    "chaoticus_version", "chaoticus_last_error", "chaoticus_dim", "chaoticus_n_samples",
    "chaoticus_integrate_fixed", "chaoticus_integrate_adaptive", "chaoticus_sali", "chaoticus_gali",
    "chaoticus_ld", "chaoticus_ld_adaptive", "chaoticus_ld_neighbours", "chaoticus_lyap", "chaoticus_ld_host",
    "chaoticus_ld_adaptive_host", "chaoticus_ld_neighbours_host", "chaoticus_sali_host", "chaoticus_gali_host",
    "chaoticus_lyap_host", "chaoticus_integrate_host", "chaoticus_kernel_info", "chaoticus_set_option",
    "chaoticus_ld_neighbour_diffs_noalloc",
]
NOALLOC_MAX_DOUBLES = 1 << 20   # CHS_NOALLOC_MAX_DOUBLES


class ChaoticusError(RuntimeError):
    pass


class _Problem(C.Structure):
    _fields_ = [("system", C.c_int), ("n_params", C.c_int), ("params", C.POINTER(C.c_double))]


class _Stepper(C.Structure):
    _fields_ = [("adaptive", C.c_int), ("t0", C.c_double), ("h", C.c_double), ("n_steps", C.c_longlong),
                ("t_end", C.c_double), ("rtol", C.c_double), ("atol", C.c_double), ("h0", C.c_double),
                ("max_steps", C.c_longlong)]


class _Report(C.Structure):
    _fields_ = [("n_accepted", C.c_void_p), ("n_rejected", C.c_void_p), ("status", C.c_void_p),
                ("t_final", C.c_void_p), ("carry", C.c_void_p), ("resume", C.c_int)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2507_00622_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, ll, dbl, i = C.c_void_p, C.c_longlong, C.c_double, C.c_int
    PP, SP, RP = C.POINTER(_Problem), C.POINTER(_Stepper), C.POINTER(_Report)
    lib.chaoticus_last_error.restype = C.c_char_p
    lib.chaoticus_dim.argtypes = [PP]
    lib.chaoticus_n_samples.restype = ll
    lib.chaoticus_n_samples.argtypes = [ll, i, i]
    lib.chaoticus_integrate_fixed.argtypes = [PP, ll, vp, dbl, dbl, ll, RP, vp]
    lib.chaoticus_integrate_adaptive.argtypes = [PP, ll, vp, SP, RP, vp]
    lib.chaoticus_sali.argtypes = [PP, ll, vp, vp, SP, i, i, vp, vp, RP, vp]
    lib.chaoticus_gali.argtypes = [PP, ll, vp, vp, i, SP, i, i, vp, vp, RP, vp]
    lib.chaoticus_ld.argtypes = [PP, ll, vp, dbl, dbl, ll, vp, vp, vp]
    lib.chaoticus_ld_adaptive.argtypes = [PP, ll, vp, SP, vp, vp, RP, vp]
    lib.chaoticus_ld_adaptive_host.argtypes = [PP, ll, vp, SP, vp, vp, RP]
    lib.chaoticus_ld_neighbours.argtypes = [PP, ll, vp, dbl, dbl, dbl, ll, vp, vp, vp, vp, vp]
    lib.chaoticus_ld_neighbours_host.argtypes = [PP, ll, vp, dbl, dbl, dbl, ll, vp, vp, vp, vp]
    lib.chaoticus_ld_neighbour_diffs_noalloc.argtypes = [PP, ll, vp, dbl, dbl, dbl, ll, vp, vp, vp]
    lib.chaoticus_lyap.argtypes = [PP, ll, vp, vp, i, SP, i, vp, vp, RP, vp]
    lib.chaoticus_ld_host.argtypes = [PP, ll, vp, dbl, dbl, ll, vp, vp]
    lib.chaoticus_sali_host.argtypes = [PP, ll, vp, vp, SP, i, i, vp, vp, RP]
    lib.chaoticus_gali_host.argtypes = [PP, ll, vp, vp, i, SP, i, i, vp, vp, RP]
    lib.chaoticus_lyap_host.argtypes = [PP, ll, vp, vp, i, SP, i, vp, vp, RP]
    lib.chaoticus_integrate_host.argtypes = [PP, ll, vp, SP, RP]
    lib.chaoticus_kernel_info.argtypes = [PP, i, i, i, ll, C.POINTER(C.c_int)]
    lib.chaoticus_set_option.argtypes = [C.c_char_p, i]
    return lib


_lib = _load()


def version():
    return _lib.chaoticus_version()


def _check(rc):
    if rc != 0:
        raise ChaoticusError(f"chaoticus rc={rc}: {_lib.chaoticus_last_error().decode()}")


def _problem(system, params):
    arr = np.ascontiguousarray(np.asarray([] if params is None else params, dtype=np.float64).ravel())
    buf = (C.c_double * max(1, arr.size))(*arr.tolist())
    pb = _Problem(int(system), int(arr.size), C.cast(buf, C.POINTER(C.c_double)))
    pb._keep = buf
    return pb


def dim(system, params=None):
    return _lib.chaoticus_dim(C.byref(_problem(system, params)))


def _dim(pb):
    n = _lib.chaoticus_dim(C.byref(pb))
    if n < 0:
        raise ChaoticusError(f"unknown system id {pb.system} or bad parameter list")
    return n


def n_samples(n_steps, renorm_every, sample_every):
    return int(_lib.chaoticus_n_samples(n_steps, renorm_every, sample_every))


def _stepper(adaptive=False, t0=0.0, h=0.0, n_steps=0, t_end=0.0, rtol=0.0, atol=0.0, h0=0.0, max_steps=0):
    return _Stepper(int(bool(adaptive)), t0, h, int(n_steps), t_end, rtol, atol, h0, int(max_steps))


def _dev(t, shape, name, dtype=torch.float64):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()
            and tuple(t.shape) == tuple(shape)):
        raise ValueError(f"{name}: need a contiguous CUDA {dtype} tensor of shape {tuple(shape)}")
    return t.data_ptr()


def _stream():
    return torch.cuda.current_stream().cuda_stream


class Report:
    """Per-trajectory report arrays (device tensors) and continuation state (chs_report).

    n: phase-space dimension; if given, a `carry` tensor [n, n_ic] is attached (the carried
    rounding words of the orbit update).  Set `resume = True` before a continuation call."""

    def __init__(self, n_ic, device, n=None):
        self.n_accepted = torch.zeros(n_ic, dtype=torch.int64, device=device)
        self.n_rejected = torch.zeros(n_ic, dtype=torch.int64, device=device)
        self.status = torch.zeros(n_ic, dtype=torch.int32, device=device)
        self.t_final = torch.zeros(n_ic, dtype=torch.float64, device=device)
        self.carry = torch.zeros((n, n_ic), dtype=torch.float64, device=device) if n else None
        self.resume = False

    def _struct(self):
        return _Report(self.n_accepted.data_ptr(), self.n_rejected.data_ptr(), self.status.data_ptr(),
                       self.t_final.data_ptr(), self.carry.data_ptr() if self.carry is not None else None,
                       int(bool(self.resume)))


class HostReport:
    """As Report, with host (numpy) arrays, for the *_host entry points."""

    def __init__(self, n_ic, n=None):
        self.n_accepted = np.zeros(n_ic, dtype=np.int64)
        self.n_rejected = np.zeros(n_ic, dtype=np.int64)
        self.status = np.zeros(n_ic, dtype=np.int32)
        self.t_final = np.zeros(n_ic)
        self.carry = np.zeros((n, n_ic)) if n else None
        self.resume = False

    def _struct(self):
        return _Report(self.n_accepted.ctypes.data, self.n_rejected.ctypes.data, self.status.ctypes.data,
                       self.t_final.ctypes.data, self.carry.ctypes.data if self.carry is not None else None,
                       int(bool(self.resume)))


def _rep(report):
    if report is None:
        return None
    report._c = report._struct()   # kept alive on the object for the duration of the call
    return C.byref(report._c)


# ---- the six entry points (same names as the C ABI, without the prefix) ----------------------
def integrate_fixed(system, params, y, t0, h, n_steps, report=None):
    pb = _problem(system, params)
    n = _dim(pb)
    _check(_lib.chaoticus_integrate_fixed(C.byref(pb), y.shape[1], _dev(y, (n, y.shape[1]), "y"), t0, h,
                                          int(n_steps), _rep(report), _stream()))


def integrate_adaptive(system, params, y, t0, t_end, rtol, atol, h0=0.0, max_steps=0, report=None):
    pb = _problem(system, params)
    n = _dim(pb)
    st = _stepper(True, t0=t0, t_end=t_end, rtol=rtol, atol=atol, h0=h0, max_steps=max_steps)
    _check(_lib.chaoticus_integrate_adaptive(C.byref(pb), y.shape[1], _dev(y, (n, y.shape[1]), "y"), C.byref(st),
                                             _rep(report), _stream()))


def _indicator(fn, system, params, y, w, k, renorm_every, sample_every, lognorm, report, stepper, with_k):
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y.shape[1]
    st = _stepper(**stepper)
    ns = 1 if st.adaptive else n_samples(st.n_steps, renorm_every, sample_every)
    out = torch.empty((ns, n_ic), dtype=torch.float64, device=y.device)
    args = [C.byref(pb), n_ic, _dev(y, (n, n_ic), "y"), _dev(w, (k, n, n_ic), "w")]
    if with_k:
        args.append(k)
    args += [C.byref(st), renorm_every, sample_every, out.data_ptr(), _dev(lognorm, (k, n_ic), "lognorm"),
             _rep(report), _stream()]
    _check(fn(*args))
    return out


def sali(system, params, y, w, *, renorm_every=1, sample_every=0, lognorm=None, report=None, **stepper):
    """Returns sali [n_samples, n_ic] (last row = value at the end)."""
    return _indicator(_lib.chaoticus_sali, system, params, y, w, 2, renorm_every, sample_every, lognorm, report,
                      stepper, False)


def gali(system, params, y, w, *, renorm_every=1, sample_every=0, lognorm=None, report=None, **stepper):
    return _indicator(_lib.chaoticus_gali, system, params, y, w, w.shape[0], renorm_every, sample_every, lognorm,
                      report, stepper, True)


def lyap(system, params, y, w, *, renorm_every=1, logsum=None, report=None, **stepper):
    """Returns lambda [k, n_ic]."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic, k = y.shape[1], w.shape[0]
    st = _stepper(**stepper)
    lam = torch.empty((k, n_ic), dtype=torch.float64, device=y.device)
    _check(_lib.chaoticus_lyap(C.byref(pb), n_ic, _dev(y, (n, n_ic), "y"), _dev(w, (k, n, n_ic), "w"), k,
                               C.byref(st), renorm_every, lam.data_ptr(), _dev(logsum, (k, n_ic), "logsum"),
                               _rep(report), _stream()))
    return lam


def ld(system, params, y0, t0, h, n_steps, *, forward=True, backward=True, out_fwd=None, out_bwd=None):
    """Returns (ld_fwd, ld_bwd), each [n_ic] or None.  y0 is not modified."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    f = (out_fwd if out_fwd is not None else torch.empty(n_ic, dtype=torch.float64, device=y0.device)) if forward else None
    b = (out_bwd if out_bwd is not None else torch.empty(n_ic, dtype=torch.float64, device=y0.device)) if backward else None
    _check(_lib.chaoticus_ld(C.byref(pb), n_ic, _dev(y0, (n, n_ic), "y0"), t0, h, int(n_steps),
                             _dev(f, (n_ic,), "ld_fwd"), _dev(b, (n_ic,), "ld_bwd"), _stream()))
    return f, b


class LdReport(Report):
    """Report of chaoticus_ld_adaptive: every array is [2, n_ic] (row 0 forward, row 1 backward)."""

    def __init__(self, n_ic, device):
        self.n_accepted = torch.zeros((2, n_ic), dtype=torch.int64, device=device)
        self.n_rejected = torch.zeros((2, n_ic), dtype=torch.int64, device=device)
        self.status = torch.zeros((2, n_ic), dtype=torch.int32, device=device)
        self.t_final = torch.zeros((2, n_ic), dtype=torch.float64, device=device)
        self.carry = None
        self.resume = False


def ld_adaptive(system, params, y0, t0, tau, *, rtol, atol, h0=0.0, max_steps=0, forward=True, backward=True,
                report=None):
    """Arc-length LD over [t0, t0 +- tau] with the adaptive solver (augmented ODE, M' = |f|).
    Returns (ld_fwd, ld_bwd), each [n_ic] or None.  y0 is not modified.  report: an LdReport."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    st = _stepper(adaptive=True, t0=t0, t_end=t0 + tau, rtol=rtol, atol=atol, h0=h0, max_steps=max_steps)
    f = torch.empty(n_ic, dtype=torch.float64, device=y0.device) if forward else None
    b = torch.empty(n_ic, dtype=torch.float64, device=y0.device) if backward else None
    _check(_lib.chaoticus_ld_adaptive(C.byref(pb), n_ic, _dev(y0, (n, n_ic), "y0"), C.byref(st),
                                      _dev(f, (n_ic,), "ld_fwd"), _dev(b, (n_ic,), "ld_bwd"), _rep(report), _stream()))
    return f, b


class HostLdReport(HostReport):
    """As LdReport, with host (numpy) arrays [2, n_ic], for ld_adaptive_host."""

    def __init__(self, n_ic):
        self.n_accepted = np.zeros((2, n_ic), dtype=np.int64)
        self.n_rejected = np.zeros((2, n_ic), dtype=np.int64)
        self.status = np.zeros((2, n_ic), dtype=np.int32)
        self.t_final = np.zeros((2, n_ic))
        self.carry = None
        self.resume = False


def ld_adaptive_host(system, params, y0, t0, tau, ld_fwd, ld_bwd, *, rtol, atol, h0=0.0, max_steps=0, report=None):
    """HOST buffers (numpy): y0 [n, n_ic]; ld_fwd / ld_bwd [n_ic] or None, filled in place.
    report: a HostLdReport (status, step counts and time reached per direction and IC: a trajectory that
    did not end with status 0 has NaN in ld_fwd / ld_bwd, and the report says why)."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    if report is not None and tuple(report.status.shape) != (2, n_ic):
        raise ValueError(f"report: need a HostLdReport({n_ic}) (arrays [2, n_ic])")
    st = _stepper(adaptive=True, t0=t0, t_end=t0 + tau, rtol=rtol, atol=atol, h0=h0, max_steps=max_steps)
    _check(_lib.chaoticus_ld_adaptive_host(C.byref(pb), n_ic, _host(y0, (n, n_ic), "y0"), C.byref(st),
                                           _host(ld_fwd, (n_ic,), "ld_fwd"), _host(ld_bwd, (n_ic,), "ld_bwd"),
                                           _rep(report)))


def ld_neighbours(system, params, y0, sigma, t0, h, n_steps, *, forward=True, backward=True, diffs=True,
                  out_fwd=None, out_bwd=None):
    """LD of every IC and of its 2n axis neighbours x0 +- sigma e_i, generated on the device.
    Returns dict(fwd [1+2n, n_ic], bwd, diff_fwd [2n, n_ic], diff_bwd); absent ones are None."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    new = lambda rows: torch.empty((rows, n_ic), dtype=torch.float64, device=y0.device)
    f = (out_fwd if out_fwd is not None else new(1 + 2 * n)) if forward else None
    b = (out_bwd if out_bwd is not None else new(1 + 2 * n)) if backward else None
    df = new(2 * n) if (forward and diffs) else None
    db = new(2 * n) if (backward and diffs) else None
    _check(_lib.chaoticus_ld_neighbours(C.byref(pb), n_ic, _dev(y0, (n, n_ic), "y0"), sigma, t0, h, int(n_steps),
                                        _dev(f, (1 + 2 * n, n_ic), "ld_fwd"), _dev(b, (1 + 2 * n, n_ic), "ld_bwd"),
                                        _dev(df, (2 * n, n_ic), "diff_fwd"), _dev(db, (2 * n, n_ic), "diff_bwd"),
                                        _stream()))
    return dict(fwd=f, bwd=b, diff_fwd=df, diff_bwd=db)


def ld_neighbour_diffs_noalloc(system, params, y0, sigma, t0, h, n_steps, diff_fwd=None, diff_bwd=None):
    """chaoticus_ld_neighbour_diffs_noalloc: the differences |M(x0 +- sigma e_i) - M(x0)| of ld_neighbours for
    callers that cannot allocate device memory (an embedding application owns all of the HBM, or the loop
    cannot afford cudaMalloc's device-wide synchronisation).  The caller passes the outputs diff_fwd / diff_bwd
    (CUDA float64 [2n, n_ic], either may be None) and gets them filled; the members' descriptors stay in a fixed
    8 MiB array inside the library, so (1 + 2n) * n_ic (rounded up to 32) per direction must fit in
    NOALLOC_MAX_DOUBLES, else ChaoticusError.  This wrapper allocates nothing either.  All calls share that
    array: calls whose GPU work overlaps (different streams) race.  Returns None."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    _check(_lib.chaoticus_ld_neighbour_diffs_noalloc(
        C.byref(pb), n_ic, _dev(y0, (n, n_ic), "y0"), sigma, t0, h, int(n_steps),
        _dev(diff_fwd, (2 * n, n_ic), "diff_fwd"), _dev(diff_bwd, (2 * n, n_ic), "diff_bwd"), _stream()))


# ---- host-buffer forms ------------------------------------------------------------------------
def _host(a, shape, name, dtype=np.float64):
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or not a.is_contiguous() or tuple(a.shape) != tuple(shape):
            raise ValueError(f"{name}: need a contiguous host tensor of shape {tuple(shape)}")
        return a.data_ptr()
    if a.dtype != dtype or not a.flags.c_contiguous or tuple(a.shape) != tuple(shape):
        raise ValueError(f"{name}: need a C-contiguous {dtype} array of shape {tuple(shape)}")
    return a.ctypes.data


def ld_host(system, params, y0, t0, h, n_steps, ld_fwd=None, ld_bwd=None):
    """y0, ld_fwd, ld_bwd: host numpy arrays or (pinned) host torch tensors."""
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    _check(_lib.chaoticus_ld_host(C.byref(pb), n_ic, _host(y0, (n, n_ic), "y0"), t0, h, int(n_steps),
                                  _host(ld_fwd, (n_ic,), "ld_fwd"), _host(ld_bwd, (n_ic,), "ld_bwd")))


def ld_neighbours_host(system, params, y0, sigma, t0, h, n_steps, ld_fwd=None, ld_bwd=None, diff_fwd=None,
                       diff_bwd=None):
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y0.shape[1]
    _check(_lib.chaoticus_ld_neighbours_host(
        C.byref(pb), n_ic, _host(y0, (n, n_ic), "y0"), sigma, t0, h, int(n_steps),
        _host(ld_fwd, (1 + 2 * n, n_ic), "ld_fwd"), _host(ld_bwd, (1 + 2 * n, n_ic), "ld_bwd"),
        _host(diff_fwd, (2 * n, n_ic), "diff_fwd"), _host(diff_bwd, (2 * n, n_ic), "diff_bwd")))


def sali_host(system, params, y, w, sali_out, *, renorm_every=1, sample_every=0, lognorm=None, report=None,
              **stepper):
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic = y.shape[1]
    st = _stepper(**stepper)
    ns = 1 if st.adaptive else n_samples(st.n_steps, renorm_every, sample_every)
    _check(_lib.chaoticus_sali_host(C.byref(pb), n_ic, _host(y, (n, n_ic), "y"), _host(w, (2, n, n_ic), "w"),
                                    C.byref(st), renorm_every, sample_every, _host(sali_out, (ns, n_ic), "sali"),
                                    _host(lognorm, (2, n_ic), "lognorm"), _rep(report)))


def gali_host(system, params, y, w, gali_out, *, renorm_every=1, sample_every=0, lognorm=None, report=None,
              **stepper):
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic, k = y.shape[1], w.shape[0]
    st = _stepper(**stepper)
    ns = 1 if st.adaptive else n_samples(st.n_steps, renorm_every, sample_every)
    _check(_lib.chaoticus_gali_host(C.byref(pb), n_ic, _host(y, (n, n_ic), "y"), _host(w, (k, n, n_ic), "w"), k,
                                    C.byref(st), renorm_every, sample_every, _host(gali_out, (ns, n_ic), "gali"),
                                    _host(lognorm, (k, n_ic), "lognorm"), _rep(report)))


def lyap_host(system, params, y, w, lambda_out, *, renorm_every=1, logsum=None, report=None, **stepper):
    pb = _problem(system, params)
    n = _dim(pb)
    n_ic, k = y.shape[1], w.shape[0]
    st = _stepper(**stepper)
    _check(_lib.chaoticus_lyap_host(C.byref(pb), n_ic, _host(y, (n, n_ic), "y"), _host(w, (k, n, n_ic), "w"), k,
                                    C.byref(st), renorm_every, _host(lambda_out, (k, n_ic), "lambda"),
                                    _host(logsum, (k, n_ic), "logsum"), _rep(report)))


def integrate_host(system, params, y, report=None, **stepper):
    pb = _problem(system, params)
    n = _dim(pb)
    st = _stepper(**stepper)
    _check(_lib.chaoticus_integrate_host(C.byref(pb), y.shape[1], _host(y, (n, y.shape[1]), "y"), C.byref(st),
                                         _rep(report)))


def set_option(name, value):
    """Process-wide library option (include/chaoticus.h chaoticus_set_option), e.g. ("adaptive_refill", 1)."""
    _check(_lib.chaoticus_set_option(name.encode(), int(value)))


# ---- reporting ---------------------------------------------------------------------------------
def kernel_info(system, params, what, k=0, adaptive=False, n_ic=1):
    """dict(tpb, blocks, lanes, regs, spill_bytes) of the kernel a call would launch."""
    pb = _problem(system, params)
    info = (C.c_int * 5)()
    _check(_lib.chaoticus_kernel_info(C.byref(pb), what, k, int(adaptive), n_ic, info))
    return dict(tpb=info[0], blocks=info[1], lanes=info[2], regs=info[3], spill_bytes=info[4])
