"""ctypes front end of the CPU oracle (oracle/chaos_oracle.c).

TEST INFRASTRUCTURE -- not part of the product path.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It imports nothing from paper_2507_00622_b200 and the CUDA path imports
nothing from here.

Two builds of the same C source: precision="f64" (double: the timed CPU baseline) and
precision="f80" (x86 long double: the parity "truth").  All arrays are numpy float64 in
the library's layout: y [n, n_ic], w [k, n, n_ic] (component-major, IC-minor).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "chaos_oracle.c")
_LIBS = {}

SYS_HENON_HEILES, SYS_COUPLED3, SYS_FPUT, SYS_DOUBLE_PENDULUM = 0, 1, 2, 3
MODE_NONE, MODE_NORM, MODE_MGS = 0, 1, 2
IND_NONE, IND_SALI, IND_GALI = 0, 1, 2

_dp = C.POINTER(C.c_double)
_lp = C.POINTER(C.c_longlong)
_ip = C.POINTER(C.c_int)


def build(force=False):
    """Compile liborc_f64.so and liborc_f80.so beside the source (gcc, -O2, OpenMP)."""
    outs = {}
    for prec, flag in (("f64", []), ("f80", ["-DORC_REAL_IS_LONG_DOUBLE"])):
        out = os.path.join(_HERE, f"liborc_{prec}.so")
        deps = [_SRC, os.path.join(_HERE, "dop853_tableau.h")]
        if force or not os.path.exists(out) or any(os.path.getmtime(d) > os.path.getmtime(out) for d in deps):
            cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", *flag, "-o", out, _SRC, "-lm"]
            subprocess.run(cmd, check=True, cwd=_HERE)
        outs[prec] = out
    return outs


def _lib(precision):
    if precision not in _LIBS:
        path = build()[precision]
        lib = C.CDLL(path)
        lib.orc_run.restype = C.c_int
        lib.orc_run.argtypes = [C.c_int, _dp, C.c_longlong, _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double,
                                C.c_longlong, C.c_double, C.c_double, C.c_double, C.c_double, C.c_longlong,
                                C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _lp, _lp, _ip, _dp, C.c_int]
        lib.orc_ld.restype = C.c_int
        lib.orc_ld.argtypes = [C.c_int, _dp, C.c_longlong, _dp, C.c_double, C.c_double, C.c_longlong, _dp, _dp,
                               C.c_int]
        lib.orc_ld_neighbours.restype = C.c_int
        lib.orc_ld_neighbours.argtypes = [C.c_int, _dp, C.c_longlong, _dp, C.c_double, C.c_double, C.c_double,
                                          C.c_longlong, _dp, _dp, _dp, _dp, C.c_int]
        lib.orc_ld_adaptive.restype = C.c_int
        lib.orc_ld_adaptive.argtypes = [C.c_int, _dp, C.c_longlong, _dp, C.c_double, C.c_double, C.c_double,
                                        C.c_double, C.c_double, C.c_longlong, _dp, _dp, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_int]
        lib.orc_rhs.argtypes = [C.c_int, _dp, C.c_int, _dp, _dp]
        lib.orc_energy.argtypes = [C.c_int, _dp, C.c_longlong, _dp, _dp]
        lib.orc_step.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_double, _dp, C.c_double, C.c_double, _dp]
        lib.orc_trace_adaptive.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_double, C.c_double, C.c_double,
                                           C.c_double, C.c_double, C.c_longlong, _dp, _lp, _lp]
        lib.orc_indicator.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp]
        lib.orc_n_samples.restype = C.c_longlong
        lib.orc_n_samples.argtypes = [C.c_longlong, C.c_int, C.c_int]
        lib.orc_dim.argtypes = [C.c_int, _dp]
        _LIBS[precision] = lib
    return _LIBS[precision]


def default_threads():
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _params(params):
    a = np.ascontiguousarray(np.asarray(params if params is not None else [0.0], dtype=np.float64).ravel())
    if a.size == 0:
        a = np.zeros(1)
    return a


def _chk(a, shape, name):
    if a.dtype != np.float64 or not a.flags.c_contiguous or tuple(a.shape) != tuple(shape):
        raise ValueError(f"{name}: need C-contiguous float64 of shape {shape}, got {a.dtype} {a.shape}")


def dim(system, params=None):
    pr = _params(params)
    return _lib("f64").orc_dim(system, _p(pr))


def n_samples(n_steps, renorm_every, sample_every):
    return int(_lib("f64").orc_n_samples(n_steps, max(1, renorm_every), sample_every))


def run(system, params, y, w=None, *, adaptive=False, t0=0.0, h=0.0, n_steps=0, t_end=0.0, rtol=0.0, atol=0.0,
        h0=0.0, max_steps=0, mode=MODE_NONE, indicator=IND_NONE, renorm_every=1, sample_every=0,
        want_series=False, logacc=None, want_lambda=False, precision="f64", threads=None):
    """General ensemble run; y (and w) advanced IN PLACE.  Returns a dict of outputs."""
    lib = _lib(precision)
    pr = _params(params)
    n = dim(system, pr)
    n_ic = y.shape[1]
    _chk(y, (n, n_ic), "y")
    k = 0 if w is None else w.shape[0]
    if w is not None:
        _chk(w, (k, n, n_ic), "w")
    ns = 1 if adaptive else n_samples(n_steps, renorm_every, sample_every)
    series = np.empty((ns, n_ic)) if want_series else None
    lam = np.empty((k, n_ic)) if want_lambda else None
    if logacc is not None:
        _chk(logacc, (k, n_ic), "logacc")
    n_acc = np.zeros(n_ic, dtype=np.int64)
    n_rej = np.zeros(n_ic, dtype=np.int64)
    status = np.zeros(n_ic, dtype=np.int32)
    t_final = np.zeros(n_ic)
    rc = lib.orc_run(system, _p(pr), n_ic, _p(y), _p(w), k, int(adaptive), t0, h, n_steps, t_end, rtol, atol,
                     h0, max_steps, mode, indicator, renorm_every, sample_every, _p(series), _p(logacc), _p(lam),
                     n_acc.ctypes.data_as(_lp), n_rej.ctypes.data_as(_lp), status.ctypes.data_as(_ip),
                     _p(t_final), threads or default_threads())
    if rc != 0:
        raise ValueError(f"orc_run: invalid arguments (rc={rc})")
    return dict(series=series, lam=lam, n_accepted=n_acc, n_rejected=n_rej, status=status, t_final=t_final)


# ---- entry points named after the library's (same meaning of the arguments) ----------------
def integrate_fixed(system, params, y, t0, h, n_steps, **kw):
    return run(system, params, y, None, t0=t0, h=h, n_steps=n_steps, **kw)


def integrate_adaptive(system, params, y, t0, t_end, rtol, atol, h0=0.0, max_steps=0, **kw):
    return run(system, params, y, None, adaptive=True, t0=t0, t_end=t_end, rtol=rtol, atol=atol, h0=h0,
               max_steps=max_steps, **kw)


def sali(system, params, y, w, *, renorm_every=1, sample_every=0, lognorm=None, **stepper):
    return run(system, params, y, w, mode=MODE_NORM, indicator=IND_SALI, renorm_every=renorm_every,
               sample_every=sample_every, want_series=True, logacc=lognorm, **stepper)


def gali(system, params, y, w, *, renorm_every=1, sample_every=0, lognorm=None, **stepper):
    return run(system, params, y, w, mode=MODE_NORM, indicator=IND_GALI, renorm_every=renorm_every,
               sample_every=sample_every, want_series=True, logacc=lognorm, **stepper)


def lyap(system, params, y, w, *, renorm_every=1, logsum=None, **stepper):
    return run(system, params, y, w, mode=MODE_MGS, renorm_every=renorm_every, want_lambda=True, logacc=logsum,
               **stepper)


def ld(system, params, y0, t0, h, n_steps, *, forward=True, backward=True, precision="f64", threads=None):
    lib = _lib(precision)
    pr = _params(params)
    n = dim(system, pr)
    n_ic = y0.shape[1]
    _chk(y0, (n, n_ic), "y0")
    f = np.empty(n_ic) if forward else None
    b = np.empty(n_ic) if backward else None
    rc = lib.orc_ld(system, _p(pr), n_ic, _p(y0), t0, h, n_steps, _p(f), _p(b), threads or default_threads())
    if rc != 0:
        raise ValueError("orc_ld: invalid arguments")
    return f, b


def ld_adaptive(system, params, y0, t0, tau, *, rtol, atol, h0=0.0, max_steps=0, forward=True, backward=True,
                precision="f64", threads=None):
    """Arc-length LD over [t0, t0 +- tau] with the adaptive solver on the augmented ODE (y, M), M' = |f|.
    Returns dict(fwd, bwd [n_ic] or None, n_accepted, n_rejected, status [2, n_ic]: row 0 forward, 1 backward)."""
    lib = _lib(precision)
    pr = _params(params)
    n = dim(system, pr)
    n_ic = y0.shape[1]
    _chk(y0, (n, n_ic), "y0")
    f = np.empty(n_ic) if forward else None
    b = np.empty(n_ic) if backward else None
    na, nr = np.zeros((2, n_ic), dtype=np.int64), np.zeros((2, n_ic), dtype=np.int64)
    st = np.zeros((2, n_ic), dtype=np.int32)
    rc = lib.orc_ld_adaptive(system, _p(pr), n_ic, _p(y0), t0, tau, rtol, atol, h0, max_steps, _p(f), _p(b),
                             na.ctypes.data, nr.ctypes.data, st.ctypes.data, threads or default_threads())
    if rc != 0:
        raise ValueError("orc_ld_adaptive: invalid arguments")
    return dict(fwd=f, bwd=b, n_accepted=na, n_rejected=nr, status=st)


def ld_neighbours(system, params, y0, sigma, t0, h, n_steps, *, forward=True, backward=True, diffs=True,
                  precision="f64", threads=None):
    """LD of every IC and of its 2n axis neighbours x0 +- sigma e_i (rows: centre, +e_0, -e_0, +e_1, ...).
    Returns dict(fwd [1+2n, n_ic], bwd, diff_fwd [2n, n_ic], diff_bwd); absent ones are None."""
    lib = _lib(precision)
    pr = _params(params)
    n = dim(system, pr)
    n_ic = y0.shape[1]
    _chk(y0, (n, n_ic), "y0")
    f = np.empty((1 + 2 * n, n_ic)) if forward else None
    b = np.empty((1 + 2 * n, n_ic)) if backward else None
    df = np.empty((2 * n, n_ic)) if (forward and diffs) else None
    db = np.empty((2 * n, n_ic)) if (backward and diffs) else None
    rc = lib.orc_ld_neighbours(system, _p(pr), n_ic, _p(y0), sigma, t0, h, n_steps, _p(f), _p(b), _p(df), _p(db),
                               threads or default_threads())
    if rc != 0:
        raise ValueError("orc_ld_neighbours: invalid arguments")
    return dict(fwd=f, bwd=b, diff_fwd=df, diff_bwd=db)


# ---- single-trajectory helpers used by the pins --------------------------------------------
def rhs(system, params, Y, k=0, precision="f64"):
    pr = _params(params)
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    F = np.empty_like(Y)
    assert _lib(precision).orc_rhs(system, _p(pr), k, _p(Y), _p(F)) == 0
    return F


def energy(system, params, y, precision="f80"):
    pr = _params(params)
    y = np.ascontiguousarray(y, dtype=np.float64)
    H = np.empty(y.shape[1])
    assert _lib(precision).orc_energy(system, _p(pr), y.shape[1], _p(y), _p(H)) == 0
    return H


def step(system, params, Y, h, k=0, rtol=1.0, atol=1.0, precision="f64"):
    """One DOP853 step of one augmented state (AoS).  Returns (Y_new, K[12, D], err_norm)."""
    pr = _params(params)
    Y = np.array(Y, dtype=np.float64, order="C")
    K = np.empty((12, Y.size))
    err = C.c_double(0.0)
    assert _lib(precision).orc_step(system, _p(pr), k, _p(Y), h, _p(K), rtol, atol, C.byref(err)) == 0
    return Y, K, err.value


def trace_adaptive(system, params, Y, t0, t_end, rtol, atol, k=0, h0=0.0, max_rec=1 << 20, precision="f64"):
    pr = _params(params)
    Y = np.array(Y, dtype=np.float64, order="C")
    t_rec = np.zeros(max_rec)
    na, nr = C.c_longlong(0), C.c_longlong(0)
    rc = _lib(precision).orc_trace_adaptive(system, _p(pr), k, _p(Y), t0, t_end, rtol, atol, h0, max_rec,
                                            _p(t_rec), C.byref(na), C.byref(nr))
    assert rc == 0
    return Y, t_rec[: min(na.value, max_rec)].copy(), na.value, nr.value


def indicator(what, W, precision="f64"):
    """what: 'sali' | 'gali' | 'renorm' | 'mgs'; W [k, n] (rows = vectors)."""
    W = np.array(W, dtype=np.float64, order="C")
    k, n = W.shape
    code = {"sali": 0, "gali": 1, "renorm": 2, "mgs": 3}[what]
    out = np.zeros(max(k, 1))
    assert _lib(precision).orc_indicator(code, n, k, _p(W), _p(out)) == 0
    if code < 2:
        return out[0]
    return W, out[:k]
