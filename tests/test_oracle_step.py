"""Pins of the oracle's integrator (oracle/chaos_oracle.c) against things other than itself:
closed forms, Hamilton's equations from the printed Hamiltonians, the order-8 slope, energy
conservation, SciPy's rk_step / solve_ivp(DOP853) as library routines (the paper's own CPU
comparator), and brute-force finite differences.  CPU only.
"""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as wl

HH, C3, FPUT = 0, 1, 2


# ----------------------------------------------------------------------------- Hamiltonians
# written from the paper's printed H (Eq.(4); Eq.(6) with the N+1
# spring reading R4; BASELINE.json configs[3]) -- NOT from the oracle's RHS.
def H_hh(y):
    x, yy, px, py = y
    return 0.5 * (px * px + py * py) + 0.5 * (x * x + yy * yy) + x * x * yy - yy ** 3 / 3


def H_c3(y, P):
    w = np.array(P[:3])
    e = P[3]
    q, p = y[:3], y[3:]
    return 0.5 * p @ p + 0.5 * (w * w) @ (q * q) + e * q[0] ** 2 * q[1] + e * q[1] ** 2 * q[2]


def H_fput(y, P):
    N = int(P[0])
    k, al, be = P[1:]
    q = np.concatenate([[0.0], y[:N], [0.0]])
    d = np.diff(q)
    return 0.5 * y[N:] @ y[N:] + (k / 2) * (d ** 2).sum() + (al / 3) * (d ** 3).sum() + (be / 4) * (d ** 4).sum()


CASES = [
    (HH, None, H_hh, np.array([0.13, -0.21, 0.3, 0.17])),
    (C3, wl.coupled3_params(0.1), None, np.array([0.2, -0.1, 0.15, 0.1, 0.25, -0.3])),
    (FPUT, np.array([5.0, 1.3, 0.7, 0.9]), None, np.array([0.3, -0.2, 0.5, 0.1, -0.4, 0.2, 0.1, -0.3, 0.25, 0.05])),
    (FPUT, wl.fput_params(8), None, None),
]


def _H(sys, P):
    if sys == HH:
        return H_hh
    if sys == C3:
        return lambda y: H_c3(y, P)
    return lambda y: H_fput(y, P)


@pytest.mark.parametrize("sys,P,_h,y0", CASES)
def test_rhs_is_hamiltons_equations(orc, sys, P, _h, y0):
    """f = (dH/dp, -dH/dq) by 4th-order central differences of the printed H."""
    if y0 is None:
        y0 = wl.fput_ics(3, 8, 2)[:, 1].copy()
    H = _H(sys, P)
    n = y0.size
    N = n // 2
    f = orc.rhs(sys, P, y0, precision="f80")
    d = 1e-3
    g = np.zeros(n)
    for c in range(n):
        e = np.zeros(n)
        e[c] = d
        g[c] = (8 * (H(y0 + e) - H(y0 - e)) - (H(y0 + 2 * e) - H(y0 - 2 * e))) / (12 * d)
    expect = np.concatenate([g[N:], -g[:N]])
    assert np.max(np.abs(f - expect)) < 1e-9


@pytest.mark.parametrize("sys,P,_h,y0", CASES)
def test_variational_rhs_is_jacobian_of_rhs(orc, sys, P, _h, y0):
    """dw/dt = Df(x) w: compare with central differences of the orbit RHS (brute force)."""
    if y0 is None:
        y0 = wl.fput_ics(3, 8, 2)[:, 2].copy()
    n = y0.size
    rng = np.random.default_rng(5)
    w = rng.standard_normal((2, n))
    F = orc.rhs(sys, P, np.concatenate([y0, w[0], w[1]]), k=2, precision="f80")
    d = 1e-4
    for v in range(2):
        # the RHS is polynomial of degree <= 3: the 4th-order stencil is exact up to rounding
        fd = (8 * (orc.rhs(sys, P, y0 + d * w[v], precision="f80") - orc.rhs(sys, P, y0 - d * w[v], precision="f80"))
              - (orc.rhs(sys, P, y0 + 2 * d * w[v], precision="f80") - orc.rhs(sys, P, y0 - 2 * d * w[v], precision="f80"))) / (12 * d)
        assert np.max(np.abs(F[n * (v + 1): n * (v + 2)] - fd)) < 1e-9


def test_energy_function_matches_printed_hamiltonians(orc):
    rng = np.random.default_rng(3)
    for sys, P, n in ((HH, None, 4), (C3, wl.coupled3_params(0.1), 6), (FPUT, np.array([6.0, 1.1, 0.3, 0.8]), 12)):
        y = rng.uniform(-0.5, 0.5, size=(n, 7))
        H = orc.energy(sys, P, y)
        ref = np.array([_H(sys, P)(y[:, i]) for i in range(7)])
        assert np.max(np.abs(H - ref)) < 1e-14


# ----------------------------------------------------------------------------- exp(At)
@pytest.mark.parametrize("prec,tol", [("f80", 2e-13), ("f64", 5e-12)])
def test_uncoupled_oscillators_closed_form(orc, prec, tol):
    """eps = 0: q_i(t) = q_i0 cos(w_i t) + p_i0/w_i sin(w_i t): the exp(At) pin (north_star)."""
    P = wl.coupled3_params(0.0)
    w = P[:3]
    rng = np.random.default_rng(11)
    y0 = rng.uniform(-0.5, 0.5, size=(6, 16))
    y = y0.copy()
    T, h = 100.0, 0.01
    orc.integrate_fixed(C3, P, y, 0.0, h, int(round(T / h)), precision=prec)
    q0, p0 = y0[:3], y0[3:]
    c, s = np.cos(w * T)[:, None], np.sin(w * T)[:, None]
    q = q0 * c + p0 / w[:, None] * s
    p = -q0 * w[:, None] * s + p0 * c
    ref = np.concatenate([q, p])
    rel = np.linalg.norm(y - ref, axis=0) / np.linalg.norm(ref, axis=0)
    assert rel.max() < tol


def test_uncoupled_tangent_map_is_the_same_rotation(orc):
    """Linear system: deviation vectors obey the same closed form as the orbit."""
    P = wl.coupled3_params(0.0)
    w = P[:3]
    y = np.random.default_rng(1).uniform(-0.5, 0.5, size=(6, 4))
    dv0 = wl.deviation_vectors(4, 3, 6, 9, "raw")
    dv = dv0.copy()
    T = 20.0
    orc.run(C3, P, y, dv, t0=0.0, h=0.01, n_steps=2000, mode=orc.MODE_NONE, precision="f80")
    c, s = np.cos(w * T)[:, None], np.sin(w * T)[:, None]
    for v in range(3):
        q0, p0 = dv0[v, :3], dv0[v, 3:]
        ref = np.concatenate([q0 * c + p0 / w[:, None] * s, -q0 * w[:, None] * s + p0 * c])
        assert np.max(np.abs(dv[v] - ref)) < 1e-12


# ----------------------------------------------------------------------------- order 8
def test_order_eight_slope(orc):
    """Global error on a Henon-Heiles orbit falls like h^8 (DESIGN.md pins; accept 7.6-8.6)."""
    y0 = wl.hh_grid(0.125, 8, 8)[:, 27:28].copy()
    T = 16.0
    ref = y0.copy()
    orc.integrate_fixed(HH, None, ref, 0.0, T / 4096, 4096, precision="f80")
    errs = []
    hs = [1.0, 0.5, 0.25, 0.125]
    for h in hs:
        y = y0.copy()
        orc.integrate_fixed(HH, None, y, 0.0, h, int(round(T / h)), precision="f80")
        errs.append(np.linalg.norm(y - ref))
    slopes = [np.log2(errs[i] / errs[i + 1]) for i in range(3)]
    assert errs[0] < 1e-3 and errs[-1] < 1e-10
    assert all(7.6 < s < 8.6 for s in slopes), (errs, slopes)


# ----------------------------------------------------------------------------- energy drift
@pytest.mark.parametrize("name,n_ic,steps,bound", [("C1", 16, 10_000, 1e-12), ("C4", 8, 20_000, 1e-12),
                                                   ("C5", 8, 10_000, 1e-11)])
def test_energy_conservation(orc, name, n_ic, steps, bound):
    cfg = wl.config(name, n_ic)
    y = cfg["y"].copy()
    H0 = orc.energy(cfg["system"], cfg["params"], y)
    assert np.max(np.abs(H0 - cfg["E"])) < 1e-13          # the generator puts ICs on the surface
    orc.integrate_fixed(cfg["system"], cfg["params"], y, 0.0, cfg["h"], steps, precision="f64")
    H1 = orc.energy(cfg["system"], cfg["params"], y)
    assert np.max(np.abs(H1 - H0)) < bound


def test_backward_integration_returns(orc):
    """h < 0 is allowed (backward LD pass): forward then backward returns to the start."""
    y0 = wl.hh_grid(0.125, 4, 4)
    y = y0.copy()
    orc.integrate_fixed(HH, None, y, 0.0, 0.01, 1000, precision="f80")
    orc.integrate_fixed(HH, None, y, 10.0, -0.01, 1000, precision="f80")
    assert np.max(np.abs(y - y0)) < 1e-13


# ----------------------------------------------------------------------------- SciPy as a library
def _scipy_fun(orc, sys, P, k):
    return lambda t, Y: orc.rhs(sys, P, Y, k=k, precision="f64")


def test_single_step_matches_scipy_rk_step(orc):
    """Library routine: scipy's rk_step with scipy's own DOP853 tableau, step by step."""
    from scipy.integrate._ivp import dop853_coefficients as dc
    from scipy.integrate._ivp.rk import rk_step
    y0 = wl.hh_grid(0.125, 4, 4)[:, 5]
    w = wl.deviation_vectors(1, 2, 4, 0, "unit")[:, :, 0]
    Y = np.concatenate([y0, w[0], w[1]])
    fun = _scipy_fun(orc, HH, None, 2)
    A, B, Cc = dc.A[:12, :12], dc.B, dc.C[:12]
    for h in (0.01, -0.05, 0.3):
        Yo, Yl = Y.copy(), Y.copy()
        for _ in range(20):
            Yo, Ko, _err = orc.step(HH, None, Yo, h, k=2)
            K = np.empty((13, Y.size))
            Yl, _f = rk_step(fun, 0.0, Yl, fun(0.0, Yl), h, A, B, Cc, K)
            # late stages sum terms with |a_ij| up to 43.5: rounding is amplified ~50x over eps
            assert np.max(np.abs(Ko - K[:12])) <= 1e-13 * max(1.0, np.abs(K).max())
            assert np.max(np.abs(Yo - Yl)) <= 2e-15 * max(1.0, np.abs(Yl).max())
            Yl = Yo.copy()      # resynchronise so the check is per step


def test_error_norm_matches_scipy_formula_inputs(orc):
    """The (5,3) error norm equals SciPy's DOP853._estimate_error_norm on the same K."""
    from scipy.integrate import DOP853
    y0 = wl.hh_grid(1 / 6, 4, 4)[:, 9]
    w = wl.deviation_vectors(1, 2, 4, 3, "unit")[:, :, 0]
    Y = np.concatenate([y0, w[0], w[1]])
    fun = _scipy_fun(orc, HH, None, 2)
    rtol = atol = 1e-9
    for h in (0.05, 0.4, 1.0):
        Yn, K, err = orc.step(HH, None, Y, h, k=2, rtol=rtol, atol=atol)
        s = DOP853(fun, 0.0, Y, 10.0, rtol=rtol, atol=atol)
        Kf = np.zeros_like(s.K)
        Kf[:12] = K
        scale = atol + np.maximum(np.abs(Y), np.abs(Yn)) * rtol
        ref = s._estimate_error_norm(Kf, h, scale)
        # E5.K cancels O(1) terms down to the local error: absolute floor ~ eps |h| / atol
        assert abs(err - ref) <= 1e-9 * ref + 2.2e-16 * abs(h) / atol
        assert ref > 1e-8


@pytest.mark.parametrize("tol,k,h0,t_tol", [
    (1e-6, 2, 0.5, 1e-9), (1e-6, 2, 2.0, 1e-9), (1e-8, 2, 0.3, 1e-8), (1e-10, 0, 0.2, 1e-8),   # first step given
    (1e-6, 2, 0.0, 1e-6), (1e-12, 2, 0.0, 5e-5), (1e-12, 0, 0.0, 5e-5),                         # automatic h0
])
def test_adaptive_steps_match_solve_ivp(orc, tol, k, h0, t_tol):
    """Same accepted steps as solve_ivp(method='DOP853') on the augmented system (no
    renormalisation): pins the controller constants, the (5,3) error norm, the starting-step
    heuristic and the t_end clipping (reading R2).  With the automatic (tiny) first step the
    first error estimate is pure rounding noise (E5.K cancels to ~1e-18), so the second step
    size -- and from then on every t_n -- carries an offset of ~1e-5 h that depends on the
    summation order; with the first step given, times agree to ~1e-9."""
    from scipy.integrate import solve_ivp
    y0 = wl.hh_grid(1 / 6, 4, 4)[:, 9]
    Y = y0.copy()
    if k:
        w = wl.deviation_vectors(1, k, 4, 0, "unit")[:, :, 0]
        Y = np.concatenate([y0, w.ravel()])
    T = 30.0
    kw = dict(first_step=h0) if h0 > 0 else {}
    sol = solve_ivp(_scipy_fun(orc, HH, None, k), (0.0, T), Y, method="DOP853", rtol=tol, atol=tol, **kw)
    Yo, t_rec, na, nr = orc.trace_adaptive(HH, None, Y, 0.0, T, tol, tol, k=k, h0=h0, precision="f64")
    assert na == len(sol.t) - 1
    # solve_ivp evaluates f once at t0 (+1 for the starting-step probe) and 12 times per attempt
    assert sol.nfev == (1 if h0 > 0 else 2) + 12 * (na + nr)
    if h0 == 0:      # the first step is exactly the starting-step heuristic's h0
        assert abs(t_rec[0] - sol.t[1]) < 1e-15
    assert np.max(np.abs(t_rec - sol.t[1:])) < t_tol
    assert t_rec[-1] == T
    assert np.max(np.abs(Yo - sol.y[:, -1])) < max(1e-9, 100 * tol) * np.abs(sol.y[:, -1]).max()


def test_adaptive_backward_and_energy(orc):
    cfg = wl.config("C3", 16)
    y = cfg["y"].copy()
    H0 = orc.energy(HH, None, y)
    out = orc.integrate_adaptive(HH, None, y, 0.0, 100.0, 1e-12, 1e-12)
    assert np.all(out["status"] == 0) and np.all(out["t_final"] == 100.0)
    assert np.max(np.abs(orc.energy(HH, None, y) - H0)) < 1e-11
    steps_per_unit = out["n_accepted"].mean() / 100.0
    assert 5.0 < steps_per_unit < 15.0
    assert out["n_rejected"].sum() < 0.15 * out["n_accepted"].sum()
    # backward in time (t_end < t0) over a short, non-chaotic span returns to the start
    y = cfg["y"].copy()
    orc.integrate_adaptive(HH, None, y, 0.0, 10.0, 1e-12, 1e-12)
    out = orc.integrate_adaptive(HH, None, y, 10.0, 0.0, 1e-12, 1e-12)
    assert np.all(out["t_final"] == 0.0) and np.all(out["status"] == 0)
    assert np.max(np.abs(y - cfg["y"])) < 1e-9


# ----------------------------------------------------------------------------- deviation vectors, brute force
@pytest.mark.parametrize("name", ["C1", "C4", "C5"])
def test_deviation_vectors_match_finite_differences(orc, name):
    """w(t) = [x(t; x0 + d w0) - x(t; x0 - d w0)] / (2d) on tiny inputs, t = 5."""
    cfg = wl.config(name, 4)
    sys, P = cfg["system"], cfg["params"]
    y0, w0 = cfg["y"], cfg["w"][:2].copy()
    steps = int(round(5.0 / cfg["h"]))
    y, w = y0.copy(), w0.copy()
    orc.run(sys, P, y, w, t0=0.0, h=cfg["h"], n_steps=steps, mode=orc.MODE_NONE, precision="f80")
    d = 1e-6
    for v in range(2):
        yp, ym = y0 + d * w0[v], y0 - d * w0[v]
        orc.integrate_fixed(sys, P, yp, 0.0, cfg["h"], steps, precision="f80")
        orc.integrate_fixed(sys, P, ym, 0.0, cfg["h"], steps, precision="f80")
        fd = (yp - ym) / (2 * d)
        rel = np.linalg.norm(fd - w[v], axis=0) / np.linalg.norm(w[v], axis=0)
        assert rel.max() < 1e-7, (name, v, rel)
