"""Pins of the oracle's per-trajectory STATUS paths, of its adaptive renormalisation schedule and
of the backward-time exponent convention (oracle/chaos_oracle.c run_traj) against things other
than the oracle: SciPy's solve_ivp(DOP853) as a library routine (the controller the oracle restates,
DESIGN.md R2), closed forms of linear systems (scipy.linalg.expm), and time-reversal symmetry.
CPU only.
"""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as wl

HH, C3, FPUT = 0, 1, 2
ST_OK, ST_NONFINITE, ST_UNDERFLOW, ST_MAXSTEPS = 0, 1, 2, 3


def _hh_fun(t, y):
    """Hamilton's equations of PAPER.md:91 Eq.(5), typed here for SciPy (not the oracle's code)."""
    x, yy, px, py = y
    return [px, py, -x - 2 * x * yy, -yy - x * x + yy * yy]


def test_max_steps_status_counts_attempts(orc):
    """ST_MAXSTEPS: the run stops after exactly max_steps ATTEMPTS (accepted + rejected), at the
    time solve_ivp has reached after the same number of accepted steps; outputs are NaN."""
    from scipy.integrate import solve_ivp
    y0 = wl.hh_grid(1 / 6, 4, 4)[:, 5:6].copy()
    tol, h0, K = 1e-9, 0.4, 37
    sol = solve_ivp(_hh_fun, (0.0, 200.0), y0[:, 0], method="DOP853", rtol=tol, atol=tol, first_step=h0)
    y = y0.copy()
    out = orc.integrate_adaptive(HH, None, y, 0.0, 200.0, tol, tol, h0=h0, max_steps=K, precision="f64")
    assert out["status"][0] == ST_MAXSTEPS
    na, nr = int(out["n_accepted"][0]), int(out["n_rejected"][0])
    assert na + nr == K and na > 0
    assert abs(out["t_final"][0] - sol.t[na]) < 1e-8        # same accepted times as the library routine
    assert np.isnan(y).all()                                 # status != OK => NaN outputs (R17)
    # a bound that is not reached changes nothing
    y1, y2 = y0.copy(), y0.copy()
    o1 = orc.integrate_adaptive(HH, None, y1, 0.0, 20.0, tol, tol, h0=h0, max_steps=100000, precision="f64")
    o2 = orc.integrate_adaptive(HH, None, y2, 0.0, 20.0, tol, tol, h0=h0, max_steps=0, precision="f64")
    assert o1["status"][0] == ST_OK and (y1 == y2).all() and o1["n_accepted"][0] == o2["n_accepted"][0]
    # exactly enough attempts: status OK; one fewer: MAXSTEPS
    tot = int(o2["n_accepted"][0] + o2["n_rejected"][0])
    y3 = y0.copy()
    assert orc.integrate_adaptive(HH, None, y3, 0.0, 20.0, tol, tol, h0=h0, max_steps=tot, precision="f64")["status"][0] == ST_OK
    assert (y3 == y2).all()
    y4 = y0.copy()
    assert orc.integrate_adaptive(HH, None, y4, 0.0, 20.0, tol, tol, h0=h0, max_steps=tot - 1, precision="f64")["status"][0] == ST_MAXSTEPS


def test_step_underflow_status(orc):
    """ST_UNDERFLOW: at t0 = 1e17 the spacing of doubles is 16, the smallest admissible step
    10 ulp = 160 is hopeless for Henon-Heiles, its rejection shrinks h below 10 ulp: exactly one
    rejected attempt, nothing accepted, t unchanged.  solve_ivp fails on the same input with its
    'step size is less than spacing between numbers' status."""
    from scipy.integrate import solve_ivp
    y0 = wl.hh_grid(0.125, 4, 4)[:, 5:6].copy()
    t0 = 1e17
    sol = solve_ivp(_hh_fun, (t0, t0 + 1e6), y0[:, 0], method="DOP853", rtol=1e-9, atol=1e-9, first_step=160.0)
    assert sol.status == -1 and "spacing" in sol.message and len(sol.t) == 1
    y = y0.copy()
    out = orc.integrate_adaptive(HH, None, y, t0, t0 + 1e6, 1e-9, 1e-9, h0=160.0, precision="f64")
    assert out["status"][0] == ST_UNDERFLOW
    assert out["n_accepted"][0] == 0 and out["n_rejected"][0] == 1 and out["t_final"][0] == t0
    assert np.isnan(y).all()


def test_nonfinite_status_at_the_blow_up_time(orc):
    """ST_NONFINITE: an escaping Henon-Heiles orbit (y'' ~ y^2) blows up in finite time t*.  The
    fixed-step run must flag it within a few steps after t*, t* taken from SciPy's adaptive run
    (whose step size collapses there); the other trajectories of the ensemble are untouched."""
    from scipy.integrate import solve_ivp
    y0 = wl.hh_grid(0.125, 3, 3).copy()
    y0[:, 4] = [0.0, 3.0, 0.0, 5.0]
    big = lambda t, y: abs(y[1]) - 1e12
    big.terminal = True
    sol = solve_ivp(_hh_fun, (0.0, 50.0), y0[:, 4], method="DOP853", rtol=1e-10, atol=1e-10, events=big)
    t_star = sol.t[-1]
    assert 0.1 < t_star < 5.0
    h = 0.005
    y = y0.copy()
    out = orc.integrate_fixed(HH, None, y, 0.0, h, 4000, precision="f64")
    assert out["status"][4] == ST_NONFINITE and np.isnan(y[:, 4]).all()
    assert t_star - 2 * h <= out["t_final"][4] <= t_star + 0.5
    ok = np.delete(np.arange(9), 4)
    assert (out["status"][ok] == ST_OK).all() and np.isfinite(y[:, ok]).all()
    assert (out["n_accepted"][ok] == 4000).all()
    # adaptive: flagged as non-finite or as step-size underflow, before t_end
    y = y0.copy()
    out = orc.integrate_adaptive(HH, None, y, 0.0, 50.0, 1e-10, 1e-10, max_steps=200000, precision="f64")
    assert out["status"][4] in (ST_NONFINITE, ST_UNDERFLOW) and np.isnan(y[:, 4]).all()
    assert abs(out["t_final"][4] - t_star) < 0.05
    assert (out["status"][ok] == ST_OK).all() and (out["t_final"][ok] == 50.0).all()


@pytest.mark.parametrize("m", [1, 3, 7])
def test_adaptive_renormalisation_schedule_on_an_unstable_linear_chain(orc, m):
    """Adaptive run WITH renormalisation every m accepted steps (run_traj's n_acc % m schedule) on a
    LINEAR hyperbolic system: the FPUT chain with k = -1, alpha = beta = 0 (H = p^2/2 - sum Dq^2/2),
    whose tangent map is exp(A t) with A = [[0, I], [-K, 0]], K = -tridiag(-1, 2, -1).
    Closed forms (scipy.linalg.expm): the logs of the renormalisation factors telescope to
    sum = ln |exp(A T) w0| for ANY schedule; the returned vectors are exp(A T) w0 normalised.
    Over T = 400 the growth is e^780 > DBL_MAX, so a schedule that fails to renormalise mid-run
    overflows instead."""
    from scipy.linalg import expm
    N, T = 4, 400.0
    prm = np.array([float(N), -1.0, 0.0, 0.0])
    Kmat = -(2 * np.eye(N) - np.eye(N, k=1) - np.eye(N, k=-1))
    A = np.block([[np.zeros((N, N)), np.eye(N)], [-Kmat, np.zeros((N, N))]])
    lam_max = np.sqrt(np.linalg.eigvalsh(-Kmat).max())
    assert lam_max * T > 709.0
    rng = np.random.default_rng(7)
    n_ic = 5
    y = np.zeros((2 * N, n_ic))          # the orbit sits on the fixed point: the system is linear anyway
    w = wl.deviation_vectors(n_ic, 2, 2 * N, 9, "unit")
    w0 = w.copy()
    ln = np.zeros((2, n_ic))
    out = orc.run(FPUT, prm, y, w, adaptive=True, t_end=T, rtol=1e-10, atol=1e-10, mode=orc.MODE_NORM,
                  renorm_every=m, logacc=ln, precision="f64")
    assert (out["status"] == ST_OK).all() and np.isfinite(w).all()
    # ln |exp(A T) w0| in pieces (expm(A T) itself would overflow): exp(A T) = exp(A T/8)^8 applied
    # to the vector with renormalisation, which is exact for a linear map
    P = expm(A * (T / 8))
    for ic in range(n_ic):
        for v in range(2):
            x, s = w0[v, :, ic].copy(), 0.0
            for _ in range(8):
                x = P @ x
                r = np.linalg.norm(x)
                s += np.log(r)
                x /= r
            assert abs(ln[v, ic] - s) <= 1e-6 * s
            assert np.abs(w[v, :, ic] - x).max() <= 1e-6
    assert np.abs(ln / T - lam_max).max() < 0.02          # growth rate -> the largest eigenvalue
    # the schedule is per ACCEPTED step: the controller sees vectors that have grown by e^(lam m h)
    # since the last renormalisation (absolute part of the error scale), so a longer interval can
    # only shorten the steps
    if m > 1:
        y1, w1 = np.zeros((2 * N, n_ic)), w0.copy()
        o1 = orc.run(FPUT, prm, y1, w1, adaptive=True, t_end=T, rtol=1e-10, atol=1e-10, mode=orc.MODE_NORM,
                     renorm_every=1, precision="f64")
        assert (out["n_accepted"] >= o1["n_accepted"]).all()


def test_backward_time_exponents_are_rates_per_unit_of_elapsed_time(orc):
    """DESIGN.md R18: lambda = sums / |t_final - t0|.  H is even in p, so the backward run from
    (q, p) with vectors (dq, dp) is the mirror image of the forward run from (q, -p) with
    (dq, -dp): same exponents, and the chaotic orbit's largest exponent is positive both ways."""
    cfg = wl.config("C3", 16)
    y0 = cfg["y"]
    w0 = wl.deviation_vectors(16, 2, 4, 5, "orthonormal")
    R = np.array([1.0, 1.0, -1.0, -1.0])
    yb, wb = y0.copy(), w0.copy()
    lb = orc.lyap(HH, None, yb, wb, renorm_every=5, h=-0.02, n_steps=5000, precision="f64")["lam"]
    yf, wf = y0 * R[:, None], w0 * R[None, :, None]
    lf = orc.lyap(HH, None, yf, wf, renorm_every=5, h=0.02, n_steps=5000, precision="f64")["lam"]
    assert np.abs(lb - lf).max() <= 1e-12
    assert lb[0].max() > 0.03 and (lb[0] > -1e-3).all()
    # adaptive, t_end < t0
    yb, wb = y0.copy(), w0.copy()
    la = orc.lyap(HH, None, yb, wb, renorm_every=2, adaptive=True, t_end=-100.0, rtol=1e-10, atol=1e-10,
                  precision="f64")["lam"]
    assert (la[0] > -1e-3).all() and la[0].max() > 0.03
