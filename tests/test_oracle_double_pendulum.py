"""Pins of the oracle's double pendulum (Eq.(1)-(3)); none compares the oracle with
itself: Hamilton's equations against finite differences of the Hamiltonian of Eq.(1) (the RHS is
written from Eq.(3) with C = -B^-1 dB/dx B^-1 as matrix products, the energy from Eq.(1)-(2)), the
small-angle normal-mode frequencies (textbook closed form), energy conservation, and SciPy's
DOP853 as a library integrator of an independently derived (Lagrangian) form."""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as W

DP = W.SYS_DOUBLE_PENDULUM


@pytest.mark.parametrize("prm", [(1.0, 1.0), (0.5, 2.0), (3.0, 0.7)])
def test_rhs_is_hamiltons_equations_of_eq1(orc, prm):
    rng = np.random.default_rng(0)
    for _ in range(20):
        y = rng.uniform(-2, 2, 4)
        f = orc.rhs(DP, prm, y)
        g = np.zeros(4)
        for c in range(4):
            d = 1e-6
            yp, ym = y.copy(), y.copy()
            yp[c] += d
            ym[c] -= d
            g[c] = (orc.energy(DP, prm, yp[:, None])[0] - orc.energy(DP, prm, ym[:, None])[0]) / (2 * d)
        expect = np.array([g[2], g[3], -g[0], -g[1]])     # theta' = dH/dp, p' = -dH/dtheta
        assert np.abs(f - expect).max() <= 2e-9 * max(1.0, np.abs(expect).max())


def test_small_angle_normal_modes(orc):
    """Linearised about the stable equilibrium the system has two normal modes; their squared
    frequencies are the eigenvalues of B0^-1 K with B0 = B(x=1), K = diag(alpha(1+sigma), 1)
    (quadratic forms of Eq.(1)).  A tiny-amplitude orbit started on a mode stays on it and
    oscillates with that frequency."""
    sg, al = 0.8, 1.3
    B0 = np.array([[al * al * (1 + sg), al], [al, 1.0]])
    K = np.diag([al * (1 + sg), 1.0])
    w2, V = np.linalg.eig(np.linalg.inv(B0) @ K)
    for m in range(2):
        om = np.sqrt(w2[m].real)
        v = V[:, m].real * 1e-6
        y = np.zeros((4, 1))
        y[:2, 0] = v
        T = 2 * np.pi / om
        n = 2000
        orc.integrate_fixed(DP, (sg, al), y, 0.0, T / n, n, precision="f80")
        assert np.abs(y[:2, 0] - v).max() <= 1e-10 * 1e-6 * 1e3   # back to the start after one period (to O(amp^3))
        assert np.abs(y[2:, 0]).max() <= 1e-15


def test_energy_conservation(orc):
    prm = (1.0, 1.0)
    y = W.double_pendulum_ics(64, seed=3)
    H0 = orc.energy(DP, prm, y)
    orc.integrate_fixed(DP, prm, y, 0.0, 0.01, 20000)
    assert np.abs(orc.energy(DP, prm, y) - H0).max() <= 1e-11   # paper's own level: 1e-9
    y = W.double_pendulum_ics(32, seed=4)
    H0 = orc.energy(DP, prm, y)
    r = orc.integrate_adaptive(DP, prm, y, 0.0, 100.0, 1e-11, 1e-11)
    assert (r["status"] == 0).all() and np.abs(orc.energy(DP, prm, y) - H0).max() <= 1e-9


def test_against_lagrangian_form_with_scipy(orc):
    """Independent derivation: the Lagrangian equations of motion of the double pendulum in
    physical units (m1, m2, l1, l2, g), integrated with SciPy's DOP853, mapped to the paper's
    dimensionless variables: time unit sqrt(l2/g), sigma = m1/m2, alpha = l1/l2,
    p = dL/d(theta') / (m2 l2^2 * sqrt(g/l2))."""
    from scipy.integrate import solve_ivp
    m1, m2, l1, l2, g = 1.7, 0.9, 1.2, 0.8, 9.81
    sg, al = m1 / m2, l1 / l2
    th = np.array([0.9, -0.4])
    om = np.array([0.3, -0.5])            # physical angular velocities

    def lag(t, s):
        a, b, wa, wb = s
        d = a - b
        M = np.array([[(m1 + m2) * l1 * l1, m2 * l1 * l2 * np.cos(d)], [m2 * l1 * l2 * np.cos(d), m2 * l2 * l2]])
        rhs = np.array([-m2 * l1 * l2 * wb * wb * np.sin(d) - (m1 + m2) * g * l1 * np.sin(a),
                        m2 * l1 * l2 * wa * wa * np.sin(d) - m2 * g * l2 * np.sin(b)])
        acc = np.linalg.solve(M, rhs)
        return [wa, wb, acc[0], acc[1]]

    tau = np.sqrt(l2 / g)
    t_phys = 7.0 * tau
    sol = solve_ivp(lag, [0, t_phys], [th[0], th[1], om[0], om[1]], method="DOP853", rtol=1e-12, atol=1e-13)

    def momenta(a, b, wa, wb):
        d = a - b
        p1 = (m1 + m2) * l1 * l1 * wa + m2 * l1 * l2 * wb * np.cos(d)
        p2 = m2 * l2 * l2 * wb + m2 * l1 * l2 * wa * np.cos(d)
        return np.array([p1, p2]) / (m2 * l2 * l2 / tau)

    y = np.zeros((4, 1))
    y[:2, 0] = th
    y[2:, 0] = momenta(th[0], th[1], om[0], om[1])
    orc.integrate_fixed(DP, (sg, al), y, 0.0, 7.0 / 4000, 4000, precision="f80")
    a, b, wa, wb = sol.y[:, -1]
    assert np.abs(y[:2, 0] - [a, b]).max() <= 1e-9
    assert np.abs(y[2:, 0] - momenta(a, b, wa, wb)).max() <= 1e-9


# ----------------------------------------------------------------------------- variational equations
@pytest.mark.parametrize("prm", [(1.0, 1.0), (0.5, 2.0), (3.0, 0.7)])
def test_variational_rhs_is_jacobian_of_eq3(orc, prm):
    """dw/dt = Df(x) w with f the right-hand side of Eq.(3): against 4th-order central differences of the
    ORBIT right-hand side (pinned above against Eq.(1)), in long double."""
    rng = np.random.default_rng(1)
    for _ in range(10):
        y = rng.uniform(-2, 2, 4)
        w = rng.standard_normal((2, 4))
        F = orc.rhs(DP, prm, np.concatenate([y, w[0], w[1]]), k=2, precision="f80")
        d = 2e-3
        for v in range(2):
            r = lambda a: orc.rhs(DP, prm, y + a * w[v], precision="f80")
            fd = (8 * (r(d) - r(-d)) - (r(2 * d) - r(-2 * d))) / (12 * d)
            assert np.abs(F[4 * (v + 1): 4 * (v + 2)] - fd).max() <= 1e-8 * max(1.0, np.abs(fd).max())


def test_deviation_vectors_match_neighbouring_orbits(orc):
    """w(t) = [x(t; x0 + d w0) - x(t; x0 - d w0)] / (2d), brute force, t = 5."""
    prm = (1.0, 1.0)
    y0 = W.double_pendulum_ics(6, seed=3)
    w0 = W.deviation_vectors(6, 2, 4, 17, "unit")
    y, w = y0.copy(), w0.copy()
    orc.run(DP, prm, y, w, t0=0.0, h=0.01, n_steps=500, mode=orc.MODE_NONE, precision="f80")
    d = 1e-6
    for v in range(2):
        yp, ym = y0 + d * w0[v], y0 - d * w0[v]
        orc.integrate_fixed(DP, prm, yp, 0.0, 0.01, 500, precision="f80")
        orc.integrate_fixed(DP, prm, ym, 0.0, 0.01, 500, precision="f80")
        fd = (yp - ym) / (2 * d)
        rel = np.linalg.norm(fd - w[v], axis=0) / np.linalg.norm(w[v], axis=0)
        assert rel.max() < 1e-6, (v, rel)


def test_small_angle_tangent_map_and_indicators(orc):
    """Near the stable equilibrium the flow is linear: the tangent map is exp(A t), A = [[0, B0^-1], [-K, 0]]
    (the quadratic forms of Eq.(1) at x = 1), so deviation vectors follow scipy.linalg.expm, SALI stays
    O(1) and the largest exponent tends to 0.  A strongly excited orbit is chaotic: SALI collapses and the
    largest exponent is positive; exponents of the full spectrum pair up and sum to zero (Hamiltonian)."""
    from scipy.linalg import expm
    sg, al = 1.0, 1.0
    B0 = np.array([[al * al * (1 + sg), al], [al, 1.0]])
    K = np.diag([al * (1 + sg), 1.0])
    A = np.block([[np.zeros((2, 2)), np.linalg.inv(B0)], [-K, np.zeros((2, 2))]])
    y = np.zeros((4, 1))
    y[:2, 0] = [1e-7, -2e-7]
    w0 = W.deviation_vectors(1, 2, 4, 3, "unit")
    w = w0.copy()
    T = 7.0
    orc.run(DP, (sg, al), y, w, t0=0.0, h=0.01, n_steps=700, mode=orc.MODE_NONE, precision="f80")
    E = expm(A * T)
    for v in range(2):
        assert np.abs(w[v, :, 0] - E @ w0[v, :, 0]).max() <= 1e-9
    # regular vs chaotic
    yr = np.zeros((4, 1))
    yr[:2, 0] = [0.3, 0.2]
    yc = np.zeros((4, 1))
    yc[:2, 0] = [2.6, 2.9]                      # both arms near the top: strongly chaotic
    out = {}
    for name, yy in (("reg", yr), ("cha", yc)):
        y1, w1 = yy.copy(), W.deviation_vectors(1, 2, 4, 5, "unit")
        s = orc.sali(DP, (sg, al), y1, w1, renorm_every=1, h=0.005, n_steps=60000, precision="f64")["series"][0, 0]
        y2, w2 = yy.copy(), W.deviation_vectors(1, 4, 4, 5, "orthonormal")
        lam = orc.lyap(DP, (sg, al), y2, w2, renorm_every=5, h=0.005, n_steps=60000, precision="f64")["lam"][:, 0]
        out[name] = (s, lam)
    assert out["reg"][0] > 1e-3 and out["cha"][0] < 1e-8
    assert out["reg"][1][0] < 0.05 and out["cha"][1][0] > 0.3
    for name in out:
        lam = out[name][1]
        assert abs(lam.sum()) < 1e-9 and np.abs(lam + lam[::-1]).max() < 0.03
