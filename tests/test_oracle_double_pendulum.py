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
