"""Seeded synthetic input generators (initial conditions and initial deviation vectors).

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds
none of the method's arithmetic (no Runge-Kutta step, no variational equations, no
indicator): only the recipes that place initial conditions on energy surfaces, as stated
in DESIGN.md "Input recipe" (readings R8-R11; BASELINE.json configs[0..4]).  It imports
neither the CUDA binding nor oracle/.

The paper's own IC sets are not published ("randomly generated
initial conditions"); these synthetic ensembles have the shapes, sizes and structure of the
five BASELINE.json configurations and stand in for them.

Layout of everything returned: float64, C-contiguous, component-major / IC-minor:
    y [n, n_ic],   w [k, n, n_ic].
"""
import numpy as np

SYS_HENON_HEILES, SYS_COUPLED3, SYS_FPUT, SYS_DOUBLE_PENDULUM = 0, 1, 2, 3

OMEGA_C3 = (1.0, 2.0 ** 0.5, 3.0 ** 0.5)


# --------------------------------------------------------------------------- Henon-Heiles
def hh_y_range(E):
    """The two roots of y^2/2 - y^3/3 = E nearest 0 (x = 0, p = 0 turning points)."""
    r = np.roots([-1.0 / 3.0, 0.5, 0.0, -E])
    r = np.sort(r[np.abs(r.imag) < 1e-12].real)
    lo = r[r < 0].max()
    hi = r[r > 0].min()
    # polish with Newton (np.roots is ~1e-15 already; keeps the recipe deterministic)
    for _ in range(3):
        lo -= (lo * lo / 2 - lo ** 3 / 3 - E) / (lo - lo * lo)
        hi -= (hi * hi / 2 - hi ** 3 / 3 - E) / (hi - hi * hi)
    return float(lo), float(hi)


def hh_grid(E, n_y, n_py, i_range=None):
    """Energy-fitted grid on the x = 0 section (reading R9): every point strictly inside
    the allowed region, px > 0 from the energy.  IC index = i * n_py + j.

    i_range = (i0, i1) restricts to rows i0 <= i < i1 of the same grid (used to shard the
    grid over ranks and to subsample without building the whole grid).
    """
    lo, hi = hh_y_range(E)
    i0, i1 = (0, n_y) if i_range is None else i_range
    i = np.arange(i0, i1, dtype=np.float64)
    j = np.arange(n_py, dtype=np.float64)
    yv = lo + (i + 0.5) * (hi - lo) / n_y
    P = np.sqrt(np.maximum(2 * E - yv * yv + (2.0 / 3.0) * yv ** 3, 0.0))
    s = 2 * (j + 0.5) / n_py - 1
    Y, S = np.meshgrid(yv, s, indexing="ij")
    Pm = np.repeat(P[:, None], n_py, axis=1)
    out = np.empty((4, Y.size))
    out[0] = 0.0
    out[1] = Y.ravel()
    out[2] = (Pm * np.sqrt(1 - S * S)).ravel()
    out[3] = (S * Pm).ravel()
    return np.ascontiguousarray(out)


# --------------------------------------------------------------------------- deviation vectors
def deviation_vectors(n_ic, k, n, seed, kind="unit"):
    """N(0,1) draws from default_rng(seed) in order [ic][vector][component] (reading R8).
    kind = "raw": as drawn; "unit": each vector scaled to norm 1; "orthonormal": the k
    vectors of each IC replaced by the Q factor of the n x k draw (sign fixed so R_ii > 0).
    """
    g = np.random.default_rng(seed).standard_normal((n_ic, k, n))
    if kind == "unit":
        g /= np.linalg.norm(g, axis=2, keepdims=True)
    elif kind == "orthonormal":
        q, r = np.linalg.qr(np.swapaxes(g, 1, 2))          # [ic, n, k]
        d = np.sign(np.diagonal(r, axis1=1, axis2=2))
        g = np.swapaxes(q * d[:, None, :], 1, 2)
    elif kind != "raw":
        raise ValueError(kind)
    return np.ascontiguousarray(np.transpose(g, (1, 2, 0)))


# --------------------------------------------------------------------------- 3-DoF coupled
def coupled3_params(eps=0.1):
    return np.array([OMEGA_C3[0], OMEGA_C3[1], OMEGA_C3[2], eps])


def coupled3_ics(n_ic, seed=1, E=0.1, eps=0.1):
    """z ~ U(-1/2,1/2)^6 in order (q1,q2,q3,p1,p2,p3), scaled by the smallest s > 0 with
    s^2 H2(z) + s^3 H3(z) = E (reading R10)."""
    z = np.random.default_rng(seed).uniform(-0.5, 0.5, size=(n_ic, 6))
    w2 = np.array(OMEGA_C3) ** 2
    H2 = 0.5 * (z[:, 3:] ** 2).sum(1) + 0.5 * (w2 * z[:, :3] ** 2).sum(1)
    H3 = eps * (z[:, 0] ** 2 * z[:, 1] + z[:, 1] ** 2 * z[:, 2])
    s = np.sqrt(E / H2)
    for _ in range(60):
        f = s * s * H2 + s ** 3 * H3 - E
        s = s - f / (2 * s * H2 + 3 * s * s * H3)
    assert np.all(s > 0) and np.all(np.abs(s * s * H2 + s ** 3 * H3 - E) < 1e-14)
    return np.ascontiguousarray((z * s[:, None]).T)


# --------------------------------------------------------------------------- FPUT-beta
def fput_params(N=8, k=1.0, alpha=0.0, beta=1.0):
    return np.array([float(N), k, alpha, beta])


def fput_ics(n_ic, N=8, seed=2, E=1.0, k=1.0, beta=1.0, noise_var=1e-3):
    """Mode-1 excitation q_i = sin(pi i/(N+1)), p = 0, plus N(0, noise_var) on all 2N
    components ([ic][q1..qN,p1..pN]), scaled so that H = E exactly (alpha = 0; reading R11).
    The chain has N+1 springs with fixed walls (reading R4)."""
    i = np.arange(1, N + 1)
    z = np.zeros((n_ic, 2 * N))
    z[:, :N] = np.sin(np.pi * i / (N + 1))
    z += np.random.default_rng(seed).normal(0.0, np.sqrt(noise_var), size=(n_ic, 2 * N))
    qpad = np.concatenate([np.zeros((n_ic, 1)), z[:, :N], np.zeros((n_ic, 1))], axis=1)
    d = np.diff(qpad, axis=1)                                # N+1 spring extensions
    H2 = 0.5 * (z[:, N:] ** 2).sum(1) + 0.5 * k * (d ** 2).sum(1)
    H4 = 0.25 * beta * (d ** 4).sum(1)
    s2 = (-H2 + np.sqrt(H2 * H2 + 4 * H4 * E)) / (2 * H4)
    return np.ascontiguousarray((z * np.sqrt(s2)[:, None]).T)


# --------------------------------------------------------------------------- double pendulum
def double_pendulum_ics(n_ic, seed=3, theta_max=2.0, p_max=1.0):
    """Random ICs of the dimensionless double pendulum (the paper does not state its
    IC set): angles uniform in [-theta_max, theta_max], momenta uniform in
    [-p_max, p_max], order [ic][theta1, theta2, p1, p2] from default_rng(seed)."""
    r = np.random.default_rng(seed).uniform(-1.0, 1.0, size=(n_ic, 4))
    r[:, :2] *= theta_max
    r[:, 2:] *= p_max
    return np.ascontiguousarray(r.T)


# --------------------------------------------------------------------------- the five configs
def config(name, n_ic=None):
    """Inputs of BASELINE.json configs[0..4] ("C1".."C5").  n_ic (optional) shrinks the
    ensemble for tests: grids become the nearest square, random ensembles are truncated
    (the first n_ic draws of the same stream)."""
    if name in ("C1", "C2", "C3"):
        E = {"C1": 0.125, "C2": 0.125, "C3": 1.0 / 6.0}[name]
        side = {"C1": 32, "C2": 1024, "C3": 512}[name]
        if n_ic is not None:
            side = int(round(n_ic ** 0.5))
        y = hh_grid(E, side, side)
        cfg = dict(system=SYS_HENON_HEILES, params=np.zeros(1), y=y, E=E, side=side)
        if name == "C1":
            cfg.update(w=deviation_vectors(y.shape[1], 2, 4, 0, "unit"), h=0.01, n_steps=10_000, renorm_every=1)
        elif name == "C2":
            cfg.update(h=0.01, n_steps=5_000)
        else:
            cfg.update(w=deviation_vectors(y.shape[1], 2, 4, 0, "unit"), t_end=1000.0, rtol=1e-12, atol=1e-12,
                       renorm_every=1)
        return cfg
    if name == "C4":
        n = 65_536 if n_ic is None else n_ic
        return dict(system=SYS_COUPLED3, params=coupled3_params(0.1), y=coupled3_ics(n, 1, 0.1, 0.1),
                    w=deviation_vectors(n, 6, 6, 101, "orthonormal"), h=0.01, n_steps=100_000, renorm_every=10,
                    E=0.1)
    if name == "C5":
        n = 65_536 if n_ic is None else n_ic
        return dict(system=SYS_FPUT, params=fput_params(8, 1.0, 0.0, 1.0), y=fput_ics(n, 8, 2, 1.0),
                    w=deviation_vectors(n, 4, 16, 102, "orthonormal"), h=0.05, n_steps=20_000, renorm_every=10,
                    E=1.0)
    raise ValueError(name)
