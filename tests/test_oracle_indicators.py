"""Pins of the oracle's indicator code: SALI, GALI_k (SVD), renormalisation / mLE, the
Lyapunov spectrum (modified Gram-Schmidt) and the arc-length Lagrangian descriptor, against
LAPACK routines, exact identities, closed forms, symmetries and the known qualitative
behaviour (north_star list).  CPU only.
"""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as wl

HH, C3, FPUT = 0, 1, 2


# ----------------------------------------------------------------------------- pure indicator arithmetic
def test_sali_definition_and_gali2_identity(orc):
    """SALI = min(|w1+w2|, |w1-w2|) and GALI_2 = 1/2 |w1+w2| |w1-w2| exactly
    (= |w1 ^ w2| = sin of the angle) -- ties the SALI code to the SVD code."""
    rng = np.random.default_rng(0)
    for n in (4, 6, 16):
        for _ in range(20):
            W = rng.standard_normal((2, n))
            W /= np.linalg.norm(W, axis=1, keepdims=True)
            s = orc.indicator("sali", W, "f80")
            g = orc.indicator("gali", W, "f80")
            sp, sm = np.linalg.norm(W[0] + W[1]), np.linalg.norm(W[0] - W[1])
            assert abs(s - min(sp, sm)) < 1e-15
            assert abs(g - 0.5 * sp * sm) < 1e-14
            ang = np.arccos(np.clip(W[0] @ W[1], -1, 1))
            assert abs(g - np.sin(ang)) < 1e-12
    # nearly aligned / anti-aligned vectors
    a = np.array([1.0, 0, 0, 0])
    for d in (1e-3, 1e-7, 1e-12):
        b = np.array([1.0, d, 0, 0])
        b /= np.linalg.norm(b)
        for sgn in (1, -1):
            assert abs(orc.indicator("sali", np.stack([a, sgn * b]), "f80") - d) < 2e-3 * d + 1e-17


@pytest.mark.parametrize("n,k", [(4, 2), (6, 3), (16, 4), (16, 7), (6, 6)])
def test_gali_equals_product_of_lapack_singular_values(orc, n, k):
    rng = np.random.default_rng(n * 10 + k)
    for trial in range(10):
        W = rng.standard_normal((k, n))
        if trial % 2:            # nearly dependent columns: small GALI
            W[-1] = W[0] + 1e-6 * rng.standard_normal(n)
        W /= np.linalg.norm(W, axis=1, keepdims=True)
        g = orc.indicator("gali", W, "f80")
        sv = np.linalg.svd(W.T, compute_uv=False)
        assert abs(g - np.prod(sv)) <= 1e-12 * np.prod(sv) + 5e-16      # LAPACK (f64): sigma_min +- eps sigma_max
        # cross-checks: product of |r_ii| of a QR; sqrt(det(W W^T)) while well conditioned
        r = np.linalg.qr(W.T, mode="r")
        assert abs(g - np.prod(np.abs(np.diag(r)))) <= 1e-10 * g + 5e-16
        if g > 1e-3:        # the Gram determinant squares the condition number
            assert abs(g - np.sqrt(np.linalg.det(W @ W.T))) <= 1e-8 * g
    Q = np.linalg.qr(rng.standard_normal((n, k)))[0].T
    assert abs(orc.indicator("gali", Q, "f80") - 1.0) < 1e-14      # orthonormal => GALI_k = 1


def test_mgs_is_a_qr_factorisation(orc):
    """Modified Gram-Schmidt = QR with r_vv > 0: same Q (up to sign fixed by r_vv > 0) and
    ln r_vv as LAPACK's QR ("via QR factorization")."""
    rng = np.random.default_rng(4)
    for n, k in ((6, 6), (16, 4), (4, 2)):
        W = rng.standard_normal((k, n))
        Q, logs = orc.indicator("mgs", W, "f80")
        q, r = np.linalg.qr(W.T)
        sgn = np.sign(np.diag(r))
        assert np.max(np.abs(Q.T - q * sgn)) < 1e-13
        assert np.max(np.abs(logs - np.log(np.abs(np.diag(r))))) < 1e-13
        assert np.max(np.abs(Q @ Q.T - np.eye(k))) < 1e-14


def test_renormalise(orc):
    rng = np.random.default_rng(8)
    W = rng.standard_normal((3, 6)) * np.array([[1e-5], [1.0], [1e7]])
    U, logs = orc.indicator("renorm", W, "f80")
    nrm = np.linalg.norm(W, axis=1)
    assert np.max(np.abs(logs - np.log(nrm))) < 1e-13
    assert np.max(np.abs(U - W / nrm[:, None])) < 1e-15
    # not orthogonalised: angles unchanged
    assert abs(U[0] @ U[1] - (W[0] @ W[1]) / (nrm[0] * nrm[1])) < 1e-15


# ----------------------------------------------------------------------------- SALI behaviour
def test_sali_constant_for_isotropic_oscillator(orc):
    """All w_i = 1, eps = 0: the tangent map is a rotation of phase space by angle t, angles
    between deviation vectors are preserved => SALI(t) == SALI(0)."""
    P = np.array([1.0, 1.0, 1.0, 0.0])
    n_ic = 8
    y = np.random.default_rng(2).uniform(-0.5, 0.5, size=(6, n_ic))
    w = wl.deviation_vectors(n_ic, 2, 6, 7, "unit")
    s0 = np.minimum(np.linalg.norm(w[0] + w[1], axis=0), np.linalg.norm(w[0] - w[1], axis=0))
    out = orc.sali(C3, P, y, w, t0=0.0, h=0.01, n_steps=5000, renorm_every=1, sample_every=1000, precision="f80")
    assert out["series"].shape == (6, n_ic)
    assert np.max(np.abs(out["series"] - s0[None, :])) < 1e-12


def test_sali_regular_vs_chaotic(orc):
    """SALI stays O(1) on regular orbits and decays exponentially (to < 1e-8) on chaotic
    orbits of Henon-Heiles at E = 1/8 (refs [56,57]; north_star).  The two ICs on the x = 0
    section: (y, py) = (0.25, 0) lies in the main regular island, (-0.15, 0) in the chaotic
    sea.  ln SALI decays at the rate of the mLE estimate from the same run."""
    E = 1.0 / 8.0
    ics = []
    for yv, pyv in ((0.25, 0.0), (-0.15, 0.0)):            # regular island / chaotic sea
        px = np.sqrt(2 * E - pyv * pyv - yv * yv + 2 * yv ** 3 / 3)
        ics.append([0.0, yv, px, pyv])
    y = np.ascontiguousarray(np.array(ics).T)
    w = wl.deviation_vectors(2, 2, 4, 0, "unit")
    L = np.zeros((2, 2))
    out = orc.sali(HH, None, y, w, t0=0.0, h=0.05, n_steps=20_000, renorm_every=1, sample_every=2000, lognorm=L,
                   precision="f64")
    ser = out["series"]                                       # t = 100, 200, ..., 1000, final
    assert ser[-1, 0] > 1e-2 and ser[:, 0].min() > 1e-3, ser[:, 0]    # regular: O(1) (oscillates)
    assert ser[-1, 1] < 1e-8, ser[:, 1]                               # chaotic: decayed
    lam = L[0] / 1000.0                                       # finite-time mLE estimates
    assert lam[1] > 0.03 and lam[0] < 0.02
    # exponential decay on the chaotic orbit: SALI ~ exp(-(l1 - l2) t) = exp(-l1 t) in 2 DoF
    t = 100.0 * np.arange(1, 11)
    ok = ser[:10, 1] > 1e-12
    assert ok.sum() >= 3
    slope = np.polyfit(t[ok], np.log(ser[:10, 1][ok]), 1)[0]
    assert -2.5 * lam[1] < slope < -0.4 * lam[1], (slope, lam)


def test_c1_like_horizon_all_regular_class(orc):
    """At C1's horizon (t = 100, E = 1/8) no orbit has SALI < 1e-8 yet."""
    cfg = wl.config("C1", 64)
    y, w = cfg["y"].copy(), cfg["w"].copy()
    out = orc.sali(HH, None, y, w, t0=0.0, h=0.05, n_steps=2000, renorm_every=1, precision="f64")
    s = out["series"][-1]
    assert np.all(s > 1e-8) and np.all(s <= np.sqrt(2) + 1e-15)


# ----------------------------------------------------------------------------- Lyapunov spectrum
def test_lyapunov_sum_zero_and_pairing(orc):
    """Hamiltonian flow: sum(lambda) = 0 (Liouville) and lambda_v + lambda_{n+1-v} ~ 0; the
    middle pair -> 0 (reading R13: an autonomous Hamiltonian has TWO zero exponents)."""
    cfg = wl.config("C4", 8)
    y, w = cfg["y"].copy(), cfg["w"].copy()
    S = np.zeros((6, 8))
    T = 1000.0
    out = orc.lyap(C3, cfg["params"], y, w, t0=0.0, h=0.01, n_steps=100_000, renorm_every=10, logsum=S,
                   precision="f64")
    lam = out["lam"]
    assert np.max(np.abs(lam - S / T)) < 1e-15
    assert np.max(np.abs(lam.sum(0))) < 1e-12
    assert np.max(np.abs(lam + lam[::-1])) < 2e-3          # finite-time effect ~ ln t / t
    assert np.max(np.abs(lam[2:4])) < 2e-3
    assert np.all(np.diff(lam, axis=0) <= 1e-3)             # ordered (weakly) descending
    # returned vectors are orthonormal
    G = np.einsum("anc,bnc->abc", w, w)
    assert np.max(np.abs(G - np.eye(6)[:, :, None])) < 1e-13


def test_lyapunov_linear_system_and_k1_consistency(orc):
    """Uncoupled oscillators: all exponents -> 0 like 1/t.  k = 1 run (plain
    renormalisation, the mLE) equals lambda_1 of the full-spectrum run from the same w_1."""
    P = wl.coupled3_params(0.0)
    y = np.random.default_rng(1).uniform(-0.5, 0.5, size=(6, 4))
    w = wl.deviation_vectors(4, 6, 6, 5, "orthonormal")
    out = orc.lyap(C3, P, y.copy(), w.copy(), t0=0.0, h=0.01, n_steps=50_000, renorm_every=10, precision="f64")
    assert np.max(np.abs(out["lam"])) < 5e-3
    cfg = wl.config("C4", 4)
    full = orc.lyap(C3, cfg["params"], cfg["y"].copy(), cfg["w"].copy(), t0=0.0, h=0.01, n_steps=20_000,
                    renorm_every=10, precision="f80")
    one = orc.lyap(C3, cfg["params"], cfg["y"].copy(), cfg["w"][:1].copy(), t0=0.0, h=0.01, n_steps=20_000,
                   renorm_every=10, precision="f80")
    assert np.max(np.abs(full["lam"][0] - one["lam"][0])) < 1e-12
    # and equals the lognorm of a MODE_NORM run on that single vector
    L = np.zeros((1, 4))
    orc.run(C3, cfg["params"], cfg["y"].copy(), cfg["w"][:1].copy(), t0=0.0, h=0.01, n_steps=20_000,
            mode=orc.MODE_NORM, renorm_every=10, logacc=L, precision="f80")
    assert np.max(np.abs(L[0] / 200.0 - one["lam"][0])) < 1e-13


def test_henon_heiles_chaotic_mle_positive(orc):
    E = 1.0 / 6.0
    yv = -0.25
    y = np.array([[0.0], [yv], [np.sqrt(2 * E - yv * yv + 2 * yv ** 3 / 3)], [0.0]])
    w = wl.deviation_vectors(1, 4, 4, 1, "orthonormal")
    out = orc.lyap(HH, None, y, w, t0=0.0, h=0.05, n_steps=40_000, renorm_every=5, precision="f64")
    lam = out["lam"][:, 0]
    assert 0.03 < lam[0] < 0.2
    assert abs(lam.sum()) < 1e-12 and abs(lam[0] + lam[3]) < 5e-3 and max(abs(lam[1]), abs(lam[2])) < 1e-2


# ----------------------------------------------------------------------------- GALI behaviour
def test_gali_series_fput(orc):
    cfg = wl.config("C5", 8)
    y, w = cfg["y"].copy(), cfg["w"].copy()
    out = orc.gali(FPUT, cfg["params"], y, w, t0=0.0, h=0.05, n_steps=2000, renorm_every=10, sample_every=50,
                   precision="f64")
    ser = out["series"]
    assert ser.shape == (5, 8)
    assert np.all(ser > 0) and np.all(ser <= 1 + 1e-14)
    # cross-check the final value against LAPACK on the returned unit vectors
    for ic in range(8):
        sv = np.linalg.svd(w[:, :, ic].T, compute_uv=False)
        assert abs(ser[-1, ic] - np.prod(sv)) < 1e-12 * np.prod(sv)
    assert np.max(np.abs(np.linalg.norm(w, axis=1) - 1)) < 1e-14


# ----------------------------------------------------------------------------- Lagrangian descriptor
def test_ld_closed_form_isotropic_oscillator(orc):
    """All w = 1, eps = 0: |f| = sqrt(|p|^2 + |q|^2) = sqrt(2E) constant => M+ = M- = tau sqrt(2E)."""
    P = np.array([1.0, 1.0, 1.0, 0.0])
    y = np.random.default_rng(3).uniform(-0.5, 0.5, size=(6, 8))
    E = 0.5 * (y ** 2).sum(0)
    f, b = orc.ld(C3, P, y, 0.0, 0.01, 5000, precision="f64")
    ref = 50.0 * np.sqrt(2 * E)
    assert np.max(np.abs(f - ref) / ref) < 1e-12 and np.max(np.abs(b - ref) / ref) < 1e-12


def test_ld_is_arc_length_of_a_known_curve(orc):
    """1-DoF content: w = (1, sqrt2, sqrt3) uncoupled, only oscillator 1 excited: the orbit
    is the circle q^2 + p^2 = r^2 traversed at unit angular speed, arc length = r * tau."""
    P = wl.coupled3_params(0.0)
    y = np.zeros((6, 3))
    y[0] = [0.3, 0.1, -0.2]
    y[3] = [0.0, 0.25, 0.1]
    r = np.sqrt(y[0] ** 2 + y[3] ** 2)
    f, b = orc.ld(C3, P, y, 0.0, 0.02, 1000, precision="f80")
    assert np.max(np.abs(f - 20.0 * r)) < 1e-13 and np.max(np.abs(b - 20.0 * r)) < 1e-13


def test_ld_mirror_symmetry_and_h_independence(orc):
    """Time reversal (p -> -p) maps the x = 0 section to itself with px -> -px; combined
    with the x -> -x reflection symmetry of Eq.(4): M-(y, py) = M+(y, -py) on the
    py-symmetric grid.  And the value does not depend on h (quadrature of order 8)."""
    side = 8
    y0 = wl.hh_grid(0.125, side, side)
    f, b = orc.ld(HH, None, y0, 0.0, 0.01, 5000, precision="f64")
    F, B = f.reshape(side, side), b.reshape(side, side)
    assert np.max(np.abs(B - F[:, ::-1])) < 1e-11
    f2, _ = orc.ld(HH, None, y0, 0.0, 0.005, 10_000, backward=False, precision="f64")
    assert np.max(np.abs(f2 - f) / f) < 1e-12
    assert f.min() > 15 and f.max() < 35 and np.all(y0 == wl.hh_grid(0.125, side, side))   # y0 untouched


def test_ld_matches_scipy_quadrature(orc):
    """Library pin: integrate (x, M) with M' = |f(x)| by solve_ivp(DOP853, tight tol)."""
    from scipy.integrate import solve_ivp
    y0 = np.ascontiguousarray(wl.hh_grid(0.125, 4, 4)[:, [2, 7, 13]])
    f, b = orc.ld(HH, None, y0, 0.0, 0.01, 1000, precision="f80")

    def fun(t, Y):
        g = orc.rhs(HH, None, Y[:4])
        return np.concatenate([g, [np.linalg.norm(g)]])
    for i in range(3):
        for sgn, val in ((1, f[i]), (-1, b[i])):
            sol = solve_ivp(fun, (0.0, sgn * 10.0), np.concatenate([y0[:, i], [0.0]]), method="DOP853", rtol=1e-13,
                            atol=1e-13)
            assert abs(abs(sol.y[4, -1]) - val) < 1e-10


def test_ld_adaptive_closed_form_and_fixed_step_value(orc):
    """Adaptive LD (augmented ODE, M' = |f|): the isotropic oscillator has |f| = sqrt(2E) constant, so
    M+ = M- = tau sqrt(2E) whatever the step sequence; on Henon-Heiles the value is the fixed-step
    quadrature's (a different discretisation of the same integral) and the mirror symmetry holds."""
    P = np.array([1.0, 1.0, 1.0, 0.0])
    y = np.random.default_rng(3).uniform(-0.5, 0.5, size=(6, 8))
    E = 0.5 * (y ** 2).sum(0)
    r = orc.ld_adaptive(C3, P, y, 0.0, 50.0, rtol=1e-12, atol=1e-12, precision="f64")
    ref = 50.0 * np.sqrt(2 * E)
    assert (r["status"] == 0).all()
    assert np.max(np.abs(r["fwd"] - ref) / ref) < 1e-11 and np.max(np.abs(r["bwd"] - ref) / ref) < 1e-11
    side = 6
    y0 = wl.hh_grid(0.125, side, side)
    f, b = orc.ld(HH, None, y0, 0.0, 0.01, 2000, precision="f80")
    ra = orc.ld_adaptive(HH, None, y0, 0.0, 20.0, rtol=1e-12, atol=1e-12, precision="f80")
    assert np.max(np.abs(ra["fwd"] / f - 1)) < 1e-10 and np.max(np.abs(ra["bwd"] / b - 1)) < 1e-10
    assert np.max(np.abs(ra["bwd"].reshape(side, side) - ra["fwd"].reshape(side, side)[:, ::-1])) < 1e-9
    assert (ra["n_accepted"] > 100).all() and np.all(y0 == wl.hh_grid(0.125, side, side))


def test_ld_adaptive_is_solve_ivp_on_the_augmented_system(orc):
    """Library pin of the step sequence: solve_ivp(DOP853) on (y, M) with the same tolerances takes the same
    number of accepted steps and ends at the same M (M takes part in the error norm, D = n + 1); backward in
    time M decreases and the descriptor is -M."""
    from scipy.integrate import solve_ivp
    y0 = np.ascontiguousarray(wl.hh_grid(1.0 / 6.0, 5, 5)[:, [3, 11, 17]])
    r = orc.ld_adaptive(HH, None, y0, 0.0, 30.0, rtol=1e-9, atol=1e-9, precision="f64", threads=1)

    def fun(t, Y):
        g = orc.rhs(HH, None, Y[:4])
        return np.concatenate([g, [np.linalg.norm(g)]])
    for i in range(3):
        for row, sgn, val in ((0, 1, r["fwd"][i]), (1, -1, r["bwd"][i])):
            sol = solve_ivp(fun, (0.0, sgn * 30.0), np.concatenate([y0[:, i], [0.0]]), method="DOP853", rtol=1e-9,
                            atol=1e-9)
            assert abs(sgn * sol.y[4, -1] - val) < 1e-11 * val
            assert abs((len(sol.t) - 1) - r["n_accepted"][row, i]) <= 1


def test_ld_adaptive_status_and_arguments(orc):
    """max_steps exhausted -> status 3 and NaN for that direction; tau = 0 -> M = 0; bad tolerances refused."""
    y0 = wl.hh_grid(0.125, 3, 3)
    r = orc.ld_adaptive(HH, None, y0, 0.0, 50.0, rtol=1e-12, atol=1e-12, max_steps=20)
    assert (r["status"] == 3).all() and np.isnan(r["fwd"]).all() and np.isnan(r["bwd"]).all()
    assert (r["n_accepted"] + r["n_rejected"] == 20).all()
    r = orc.ld_adaptive(HH, None, y0, 0.0, 0.0, rtol=1e-9, atol=1e-9)
    assert (r["fwd"] == 0).all() and (r["bwd"] == 0).all()
    with pytest.raises(ValueError):
        orc.ld_adaptive(HH, None, y0, 0.0, 1.0, rtol=0.0, atol=1e-9)


# ----------------------------------------------------------------------------- continuation / sampling
def test_checkpoint_continuation(orc):
    """One call of n steps == two calls of n/2 (split on a renormalisation boundary)."""
    cfg = wl.config("C4", 4)
    P = cfg["params"]
    ya, wa, Sa = cfg["y"].copy(), cfg["w"].copy(), np.zeros((6, 4))
    orc.lyap(C3, P, ya, wa, t0=0.0, h=0.01, n_steps=2000, renorm_every=10, logsum=Sa, precision="f64")
    yb, wb, Sb = cfg["y"].copy(), cfg["w"].copy(), np.zeros((6, 4))
    orc.lyap(C3, P, yb, wb, t0=0.0, h=0.01, n_steps=1000, renorm_every=10, logsum=Sb, precision="f64")
    orc.lyap(C3, P, yb, wb, t0=10.0, h=0.01, n_steps=1000, renorm_every=10, logsum=Sb, precision="f64")
    assert np.array_equal(ya, yb)
    assert np.max(np.abs(wa - wb)) < 1e-14 and np.max(np.abs(Sa - Sb)) < 1e-13


def test_sampling_layout(orc):
    assert orc.n_samples(100, 1, 0) == 1
    assert orc.n_samples(100, 1, 10) == 11
    assert orc.n_samples(105, 10, 2) == 6          # 11 renormalisations (last at step 105)
    cfg = wl.config("C1", 4)
    y, w = cfg["y"].copy(), cfg["w"].copy()
    out = orc.sali(HH, None, y, w, t0=0.0, h=0.01, n_steps=105, renorm_every=10, sample_every=2, precision="f64")
    ser = out["series"]
    assert ser.shape == (6, 4)
    # slot j is the value after renormalisation 2(j+1), i.e. step 20(j+1): rerun to check
    for j in range(5):
        y2, w2 = cfg["y"].copy(), cfg["w"].copy()
        o2 = orc.sali(HH, None, y2, w2, t0=0.0, h=0.01, n_steps=20 * (j + 1), renorm_every=10, precision="f64")
        assert np.max(np.abs(o2["series"][-1] - ser[j])) < 1e-13


def test_adaptive_sali_runs_and_counts(orc):
    cfg = wl.config("C3", 16)
    y, w = cfg["y"].copy(), cfg["w"].copy()
    out = orc.sali(HH, None, y, w, adaptive=True, t0=0.0, t_end=50.0, rtol=1e-12, atol=1e-12, renorm_every=1,
                   precision="f64")
    assert np.all(out["status"] == 0) and np.all(out["t_final"] == 50.0)
    assert np.all(out["n_accepted"] > 300) and np.all(out["n_accepted"] < 700)
    s = out["series"][-1]
    assert np.all((s >= 0) & (s <= np.sqrt(2) + 1e-15))
    assert np.max(np.abs(np.linalg.norm(w, axis=1) - 1)) < 1e-14


def test_invalid_arguments(orc):
    y = wl.hh_grid(0.125, 2, 2)
    w = wl.deviation_vectors(4, 3, 4, 0)
    with pytest.raises(ValueError):
        orc.sali(HH, None, y, w, t0=0.0, h=0.01, n_steps=10)            # SALI needs k = 2
    with pytest.raises(ValueError):
        orc.integrate_fixed(HH, None, y, 0.0, 0.0, 10)                   # h = 0
    with pytest.raises(ValueError):
        orc.integrate_adaptive(HH, None, y, 0.0, 1.0, 0.0, 1e-9)         # rtol = 0
    out = orc.integrate_fixed(HH, None, np.zeros((4, 0)), 0.0, 0.01, 10)  # empty ensemble: no-op
    assert out["status"].size == 0


# ----------------------------------------------------------------------------- LD neighbours
def test_ld_neighbours_closed_form_and_ordering(orc):
    """Equal frequencies, no coupling: |f| = |y| is constant along an orbit, so M(x) = tau |x| for EVERY
    initial condition, on or off the energy surface.  The members' LDs and the raw differences are then
    analytic: M(x0 +- sigma e_i) = tau |x0 +- sigma e_i|.  The components of x0 are all distinct, so a
    wrong component, a wrong sign or a wrong row order changes the expected value."""
    prm = np.array([1.0, 1.0, 1.0, 0.0])
    rng = np.random.default_rng(11)
    y0 = np.ascontiguousarray(rng.uniform(0.2, 1.0, size=(6, 9)) * rng.choice([-1.0, 1.0], size=(6, 9)))
    sigma, h, ns = 0.05, 0.01, 800
    tau = h * ns
    r = orc.ld_neighbours(C3, prm, y0, sigma, 0.0, h, ns, precision="f64")
    assert r["fwd"].shape == (13, 9) and r["diff_fwd"].shape == (12, 9)
    M0 = tau * np.linalg.norm(y0, axis=0)
    assert np.abs(r["fwd"][0] / M0 - 1).max() <= 1e-12 and np.abs(r["bwd"][0] / M0 - 1).max() <= 1e-12
    for i in range(6):
        for s, row in ((+1.0, 1 + 2 * i), (-1.0, 2 + 2 * i)):
            yd = y0.copy()
            yd[i] += s * sigma
            Md = tau * np.linalg.norm(yd, axis=0)
            assert np.abs(r["fwd"][row] / Md - 1).max() <= 1e-12, (i, s)
            assert np.abs(r["bwd"][row] / Md - 1).max() <= 1e-12, (i, s)
            assert np.abs(r["diff_fwd"][row - 1] - np.abs(Md - M0)).max() <= 1e-11, (i, s)
            assert np.abs(r["diff_bwd"][row - 1] - np.abs(Md - M0)).max() <= 1e-11, (i, s)
    # central difference of the members -> the analytic gradient tau x_i / |x|, error O(sigma^2)
    grad = (r["fwd"][1::2] - r["fwd"][2::2]) / (2 * sigma)
    exact = tau * y0 / np.linalg.norm(y0, axis=0)
    assert np.abs(grad - exact).max() <= 2.0 * tau * sigma ** 2


def test_ld_neighbours_sigma_zero_and_generator(orc):
    """sigma = 0: every member is the centre, all differences vanish exactly.  sigma > 0 on a system whose
    components are not interchangeable (Henon-Heiles): every member equals the LD of the displaced IC built
    here with numpy."""
    y0 = wl.hh_grid(0.125, 5, 4)
    r0 = orc.ld_neighbours(HH, None, y0, 0.0, 0.0, 0.01, 300, precision="f64")
    assert (r0["fwd"] == r0["fwd"][0]).all() and (r0["bwd"] == r0["bwd"][0]).all()
    assert (r0["diff_fwd"] == 0).all() and (r0["diff_bwd"] == 0).all()
    f0, b0 = orc.ld(HH, None, y0, 0.0, 0.01, 300, precision="f64")
    assert (r0["fwd"][0] == f0).all() and (r0["bwd"][0] == b0).all()
    sigma = 1e-3
    r = orc.ld_neighbours(HH, None, y0, sigma, 0.0, 0.01, 300, precision="f64")
    for m in range(1, 9):
        yd = y0.copy()
        yd[(m - 1) // 2] += sigma if (m - 1) % 2 == 0 else -sigma
        fd, bd = orc.ld(HH, None, yd, 0.0, 0.01, 300, precision="f64")
        assert (r["fwd"][m] == fd).all() and (r["bwd"][m] == bd).all(), m
        assert (r["diff_fwd"][m - 1] == np.abs(fd - f0)).all()
    # the differences shrink linearly with sigma (M is smooth over t = 3)
    r2 = orc.ld_neighbours(HH, None, y0, sigma / 2, 0.0, 0.01, 300, precision="f64")
    ratio = r["diff_fwd"] / r2["diff_fwd"]
    assert np.median(np.abs(ratio - 2.0)) <= 0.01 and np.abs(ratio - 2.0).max() <= 0.25   # (small gradients: O(sigma^2) shows)
    with pytest.raises(ValueError):
        orc.ld_neighbours(HH, None, y0, -1.0, 0.0, 0.01, 10)
