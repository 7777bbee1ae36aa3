"""GPU parity tests: the CUDA path (through the C ABI, via the ctypes binding) against the CPU
oracle on the same seeded inputs, element by element.  Sizes: the oracle finishes each in
seconds, ensembles span several thread blocks and end in a ragged tail.

Tolerances (BASELINE.json north_star):
  states, fixed step, t <= 10 Lyapunov times : |dy|_2 / |y|_2 <= 1e-10 per trajectory
  indicators on regular orbits               : relative 1e-8
The truth is the oracle in x86 80-bit long double ("f80"); the double oracle is reported too.
"""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as W

pytestmark = pytest.mark.gpu

HH, C3, FPUT = W.SYS_HENON_HEILES, W.SYS_COUPLED3, W.SYS_FPUT
TOL_STATE = 1e-10
TOL_IND = 1e-8


@pytest.fixture(scope="module")
def chs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_00622_b200 import binding
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel_state(y_gpu, y_ref):
    """per-trajectory |dy|_2/|y|_2 over the leading axis (components)."""
    y_gpu = y_gpu.reshape(-1, y_gpu.shape[-1])
    y_ref = y_ref.reshape(-1, y_ref.shape[-1])
    return np.linalg.norm(y_gpu - y_ref, axis=0) / np.linalg.norm(y_ref, axis=0)


# ---------------------------------------------------------------------------- plain integration
@pytest.mark.parametrize("h", [0.01, -0.01])
def test_integrate_fixed_hh(chs, orc, h):
    y0 = W.hh_grid(0.125, 19, 17)  # 323 ICs: 2 full blocks + ragged tail
    yo = y0.copy()
    orc.integrate_fixed(HH, None, yo, 0.0, h, 3000, precision="f80")
    yg = dev(y0)
    rep = chs.Report(y0.shape[1], "cuda")
    chs.integrate_fixed(HH, None, yg, 0.0, h, 3000, report=rep)
    r = rel_state(yg.cpu().numpy(), yo)
    assert r.max() <= TOL_STATE, r.max()
    assert (rep.status.cpu().numpy() == 0).all()
    assert (rep.n_accepted.cpu().numpy() == 3000).all()
    np.testing.assert_allclose(rep.t_final.cpu().numpy(), 3000 * h, rtol=1e-15)


def test_integrate_fixed_coupled3_exact(chs, orc):
    """eps = 0: uncoupled oscillators, closed form q cos(wt) + p/w sin(wt)."""
    prm = W.coupled3_params(0.0)
    y0 = W.coupled3_ics(200, seed=5, E=0.1, eps=0.0)
    yg = dev(y0)
    chs.integrate_fixed(C3, prm, yg, 0.0, 0.01, 5000)
    t = 50.0
    w = prm[:3][:, None]
    q = y0[:3] * np.cos(w * t) + y0[3:] / w * np.sin(w * t)
    p = -y0[:3] * w * np.sin(w * t) + y0[3:] * np.cos(w * t)
    r = rel_state(yg.cpu().numpy(), np.concatenate([q, p]))
    assert r.max() <= 1e-11, r.max()


def test_integrate_fixed_coupled3(chs, orc):
    prm = W.coupled3_params(0.1)
    y0 = W.coupled3_ics(300, seed=1)
    yo = y0.copy()
    orc.integrate_fixed(C3, prm, yo, 0.0, 0.01, 2000, precision="f80")
    yg = dev(y0)
    chs.integrate_fixed(C3, prm, yg, 0.0, 0.01, 2000)
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE


def test_resume(chs):
    """In-place continuation (checkpoint / resume): with the carried rounding
    words of the compensated orbit update handed over (chs_report.carry, resume = 1) one call of n
    steps == two calls, BIT FOR BIT.  Without the carry the boundary drops one rounding word per
    component (<= 1 ulp)."""
    y0 = W.hh_grid(0.125, 16, 16)
    a = dev(y0)
    b = dev(y0)
    chs.integrate_fixed(HH, None, a, 0.0, 0.01, 1000)
    rep = chs.Report(256, "cuda", n=4)
    chs.integrate_fixed(HH, None, b, 0.0, 0.01, 400, report=rep)
    assert rep.carry.abs().max().item() > 0.0
    rep.resume = True
    chs.integrate_fixed(HH, None, b, 4.0, 0.01, 600, report=rep)
    assert (a == b).all().item()
    # without the carry: last-digit differences only
    d = dev(y0)
    chs.integrate_fixed(HH, None, d, 0.0, 0.01, 400)
    chs.integrate_fixed(HH, None, d, 4.0, 0.01, 600)
    assert rel_state(d.cpu().numpy(), a.cpu().numpy()).max() <= 1e-13
    # and a repeated call is deterministic, bit for bit
    c = dev(y0)
    chs.integrate_fixed(HH, None, c, 0.0, 0.01, 1000)
    assert (a == c).all().item()


def test_empty_and_single(chs, orc):
    import torch
    y = torch.empty((4, 0), dtype=torch.float64, device="cuda")
    chs.integrate_fixed(HH, None, y, 0.0, 0.01, 10)
    f, b = chs.ld(HH, None, y, 0.0, 0.01, 10)
    assert f.numel() == 0 and b.numel() == 0
    y1 = W.hh_grid(0.125, 1, 1)
    yo = y1.copy()
    orc.integrate_fixed(HH, None, yo, 0.0, 0.01, 100, precision="f80")
    yg = dev(y1)
    chs.integrate_fixed(HH, None, yg, 0.0, 0.01, 100)
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE


def test_argument_errors(chs):
    import torch
    y = torch.zeros((4, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(chs.ChaoticusError):
        chs.integrate_fixed(HH, None, y, 0.0, 0.0, 10)            # h = 0
    with pytest.raises(chs.ChaoticusError):
        chs.integrate_adaptive(HH, None, y, 0.0, 1.0, 0.0, 1e-9)  # rtol = 0
    with pytest.raises(chs.ChaoticusError):
        chs.integrate_fixed(7, None, y, 0.0, 0.01, 10)            # unknown system
    w = torch.zeros((2, 4, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(chs.ChaoticusError):
        chs.sali(HH, None, y, w, renorm_every=0, h=0.01, n_steps=10)
    with pytest.raises(ValueError):
        chs.integrate_fixed(HH, None, y[:, ::2], 0.0, 0.01, 10)    # non-contiguous


def test_nonfinite_status(chs):
    """An escaping Henon-Heiles orbit (E far above 1/6) overflows: status 1, outputs NaN."""
    y0 = W.hh_grid(0.125, 4, 4)
    y0[:, 3] = [0.0, 3.0, 0.0, 5.0]   # far outside the bounded region
    yg = dev(y0)
    rep = chs.Report(16, "cuda")
    chs.integrate_fixed(HH, None, yg, 0.0, 0.05, 4000, report=rep)
    st = rep.status.cpu().numpy()
    out = yg.cpu().numpy()
    assert st[3] == chs.ST_NONFINITE and np.isnan(out[:, 3]).all()
    ok = np.delete(np.arange(16), 3)
    assert (st[ok] == 0).all() and np.isfinite(out[:, ok]).all()


DEATH_CHECK_EVERY = 8      # csrc/dop8_core.cuh kDeathCheckEvery


def _report_matches(rep, ro, t0, h, n_steps):
    """Report of a fixed-step run against the oracle's.  Live trajectories: identical.  Dead ones: the oracle
    stops at the step s after which its state is not finite; the kernels test after every 8th step and after
    the last, so they report the first tested step >= their own s -- and their own s may be s -+ 1: in the
    step of death magnitudes jump by hundreds of decades and WHICH intermediate overflows first (the kernels
    carry h^2-scaled forces) decides between two neighbouring steps.  t_final = t0 + n_accepted h on both."""
    st, na, tf = rep.status.cpu().numpy(), rep.n_accepted.cpu().numpy(), rep.t_final.cpu().numpy()
    assert np.array_equal(st, ro["status"]), (np.flatnonzero(st != ro["status"]), st[st != ro["status"]])
    s = ro["n_accepted"]
    up = lambda x: np.minimum(-(-x // DEATH_CHECK_EVERY) * DEATH_CHECK_EVERY, n_steps)
    dead = st != 0
    lo, hi = np.where(dead, up(np.maximum(s - 1, 1)), s), np.where(dead, up(s + 1), s)
    d = np.flatnonzero((na < lo) | (na > hi))
    assert d.size == 0, (d, na[d], s[d])
    assert ((na[dead] % DEATH_CHECK_EVERY == 0) | (na[dead] == n_steps)).all()
    assert np.abs(tf - (t0 + na * h)).max() <= 4e-16 * np.abs(tf).max()
    assert np.abs(tf[~dead] - ro["t_final"][~dead]).max(initial=0.0) <= 4e-16 * np.abs(tf).max()
    assert (rep.n_rejected.cpu().numpy() == 0).all()
    return st, na


@pytest.mark.parametrize("case", ["hh_integrate", "hh_sali_tile", "hh_gali3_thread", "c3_lyap", "fput8_gali4",
                                  "fput12_gali4_pad", "fput100_sali_wide", "dp_integrate", "dp_sali"])
def test_fixed_step_dead_trajectories_report_where_they_died(chs, orc, case):
    """A fixed-step trajectory whose state stops being finite (an escaping orbit: Henon-Heiles above the
    escape energy, the cubic terms of the 3-DoF system and of the alpha-FPUT chain) is reported as the oracle
    reports it: status 1, n_accepted = the step after which the state was first found non-finite (tested after
    every 8th step: _report_matches), t_final = t0 + n_accepted h, outputs NaN -- not the end of the run.  Both sides take that decision in double precision
    (oracle "f64": the 80-bit oracle overflows later).  Every layout: thread, column tile, chain tile (exact,
    padded, wide), generic first-order kernels; live neighbours in the same warp are untouched."""
    rng = np.random.default_rng(11)
    h, n_steps, m = 0.02, 2000, 7
    dead = [3, 17, 40]                                       # spread over two warps of the thread layout
    if case.startswith("hh"):
        sysid, prm = HH, None
        y0 = np.ascontiguousarray(W.hh_grid(0.125, 9, 5))     # 45 ICs
        for j, i in enumerate(dead):
            y0[:, i] = [0.0, 2.0 + j, 0.0, 3.0 + 2 * j]       # far outside the bounded region: different death steps
    elif case.startswith("c3"):
        sysid, prm = C3, W.coupled3_params(0.5)
        y0 = W.coupled3_ics(45, seed=2, eps=0.5)
        for j, i in enumerate(dead):
            y0[:, i] = [3.0 + j, -4.0, -5.0 - j, 0.0, 0.0, 0.0]
    elif case.startswith("fput"):
        N = int(case[4:].split("_")[0])
        sysid, prm = FPUT, W.fput_params(N, 1.0, 1.0, 0.0)    # alpha-FPUT: the cubic potential is unbounded below
        y0 = W.fput_ics(45, N, seed=4, E=0.01 * N)
        for j, i in enumerate(dead):
            y0[:N, i] = -(4.0 + j) * (N + 1) / 9.0 * np.sin(np.pi * np.arange(1, N + 1) / (N + 1))   # same stretch per spring
    else:
        sysid, prm = W.SYS_DOUBLE_PENDULUM, (1.0, 1.0)
        y0 = W.double_pendulum_ics(45, seed=3)
        y0[2, 3], y0[3, 17], y0[0, 40] = np.inf, -np.inf, np.nan      # the pendulum cannot escape: dead on arrival
    n, n_ic = y0.shape
    what = case.split("_")[1]
    k = {"integrate": 0, "sali": 2, "gali3": 3, "gali4": 4, "lyap": 3}[what]
    w0 = W.deviation_vectors(n_ic, k, n, 5, "orthonormal") if k else None
    rep = chs.Report(n_ic, "cuda")
    yo, yg = y0.copy(), dev(y0)
    wo, wg = (w0.copy(), dev(w0)) if k else (None, None)
    if what == "integrate":
        ro = orc.integrate_fixed(sysid, prm, yo, 0.5, h, n_steps, precision="f64")
        chs.integrate_fixed(sysid, prm, yg, 0.5, h, n_steps, report=rep)
    elif what == "sali":
        ro = orc.sali(sysid, prm, yo, wo, renorm_every=m, sample_every=20, t0=0.5, h=h, n_steps=n_steps, precision="f64")
        out = chs.sali(sysid, prm, yg, wg, renorm_every=m, sample_every=20, t0=0.5, h=h, n_steps=n_steps, report=rep)
    elif what.startswith("gali"):
        ro = orc.gali(sysid, prm, yo, wo, renorm_every=m, sample_every=20, t0=0.5, h=h, n_steps=n_steps, precision="f64")
        out = chs.gali(sysid, prm, yg, wg, renorm_every=m, sample_every=20, t0=0.5, h=h, n_steps=n_steps, report=rep)
    else:
        ro = orc.lyap(sysid, prm, yo, wo, renorm_every=m, t0=0.5, h=h, n_steps=n_steps, precision="f64")
        out = chs.lyap(sysid, prm, yg, wg, renorm_every=m, t0=0.5, h=h, n_steps=n_steps, report=rep)
    st, na = _report_matches(rep, ro, 0.5, h, n_steps)
    assert (st[dead] == chs.ST_NONFINITE).all() and (na[dead] < n_steps).all() and (na[dead] >= 1).all()
    live = np.delete(np.arange(n_ic), dead)
    assert (st[live] == 0).all() and (na[live] == n_steps).all()
    yg = yg.cpu().numpy()
    assert np.isnan(yg[:, dead]).all() and np.isnan(yo[:, dead]).all() and np.isfinite(yg[:, live]).all()
    if k:
        assert np.isnan(wg.cpu().numpy()[:, :, dead]).all() and np.isfinite(wg.cpu().numpy()[:, :, live]).all()
        out = out.cpu().numpy()
        ref = ro["lam"] if what == "lyap" else ro["series"]
        assert np.array_equal(np.isnan(out), np.isnan(ref))   # rows sampled before the death keep their values
        assert np.isnan(out[-1, dead]).all() and np.isfinite(out[:, live]).all()
    # a report with t_final only (no n_accepted array) says the same
    if what == "integrate":
        import torch
        rep2 = chs.Report(n_ic, "cuda")
        c = rep2._struct()
        c.n_accepted = None
        rep2._struct = lambda: c
        y2 = dev(y0)
        chs.integrate_fixed(sysid, prm, y2, 0.5, h, n_steps, report=rep2)
        assert torch.equal(rep2.t_final, rep.t_final) and torch.equal(rep2.status, rep.status)


# ---------------------------------------------------------------------------- Lagrangian descriptor
def test_ld_hh(chs, orc):
    y0 = W.hh_grid(0.125, 37, 37)  # 1369 ICs
    fo, bo = orc.ld(HH, None, y0, 0.0, 0.01, 1500, precision="f80")
    f, b = chs.ld(HH, None, dev(y0), 0.0, 0.01, 1500)
    f, b = f.cpu().numpy(), b.cpu().numpy()
    assert np.abs(f / fo - 1).max() <= TOL_IND and np.abs(b / bo - 1).max() <= TOL_IND
    # time-reversal + reflection symmetry on the py-symmetric grid: M-(y,py) = M+(y,-py)
    F = f.reshape(37, 37)
    B = b.reshape(37, 37)
    assert np.abs(B - F[:, ::-1]).max() <= 1e-12
    # one direction only
    f2, none = chs.ld(HH, None, dev(y0), 0.0, 0.01, 1500, backward=False)
    assert none is None and (f2.cpu().numpy() == f).all()
    none, b2 = chs.ld(HH, None, dev(y0), 0.0, 0.01, 1500, forward=False)
    assert (b2.cpu().numpy() == b).all()


def test_ld_harmonic_closed_form(chs):
    """All omega = 1, eps = 0: |f| = sqrt(2E) is constant, M+ = M- = tau sqrt(2E)."""
    prm = np.array([1.0, 1.0, 1.0, 0.0])
    rng = np.random.default_rng(3)
    y0 = np.ascontiguousarray(rng.uniform(-1, 1, size=(6, 257)))
    E = 0.5 * (y0 ** 2).sum(0)
    f, b = chs.ld(C3, prm, dev(y0), 0.0, 0.01, 2000)
    exact = 20.0 * np.sqrt(2 * E)
    assert np.abs(f.cpu().numpy() / exact - 1).max() <= 1e-12
    assert np.abs(b.cpu().numpy() / exact - 1).max() <= 1e-12


def test_ld_host_entry(chs, orc):
    y0 = W.hh_grid(0.125, 12, 12)
    f = np.empty(144)
    b = np.empty(144)
    chs.ld_host(HH, None, y0, 0.0, 0.01, 500, f, b)
    fd, bd = chs.ld(HH, None, dev(y0), 0.0, 0.01, 500)
    assert (fd.cpu().numpy() == f).all() and (bd.cpu().numpy() == b).all()


# ---------------------------------------------------------------------------- SALI, fixed step
def _sali_case(n_side=24, n_steps=2000):
    cfg = W.config("C1", n_ic=n_side * n_side)
    return cfg["y"], cfg["w"]


def test_sali_fixed_hh(chs, orc):
    y0, w0 = _sali_case()
    n_ic = y0.shape[1]
    yo, wo, lo = y0.copy(), w0.copy(), np.zeros((2, n_ic))
    ro = orc.sali(HH, None, yo, wo, renorm_every=1, sample_every=500, lognorm=lo, h=0.01, n_steps=2000,
                  precision="f80")
    yg, wg, lg = dev(y0), dev(w0), dev(np.zeros((2, n_ic)))
    sg = chs.sali(HH, None, yg, wg, renorm_every=1, sample_every=500, lognorm=lg, h=0.01, n_steps=2000)
    sg = sg.cpu().numpy()
    so = ro["series"]
    assert sg.shape == so.shape == (5, n_ic)
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    # t = 20 is far below 10 Lyapunov times for every orbit: all SALI values are O(1e-3..1)
    assert so.min() > 1e-6
    assert np.abs(sg / so - 1).max() <= TOL_IND
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    assert np.abs(lg.cpu().numpy() - lo).max() <= 1e-9
    # unit vectors on return
    nrm = np.linalg.norm(wg.cpu().numpy(), axis=1)
    assert np.abs(nrm - 1).max() <= 1e-14


def test_sali_fixed_hh_thread_layout(chs, orc):
    """Above 4096 trajectories chaoticus_sali switches from the 4-lane tile to one thread per
    trajectory (the kernel bench.py --workload C1sat times): same parity bar."""
    y0, w0 = _sali_case(67)          # 4489 ICs
    n_ic = y0.shape[1]
    assert chs.kernel_info(HH, None, chs.WHAT_SALI, k=2, n_ic=n_ic)["lanes"] == 1
    assert chs.kernel_info(HH, None, chs.WHAT_SALI, k=2, n_ic=1024)["lanes"] == 4
    yo, wo, lo = y0.copy(), w0.copy(), np.zeros((2, n_ic))
    so = orc.sali(HH, None, yo, wo, renorm_every=1, sample_every=200, lognorm=lo, h=0.01, n_steps=600,
                  precision="f80")["series"]
    yg, wg, lg = dev(y0), dev(w0), dev(np.zeros((2, n_ic)))
    sg = chs.sali(HH, None, yg, wg, renorm_every=1, sample_every=200, lognorm=lg, h=0.01, n_steps=600).cpu().numpy()
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    assert np.abs(sg / so - 1).max() <= TOL_IND
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9 and np.abs(lg.cpu().numpy() - lo).max() <= 1e-9


def test_sali_renorm_interval_and_tail(chs, orc):
    """m = 7 does not divide n_steps = 1000: a final renormalisation happens at the end."""
    y0, w0 = _sali_case(10)
    n_ic = y0.shape[1]
    yo, wo = y0.copy(), w0.copy()
    ro = orc.sali(HH, None, yo, wo, renorm_every=7, sample_every=10, h=0.01, n_steps=1000, precision="f80")
    yg, wg = dev(y0), dev(w0)
    sg = chs.sali(HH, None, yg, wg, renorm_every=7, sample_every=10, h=0.01, n_steps=1000).cpu().numpy()
    assert sg.shape == ro["series"].shape
    assert np.abs(sg / ro["series"] - 1).max() <= TOL_IND
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-10


@pytest.mark.parametrize("n_side", [12, 70])   # 4-lane tile (<= 4096 ICs) and one thread per trajectory
def test_sali_resume(chs, n_side):
    """Split at a multiple of renorm_every with carry + resume: y, w and SALI bit-identical."""
    y0, w0 = _sali_case(n_side)
    n_ic = y0.shape[1]
    a_y, a_w = dev(y0), dev(w0)
    b_y, b_w = dev(y0), dev(w0)
    sa = chs.sali(HH, None, a_y, a_w, renorm_every=5, h=0.01, n_steps=1000)
    rep = chs.Report(n_ic, "cuda", n=4)
    chs.sali(HH, None, b_y, b_w, renorm_every=5, h=0.01, n_steps=500, report=rep)
    rep.resume = True
    sb = chs.sali(HH, None, b_y, b_w, renorm_every=5, t0=5.0, h=0.01, n_steps=500, report=rep)
    assert (a_y == b_y).all().item() and (a_w == b_w).all().item() and (sa == sb).all().item()
    # without carry / resume: the boundary drops the orbit's carried word and re-normalises the
    # already-unit vectors (|w| = 1 +- ulp): last-digit differences only
    c_y, c_w = dev(y0), dev(w0)
    chs.sali(HH, None, c_y, c_w, renorm_every=5, h=0.01, n_steps=500)
    sc = chs.sali(HH, None, c_y, c_w, renorm_every=5, t0=5.0, h=0.01, n_steps=500)
    assert rel_state(c_y.cpu().numpy(), a_y.cpu().numpy()).max() <= 1e-13
    assert (a_w - c_w).abs().max().item() <= 1e-12 and ((sa - sc).abs() / sa).max().item() <= 1e-11


def test_resume_all_layouts(chs):
    """Bit-identical continuation on every layout: column tile with two columns per lane + MGS (C4's
    kernel), chain tile + GALI (C5's kernel), one thread per trajectory + MGS, the generic kernel."""
    import torch
    cases = []
    cfg = W.config("C4", n_ic=203)
    cases.append(("lyap", C3, cfg["params"], cfg["y"], cfg["w"], 0.01, 6))
    cfg = W.config("C5", n_ic=101)
    cases.append(("gali", FPUT, cfg["params"], cfg["y"], cfg["w"], 0.05, 16))
    y0 = W.hh_grid(0.125, 11, 13)
    cases.append(("lyap", HH, None, y0, W.deviation_vectors(143, 2, 4, 12, "orthonormal"), 0.01, 4))
    for what, sysid, prm, y0, w0, h, n in cases:
        fn = getattr(chs, what)
        n_ic = y0.shape[1]
        a_y, a_w, b_y, b_w = dev(y0), dev(w0), dev(y0), dev(w0)
        oa = fn(sysid, prm, a_y, a_w, renorm_every=10, h=h, n_steps=600)
        rep = chs.Report(n_ic, "cuda", n=n)
        fn(sysid, prm, b_y, b_w, renorm_every=10, h=h, n_steps=250, report=rep)
        rep.resume = True
        ob = fn(sysid, prm, b_y, b_w, renorm_every=10, t0=250 * h, h=h, n_steps=350, report=rep)
        assert torch.equal(a_y, b_y) and torch.equal(a_w, b_w), (what, sysid)
        if what == "gali":
            assert torch.equal(oa, ob)
    DP = W.SYS_DOUBLE_PENDULUM
    y0 = W.double_pendulum_ics(200, seed=3)
    a, b = dev(y0), dev(y0)
    chs.integrate_fixed(DP, (1.0, 1.0), a, 0.0, 0.01, 500)
    rep = chs.Report(200, "cuda", n=4)
    chs.integrate_fixed(DP, (1.0, 1.0), b, 0.0, 0.01, 123, report=rep)
    rep.resume = True
    chs.integrate_fixed(DP, (1.0, 1.0), b, 1.23, 0.01, 377, report=rep)
    assert torch.equal(a, b)
    # host-buffer entry point: the carry travels through host memory
    y0, w0 = _sali_case(9)
    yh, wh, sh = y0.copy(), w0.copy(), np.empty((1, 81))
    hrep = chs.HostReport(81, n=4)
    chs.sali_host(HH, None, yh, wh, sh, renorm_every=1, h=0.01, n_steps=100, report=hrep)
    hrep.resume = True
    chs.sali_host(HH, None, yh, wh, sh, renorm_every=1, t0=1.0, h=0.01, n_steps=200, report=hrep)
    yg, wg = dev(y0), dev(w0)
    sg = chs.sali(HH, None, yg, wg, renorm_every=1, h=0.01, n_steps=300)
    assert (sg.cpu().numpy() == sh).all() and (yg.cpu().numpy() == yh).all() and (wg.cpu().numpy() == wh).all()


def test_sali_host_entry(chs):
    y0, w0 = _sali_case(9)
    yh, wh, sh = y0.copy(), w0.copy(), np.empty((1, 81))
    chs.sali_host(HH, None, yh, wh, sh, renorm_every=1, h=0.01, n_steps=300)
    yg, wg = dev(y0), dev(w0)
    sg = chs.sali(HH, None, yg, wg, renorm_every=1, h=0.01, n_steps=300)
    assert (sg.cpu().numpy() == sh).all() and (yg.cpu().numpy() == yh).all() and (wg.cpu().numpy() == wh).all()


def test_sali_coupled3_tile(chs, orc):
    """Same entry point on the 3-DoF system: 4-lane tile per trajectory (orbit, w1, w2, idle)."""
    prm = W.coupled3_params(0.1)
    y0 = W.coupled3_ics(150, seed=1)
    w0 = W.deviation_vectors(150, 2, 6, 7, "unit")
    yo, wo = y0.copy(), w0.copy()
    ro = orc.sali(C3, prm, yo, wo, renorm_every=3, sample_every=100, h=0.01, n_steps=1500, precision="f80")
    yg, wg = dev(y0), dev(w0)
    sg = chs.sali(C3, prm, yg, wg, renorm_every=3, sample_every=100, h=0.01, n_steps=1500).cpu().numpy()
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    assert np.abs(sg / ro["series"] - 1).max() <= TOL_IND
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9


# ---------------------------------------------------------------------------- GALI / Lyapunov, Henon-Heiles
@pytest.mark.parametrize("k", [2, 3, 4])
def test_gali_fixed_hh(chs, orc, k):
    y0 = W.hh_grid(0.125, 13, 11)
    n_ic = y0.shape[1]
    w0 = W.deviation_vectors(n_ic, k, 4, 11, "orthonormal")
    yo, wo = y0.copy(), w0.copy()
    ro = orc.gali(HH, None, yo, wo, renorm_every=5, sample_every=40, h=0.01, n_steps=1000, precision="f80")
    yg, wg = dev(y0), dev(w0)
    gg = chs.gali(HH, None, yg, wg, renorm_every=5, sample_every=40, h=0.01, n_steps=1000).cpu().numpy()
    go = ro["series"]
    assert gg.shape == go.shape
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    big = go > 1e-12
    assert np.abs(gg[big] / go[big] - 1).max() <= TOL_IND
    assert np.abs(gg[~big] - go[~big]).max(initial=0.0) <= 1e-14


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_lyap_fixed_hh(chs, orc, k):
    y0 = W.hh_grid(0.125, 11, 13)
    n_ic = y0.shape[1]
    w0 = W.deviation_vectors(n_ic, k, 4, 12, "raw")   # not orthonormal: entry MGS is exercised
    yo, wo, so = y0.copy(), w0.copy(), np.zeros((k, n_ic))
    ro = orc.lyap(HH, None, yo, wo, renorm_every=10, logsum=so, h=0.01, n_steps=2005, precision="f80")
    yg, wg, sg = dev(y0), dev(w0), dev(np.zeros((k, n_ic)))
    lam = chs.lyap(HH, None, yg, wg, renorm_every=10, logsum=sg, h=0.01, n_steps=2005).cpu().numpy()
    T = 20.05
    den = np.maximum(np.abs(ro["lam"]).max(0), 1.0 / T)
    assert (np.abs(lam - ro["lam"]) / den).max() <= TOL_IND
    assert np.abs(sg.cpu().numpy() - so).max() <= 1e-9
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    # orthonormal on return
    Wm = np.transpose(wg.cpu().numpy(), (2, 0, 1))       # [ic, k, n]
    G = Wm @ np.transpose(Wm, (0, 2, 1))
    assert np.abs(G - np.eye(k)).max() <= 1e-13


# ---------------------------------------------------------------------------- 3-DoF Lyapunov spectrum (C4 shape)
def test_lyap_coupled3_full_spectrum(chs, orc):
    cfg = W.config("C4", n_ic=203)
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    n_ic = y0.shape[1]
    yo, wo = y0.copy(), w0.copy()
    ro = orc.lyap(C3, prm, yo, wo, renorm_every=10, h=0.01, n_steps=3000, precision="f80")
    yg, wg = dev(y0), dev(w0)
    lam = chs.lyap(C3, prm, yg, wg, renorm_every=10, h=0.01, n_steps=3000).cpu().numpy()
    T = 30.0
    den = np.maximum(np.abs(ro["lam"]).max(0), 1.0 / T)
    assert (np.abs(lam - ro["lam"]) / den).max() <= TOL_IND
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    assert np.abs(lam.sum(0)).max() <= 1e-12            # Liouville: sum of exponents = 0


def test_lyap_coupled3_mle_matches_first_exponent(chs):
    cfg = W.config("C4", n_ic=64)
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    lam6 = chs.lyap(C3, prm, dev(y0), dev(w0), renorm_every=10, h=0.01, n_steps=2000).cpu().numpy()
    lam1 = chs.lyap(C3, prm, dev(y0), dev(w0[:1].copy()), renorm_every=10, h=0.01, n_steps=2000).cpu().numpy()
    assert np.abs(lam1[0] - lam6[0]).max() <= 1e-12


# ---------------------------------------------------------------------------- adaptive DOP8(5)
def test_integrate_adaptive_hh(chs, orc):
    y0 = W.hh_grid(1.0 / 6.0, 15, 14)
    n_ic = y0.shape[1]
    yo = y0.copy()
    ro = orc.integrate_adaptive(HH, None, yo, 0.0, 50.0, 1e-12, 1e-12, precision="f80")
    yg = dev(y0)
    rep = chs.Report(n_ic, "cuda")
    chs.integrate_adaptive(HH, None, yg, 0.0, 50.0, 1e-12, 1e-12, report=rep)
    assert (rep.status.cpu().numpy() == 0).all()
    assert (rep.t_final.cpu().numpy() == 50.0).all()
    # both are solutions to tolerance 1e-12 of the same ODE; step sequences may differ by
    # isolated accept/reject flips (R16), so the state tolerance is the solver's own
    # global error level, not round-off
    assert rel_state(yg.cpu().numpy(), yo).max() <= 2e-9
    na, nr = rep.n_accepted.cpu().numpy(), rep.n_rejected.cpu().numpy()
    assert abs(na.sum() / ro["n_accepted"].sum() - 1) <= 5e-3
    assert (np.abs(na - ro["n_accepted"]) <= 2).mean() >= 0.9
    assert abs(int(nr.sum()) - int(ro["n_rejected"].sum())) <= 0.1 * ro["n_rejected"].sum() + 5


def test_sali_adaptive_hh(chs, orc):
    cfg = W.config("C3", n_ic=14 * 14)
    y0, w0 = cfg["y"], cfg["w"]
    n_ic = y0.shape[1]
    yo, wo = y0.copy(), w0.copy()
    ro = orc.sali(HH, None, yo, wo, renorm_every=1, adaptive=True, t_end=60.0, rtol=1e-12, atol=1e-12,
                  precision="f80")
    yg, wg = dev(y0), dev(w0)
    rep = chs.Report(n_ic, "cuda")
    sg = chs.sali(HH, None, yg, wg, renorm_every=1, adaptive=True, t_end=60.0, rtol=1e-12, atol=1e-12,
                  report=rep).cpu().numpy()
    so = ro["series"]
    assert (rep.status.cpu().numpy() == 0).all()
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-8
    reg = so[0] > 1e-4
    assert reg.sum() > 0.5 * n_ic
    assert np.abs(sg[0][reg] / so[0][reg] - 1).max() <= 1e-6
    assert abs(rep.n_accepted.cpu().numpy().sum() / ro["n_accepted"].sum() - 1) <= 5e-3


def test_adaptive_max_steps_and_backward(chs, orc):
    y0 = W.hh_grid(0.125, 6, 6)
    yg = dev(y0)
    rep = chs.Report(36, "cuda")
    chs.integrate_adaptive(HH, None, yg, 0.0, 100.0, 1e-10, 1e-10, max_steps=20, report=rep)
    assert (rep.status.cpu().numpy() == chs.ST_MAXSTEPS).all() and np.isnan(yg.cpu().numpy()).all()
    # backward in time (t_end < t0) against the oracle
    yo = y0.copy()
    orc.integrate_adaptive(HH, None, yo, 0.0, -20.0, 1e-11, 1e-11, precision="f80")
    yg = dev(y0)
    chs.integrate_adaptive(HH, None, yg, 0.0, -20.0, 1e-11, 1e-11)
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-8


# ---------------------------------------------------------------------------- FPUT chain (chain layout)
def test_integrate_fixed_fput(chs, orc):
    prm = W.fput_params(8, 1.0, 0.0, 1.0)
    y0 = W.fput_ics(77, 8, seed=2)
    yo = y0.copy()
    orc.integrate_fixed(FPUT, prm, yo, 0.0, 0.05, 2000, precision="f80")
    yg = dev(y0)
    chs.integrate_fixed(FPUT, prm, yg, 0.0, 0.05, 2000)
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    # alpha != 0 (the FPUT-alpha-beta force of Eq.(7)) and negative step
    prm2 = W.fput_params(8, 0.7, 0.25, 0.5)
    yo = y0.copy()
    orc.integrate_fixed(FPUT, prm2, yo, 0.0, -0.05, 1000, precision="f80")
    yg = dev(y0)
    chs.integrate_fixed(FPUT, prm2, yg, 0.0, -0.05, 1000)
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE


@pytest.mark.parametrize("k", [2, 3, 4])
def test_gali_fixed_fput(chs, orc, k):
    cfg = W.config("C5", n_ic=101)
    y0, prm = cfg["y"], cfg["params"]
    w0 = np.ascontiguousarray(cfg["w"][:k])
    yo, wo, lo = y0.copy(), w0.copy(), np.zeros((k, 101))
    ro = orc.gali(FPUT, prm, yo, wo, renorm_every=10, sample_every=25, lognorm=lo, h=0.05, n_steps=2003,
                  precision="f80")
    yg, wg, lg = dev(y0), dev(w0), dev(np.zeros((k, 101)))
    gg = chs.gali(FPUT, prm, yg, wg, renorm_every=10, sample_every=25, lognorm=lg, h=0.05, n_steps=2003)
    gg, go = gg.cpu().numpy(), ro["series"]
    assert gg.shape == go.shape
    assert go.min() > 1e-6 and np.abs(gg / go - 1).max() <= TOL_IND
    assert rel_state(yg.cpu().numpy(), yo).max() <= TOL_STATE
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    assert np.abs(lg.cpu().numpy() - lo).max() <= 1e-9


def test_gali_small_values_fput(chs, orc):
    """Nearly dependent vectors: GALI ~ 1e-9 must come out of the SVD with full relative accuracy."""
    cfg = W.config("C5", n_ic=40)
    y0, prm = cfg["y"], cfg["params"]
    w0 = cfg["w"].copy()
    w0[3] = w0[0] + 1e-9 * w0[3]
    w0[3] /= np.linalg.norm(w0[3], axis=0)
    go = orc.gali(FPUT, prm, y0.copy(), w0.copy(), renorm_every=1, h=0.05, n_steps=0, precision="f80")["series"]
    gg = chs.gali(FPUT, prm, dev(y0), dev(w0), renorm_every=1, h=0.05, n_steps=0).cpu().numpy()
    assert go.max() < 1e-8 and np.abs(gg / go - 1).max() <= 1e-6


def test_lyap_and_sali_fput(chs, orc):
    cfg = W.config("C5", n_ic=50)
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    yo, wo = y0.copy(), w0.copy()
    ro = orc.lyap(FPUT, prm, yo, wo, renorm_every=10, h=0.05, n_steps=1500, precision="f80")
    yg, wg = dev(y0), dev(w0)
    lam = chs.lyap(FPUT, prm, yg, wg, renorm_every=10, h=0.05, n_steps=1500).cpu().numpy()
    den = np.maximum(np.abs(ro["lam"]).max(0), 1.0 / 75.0)
    assert (np.abs(lam - ro["lam"]) / den).max() <= TOL_IND
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    w2 = np.ascontiguousarray(w0[:2])
    so = orc.sali(FPUT, prm, y0.copy(), w2.copy(), renorm_every=10, h=0.05, n_steps=1500, precision="f80")["series"]
    sg = chs.sali(FPUT, prm, dev(y0), dev(w2), renorm_every=10, h=0.05, n_steps=1500).cpu().numpy()
    assert np.abs(sg / so - 1).max() <= TOL_IND


def test_gali_adaptive_fput(chs, orc):
    """PAPER.md:129 (Fig. 3 workload shape): FPUT + GALI_4 with the adaptive solver, atol = 1e-8."""
    cfg = W.config("C5", n_ic=60)
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    yo, wo = y0.copy(), w0.copy()
    ro = orc.gali(FPUT, prm, yo, wo, renorm_every=1, adaptive=True, t_end=50.0, rtol=1e-8, atol=1e-8, precision="f80")
    yg, wg = dev(y0), dev(w0)
    rep = chs.Report(60, "cuda")
    gg = chs.gali(FPUT, prm, yg, wg, renorm_every=1, adaptive=True, t_end=50.0, rtol=1e-8, atol=1e-8,
                  report=rep).cpu().numpy()
    assert (rep.status.cpu().numpy() == 0).all()
    assert np.abs(gg / ro["series"] - 1).max() <= 1e-4          # both solve to tolerance 1e-8
    assert abs(rep.n_accepted.cpu().numpy().sum() / ro["n_accepted"].sum() - 1) <= 1e-2


def test_adaptive_escaping_orbit_status(chs):
    """An escaping Henon-Heiles orbit blows up in finite time: the adaptive solver must flag it
    (non-finite state or step-size underflow), return NaN for it, and leave its neighbours alone."""
    y0 = W.hh_grid(0.125, 5, 5)
    y0[:, 7] = [0.0, 3.0, 0.0, 5.0]
    yg = dev(y0)
    rep = chs.Report(25, "cuda")
    chs.integrate_adaptive(HH, None, yg, 0.0, 200.0, 1e-10, 1e-10, max_steps=200000, report=rep)
    st = rep.status.cpu().numpy()
    out = yg.cpu().numpy()
    assert st[7] in (chs.ST_NONFINITE, chs.ST_UNDERFLOW) and np.isnan(out[:, 7]).all()
    ok = np.delete(np.arange(25), 7)
    assert (st[ok] == 0).all() and np.isfinite(out[:, ok]).all()
    assert (rep.t_final.cpu().numpy()[ok] == 200.0).all()


def test_adaptive_lane_refill_is_result_neutral(chs):
    """Lane refill (persistent tiles + device work queue) changes which lane runs a trajectory,
    never its arithmetic: outputs are bit-identical with the option on and off, on a deliberately
    unequal ensemble (E = 1/6 orbits interleaved with E = 0.01 orbits that need far fewer steps)
    for the thread layout and for a tile layout."""
    import torch
    ya, yb = W.hh_grid(1.0 / 6.0, 40, 25), W.hh_grid(0.01, 40, 25)
    y0 = np.empty((4, 2000))
    y0[:, 0::2], y0[:, 1::2] = ya, yb
    w0 = W.deviation_vectors(2000, 2, 4, 0, "unit")
    cfg = W.config("C5", n_ic=300)
    outs = {}
    try:
        for mode in (0, 1):
            chs.set_option("adaptive_refill", mode)
            yg, wg, rep = dev(y0), dev(w0), chs.Report(2000, "cuda")
            s = chs.sali(HH, None, yg, wg, renorm_every=1, adaptive=True, t_end=150.0, rtol=1e-11, atol=1e-11, report=rep)
            fy, fw = dev(cfg["y"]), dev(cfg["w"])
            g = chs.gali(FPUT, cfg["params"], fy, fw, renorm_every=2, adaptive=True, t_end=40.0, rtol=1e-8, atol=1e-8)
            outs[mode] = [t.clone() for t in (s, yg, wg, rep.n_accepted, rep.n_rejected, rep.t_final, g, fy, fw)]
    finally:
        chs.set_option("adaptive_refill", 1)
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a, b)
    acc = outs[1][3].cpu().numpy()
    assert acc.max() > 1.3 * acc.min()      # the ensemble really is unequal
    with pytest.raises(chs.ChaoticusError):
        chs.set_option("no_such_option", 1)
