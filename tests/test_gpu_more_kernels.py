"""GPU parity for the wider kernel set (SURVEY.md section 8f "next" rows): other chain lengths
of the FPUT chain layout (N = 4, 16, 32; a full warp per trajectory at N = 32), the LD on the
chain layout, adaptive Lyapunov / GALI, and the remaining k of the 3-DoF system."""
import numpy as np
import pytest

from paper_2507_00622_b200 import workloads as W

pytestmark = pytest.mark.gpu
HH, C3, FPUT = W.SYS_HENON_HEILES, W.SYS_COUPLED3, W.SYS_FPUT


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


def rel_state(a, b):
    return np.linalg.norm(a - b, axis=0) / np.linalg.norm(b, axis=0)


def lam_err(lam, ref, T):
    return (np.abs(lam - ref) / np.maximum(np.abs(ref).max(0), 1.0 / T)).max()


# chain lengths by tile class (fput_launch.h): exact in-warp tiles 4, 16, 32, 64; padded tiles 3, 5, 12, 24,
# 48 (particles pinned at zero act as the wall); wide tiles (one block per trajectory) 100, 128, 200
@pytest.mark.parametrize("N", [3, 4, 5, 12, 16, 24, 32, 48, 64, 100, 128, 200])
def test_fput_other_lengths(chs, orc, N):
    n_ic = 45 if N <= 32 else (21 if N <= 64 else 7)   # ragged: a few tiles of the last block are padding
    steps = 1000 if N <= 64 else 400
    prm = W.fput_params(N, 1.0, 0.1, 0.8)
    y0 = W.fput_ics(n_ic, N, seed=3 + N, E=0.1 * N)
    w0 = W.deviation_vectors(n_ic, 4, 2 * N, 50 + N, "orthonormal")
    info = chs.kernel_info(FPUT, prm, chs.WHAT_GALI, k=4, n_ic=n_ic)
    assert info["spill_bytes"] == 0
    # plain integration
    yo = y0.copy()
    orc.integrate_fixed(FPUT, prm, yo, 0.0, 0.05, steps, precision="f80")
    yg = dev(y0)
    chs.integrate_fixed(FPUT, prm, yg, 0.0, 0.05, steps)
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-10
    # GALI_4, fixed step
    yo, wo = y0.copy(), w0.copy()
    go = orc.gali(FPUT, prm, yo, wo, renorm_every=10, sample_every=10, h=0.05, n_steps=steps, precision="f80")["series"]
    yg, wg = dev(y0), dev(w0)
    gg = chs.gali(FPUT, prm, yg, wg, renorm_every=10, sample_every=10, h=0.05, n_steps=steps).cpu().numpy()
    assert go.min() > 1e-9 and np.abs(gg / go - 1).max() <= 1e-8
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-10
    # Lyapunov k = 4 and SALI
    yo, wo = y0.copy(), w0.copy()
    lo = orc.lyap(FPUT, prm, yo, wo, renorm_every=10, h=0.05, n_steps=steps, precision="f80")["lam"]
    lg = chs.lyap(FPUT, prm, dev(y0), dev(w0), renorm_every=10, h=0.05, n_steps=steps).cpu().numpy()
    assert lam_err(lg, lo, 0.05 * steps) <= 1e-8
    w2 = np.ascontiguousarray(w0[:2])
    so = orc.sali(FPUT, prm, y0.copy(), w2.copy(), renorm_every=5, h=0.05, n_steps=600, precision="f80")["series"]
    sg = chs.sali(FPUT, prm, dev(y0), dev(w2), renorm_every=5, h=0.05, n_steps=600).cpu().numpy()
    assert np.abs(sg / so - 1).max() <= 1e-8
    # LD on the chain layout (tile-wide norm by shuffles), both directions
    fo, bo = orc.ld(FPUT, prm, y0, 0.0, 0.05, 400, precision="f80")
    f, b = chs.ld(FPUT, prm, dev(y0), 0.0, 0.05, 400)
    assert np.abs(f.cpu().numpy() / fo - 1).max() <= 1e-8 and np.abs(b.cpu().numpy() / bo - 1).max() <= 1e-8
    # adaptive integration and adaptive GALI_4 (the paper's Fig. 3 solver, atol = 1e-8: PAPER.md:129)
    yo = y0.copy()
    ro = orc.integrate_adaptive(FPUT, prm, yo, 0.0, 20.0, 1e-10, 1e-10, precision="f80")
    yg, rep = dev(y0), chs.Report(n_ic, "cuda")
    chs.integrate_adaptive(FPUT, prm, yg, 0.0, 20.0, 1e-10, 1e-10, report=rep)
    assert (rep.status.cpu().numpy() == 0).all() and rel_state(yg.cpu().numpy(), yo).max() <= 1e-7
    assert abs(rep.n_accepted.cpu().numpy().sum() / ro["n_accepted"].sum() - 1) <= 2e-2
    yo, wo = y0.copy(), w0.copy()
    ro = orc.gali(FPUT, prm, yo, wo, renorm_every=1, adaptive=True, t_end=20.0, rtol=1e-8, atol=1e-8, precision="f80")
    rep = chs.Report(n_ic, "cuda")
    ga = chs.gali(FPUT, prm, dev(y0), dev(w0), renorm_every=1, adaptive=True, t_end=20.0, rtol=1e-8, atol=1e-8,
                  report=rep).cpu().numpy()
    assert (rep.status.cpu().numpy() == 0).all()
    assert np.abs(ga / ro["series"] - 1).max() <= 1e-4
    assert abs(rep.n_accepted.cpu().numpy().sum() / ro["n_accepted"].sum() - 1) <= 2e-2


def test_fput_tile_classes_and_limits(chs):
    """Which tile a chain length runs on (lanes per trajectory), and the longest compiled chain."""
    lanes = lambda N, what, k, ad=False: chs.kernel_info(FPUT, W.fput_params(N), what, k=k, adaptive=ad, n_ic=10)["lanes"]
    assert [lanes(N, chs.WHAT_GALI, 4) for N in (3, 4, 5, 8, 9, 16, 33, 64)] == [2, 2, 4, 4, 8, 8, 32, 32]
    assert [lanes(N, chs.WHAT_GALI, 4, True) for N in (8, 12, 32, 64)] == [8, 16, 32, 64]
    assert [lanes(N, chs.WHAT_LYAP, 4) for N in (8, 40, 65, 128, 129, 256)] == [8, 64, 128, 128, 256, 256]
    with pytest.raises(chs.ChaoticusError):
        lanes(257, chs.WHAT_GALI, 4)


def test_fput8_ld_and_adaptive_set(chs, orc):
    cfg = W.config("C5", n_ic=70)
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    fo, bo = orc.ld(FPUT, prm, y0, 0.0, 0.05, 600, precision="f80")
    f, b = chs.ld(FPUT, prm, dev(y0), 0.0, 0.05, 600)
    assert np.abs(f.cpu().numpy() / fo - 1).max() <= 1e-8 and np.abs(b.cpu().numpy() / bo - 1).max() <= 1e-8
    st = dict(adaptive=True, t_end=30.0, rtol=1e-9, atol=1e-9)
    for k in (1, 4):
        wk = np.ascontiguousarray(w0[:k])
        lo = orc.lyap(FPUT, prm, y0.copy(), wk.copy(), renorm_every=3, precision="f80", **st)["lam"]
        lg = chs.lyap(FPUT, prm, dev(y0), dev(wk), renorm_every=3, **st).cpu().numpy()
        assert lam_err(lg, lo, 30.0) <= 1e-5
    for k in (2, 3):
        wk = np.ascontiguousarray(w0[:k])
        go = orc.gali(FPUT, prm, y0.copy(), wk.copy(), renorm_every=2, precision="f80", **st)["series"]
        gg = chs.gali(FPUT, prm, dev(y0), dev(wk), renorm_every=2, **st).cpu().numpy()
        assert np.abs(gg / go - 1).max() <= 1e-5
    w2 = np.ascontiguousarray(w0[:2])
    so = orc.sali(FPUT, prm, y0.copy(), w2.copy(), renorm_every=2, precision="f80", **st)["series"]
    sg = chs.sali(FPUT, prm, dev(y0), dev(w2), renorm_every=2, **st).cpu().numpy()
    assert np.abs(sg / so - 1).max() <= 1e-5
    yo = y0.copy()
    orc.integrate_adaptive(FPUT, prm, yo, 0.0, 30.0, 1e-11, 1e-11, precision="f80")
    yg = dev(y0)
    chs.integrate_adaptive(FPUT, prm, yg, 0.0, 30.0, 1e-11, 1e-11)
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-8


@pytest.mark.parametrize("k", [3, 4])
def test_hh_adaptive_gali_lyap(chs, orc, k):
    y0 = W.hh_grid(0.125, 9, 11)
    n_ic = y0.shape[1]
    w0 = W.deviation_vectors(n_ic, k, 4, 21, "orthonormal")
    st = dict(adaptive=True, t_end=40.0, rtol=1e-11, atol=1e-11)
    go = orc.gali(HH, None, y0.copy(), w0.copy(), renorm_every=1, precision="f80", **st)["series"]
    gg = chs.gali(HH, None, dev(y0), dev(w0), renorm_every=1, **st).cpu().numpy()
    big = go > 1e-10
    assert np.abs(gg[big] / go[big] - 1).max() <= 1e-5 and np.abs(gg[~big] - go[~big]).max(initial=0) <= 1e-12
    lo = orc.lyap(HH, None, y0.copy(), w0.copy(), renorm_every=2, precision="f80", **st)["lam"]
    lg = chs.lyap(HH, None, dev(y0), dev(w0), renorm_every=2, **st).cpu().numpy()
    assert lam_err(lg, lo, 40.0) <= 1e-6


@pytest.mark.parametrize("k", [1, 2])
def test_hh_adaptive_lyap_thread_layout(chs, orc, k):
    """Adaptive Lyapunov k = 1, 2 on the ONE-THREAD-PER-TRAJECTORY layout, on an unequal ensemble
    (E = 1/6 orbits interleaved with E = 0.01 orbits): a lane's Gram-Schmidt projection must only
    act when that lane renormalises, not whenever a warp-mate does (predicate `apply` of Col::mgs)
    -- against the oracle, and bit-identical with lane refill on and off."""
    import torch
    ya, yb = W.hh_grid(1.0 / 6.0, 20, 10), W.hh_grid(0.01, 20, 10)
    y0 = np.empty((4, 400))
    y0[:, 0::2], y0[:, 1::2] = ya, yb
    w0 = W.deviation_vectors(400, k, 4, 33, "raw")
    assert chs.kernel_info(HH, None, chs.WHAT_LYAP, k=k, adaptive=True, n_ic=400)["lanes"] == 1
    st = dict(adaptive=True, t_end=60.0, rtol=1e-11, atol=1e-11)
    yo, wo = y0.copy(), w0.copy()
    lo = orc.lyap(HH, None, yo, wo, renorm_every=3, precision="f80", **st)["lam"]
    outs = {}
    try:
        for mode in (0, 1):
            chs.set_option("adaptive_refill", mode)
            yg, wg, rep = dev(y0), dev(w0), chs.Report(400, "cuda")
            lg = chs.lyap(HH, None, yg, wg, renorm_every=3, report=rep, **st)
            outs[mode] = [t.clone() for t in (lg, yg, wg, rep.n_accepted, rep.n_rejected)]
    finally:
        chs.set_option("adaptive_refill", 1)
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a, b)
    lg, yg, wg = (t.cpu().numpy() for t in outs[1][:3])
    acc = outs[1][3].cpu().numpy()
    assert acc.max() > 1.3 * acc.min()
    assert lam_err(lg, lo, 60.0) <= 1e-6
    assert rel_state(yg, yo).max() <= 1e-8 and np.abs(wg - wo).max() <= 1e-6


def test_lyap_backward_time(chs, orc):
    """Backward-time runs (h < 0, or t_end < t0): exponents are growth rates per unit of |t|
    (R18), so a chaotic orbit's largest exponent is positive in both time directions."""
    cfg = W.config("C3", n_ic=100)
    y0 = cfg["y"]
    w0 = W.deviation_vectors(100, 2, 4, 5, "orthonormal")
    lo = orc.lyap(HH, None, y0.copy(), w0.copy(), renorm_every=5, h=-0.02, n_steps=4000, precision="f80")["lam"]
    lg = chs.lyap(HH, None, dev(y0), dev(w0), renorm_every=5, h=-0.02, n_steps=4000).cpu().numpy()
    assert lam_err(lg, lo, 80.0) <= 1e-8
    assert lg[0].max() > 0.02 and (lg[0] > -1e-3).all()
    st = dict(adaptive=True, t_end=-40.0, rtol=1e-11, atol=1e-11)
    lo = orc.lyap(HH, None, y0.copy(), w0.copy(), renorm_every=2, precision="f80", **st)["lam"]
    lg = chs.lyap(HH, None, dev(y0), dev(w0), renorm_every=2, **st).cpu().numpy()
    assert lam_err(lg, lo, 40.0) <= 1e-6 and (lg[0] > -1e-3).all()


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_coupled3_lyap_other_k(chs, orc, k):
    cfg = W.config("C4", n_ic=77)
    y0, prm = cfg["y"], cfg["params"]
    w0 = np.ascontiguousarray(cfg["w"][:k])
    yo, wo = y0.copy(), w0.copy()
    lo = orc.lyap(C3, prm, yo, wo, renorm_every=10, h=0.01, n_steps=1500, precision="f80")["lam"]
    yg, wg = dev(y0), dev(w0)
    lg = chs.lyap(C3, prm, yg, wg, renorm_every=10, h=0.01, n_steps=1500).cpu().numpy()
    assert lam_err(lg, lo, 15.0) <= 1e-8
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9 and rel_state(yg.cpu().numpy(), yo).max() <= 1e-10


@pytest.mark.parametrize("k", [2, 3, 4, 5, 6])
def test_coupled3_gali(chs, orc, k):
    cfg = W.config("C4", n_ic=61)
    y0, prm = cfg["y"], cfg["params"]
    w0 = np.ascontiguousarray(cfg["w"][:k])
    go = orc.gali(C3, prm, y0.copy(), w0.copy(), renorm_every=10, sample_every=30, h=0.01, n_steps=1500,
                  precision="f80")["series"]
    lg = dev(np.zeros((k, 61)))
    gg = chs.gali(C3, prm, dev(y0), dev(w0), renorm_every=10, sample_every=30, lognorm=lg, h=0.01,
                  n_steps=1500).cpu().numpy()
    assert gg.shape == go.shape
    assert go.min() > 1e-12 and np.abs(gg / go - 1).max() <= 1e-8
    if k == 6:
        # Liouville: the tangent map has determinant 1, so for 6 initially orthonormal vectors in the
        # 6-dim phase space  GALI_6(t) * prod_v |w_v|(t) = |det| = 1, with prod |w_v| = exp(sum lognorm)
        vol = gg[-1] * np.exp(lg.cpu().numpy().sum(0))
        assert np.abs(vol - 1).max() <= 1e-10


def test_coupled3_adaptive_mle_and_gali2(chs, orc):
    cfg = W.config("C4", n_ic=50)
    y0, prm = cfg["y"], cfg["params"]
    st = dict(adaptive=True, t_end=30.0, rtol=1e-10, atol=1e-10)
    w1 = np.ascontiguousarray(cfg["w"][:1])
    lo = orc.lyap(C3, prm, y0.copy(), w1.copy(), renorm_every=1, precision="f80", **st)["lam"]
    lg = chs.lyap(C3, prm, dev(y0), dev(w1), renorm_every=1, **st).cpu().numpy()
    assert lam_err(lg, lo, 30.0) <= 1e-6
    w2 = np.ascontiguousarray(cfg["w"][:2])
    go = orc.gali(C3, prm, y0.copy(), w2.copy(), renorm_every=1, precision="f80", **st)["series"]
    gg = chs.gali(C3, prm, dev(y0), dev(w2), renorm_every=1, **st).cpu().numpy()
    assert np.abs(gg / go - 1).max() <= 1e-5
    w6 = cfg["w"]
    lo = orc.lyap(C3, prm, y0.copy(), w6.copy(), renorm_every=5, precision="f80", **st)["lam"]
    lg = chs.lyap(C3, prm, dev(y0), dev(w6), renorm_every=5, **st).cpu().numpy()
    assert lam_err(lg, lo, 30.0) <= 1e-6 and np.abs(lg.sum(0)).max() <= 1e-10


def _guarded(torch, shape, fill):
    """A contiguous CUDA tensor of `shape` carved out of a larger allocation with canary words on
    both sides (compute-sanitizer is closed on this pool: bounds are checked with guards instead)."""
    n = int(np.prod(shape))
    pad = 4096
    buf = torch.full((n + 2 * pad,), 7.25e300, dtype=torch.float64, device="cuda")
    view = buf[pad:pad + n].view(*shape)
    view.copy_(torch.from_numpy(np.ascontiguousarray(fill)))
    return buf, view, pad


def _guards_intact(buf, pad):
    return bool((buf[:pad] == 7.25e300).all().item() and (buf[-pad:] == 7.25e300).all().item())


@pytest.mark.parametrize("case", ["hh_thread", "c3_tile", "fput_chain8", "fput_chain32"])
def test_no_out_of_bounds_writes(chs, case):
    import torch
    n_ic = 37      # not a multiple of any tile or block size
    if case == "hh_thread":
        sysid, prm, y0 = HH, None, W.hh_grid(0.125, 37, 1)
        w0 = W.deviation_vectors(n_ic, 2, 4, 1, "unit")
    elif case == "c3_tile":
        sysid, prm, y0 = C3, W.coupled3_params(0.1), W.coupled3_ics(n_ic, seed=1)
        w0 = W.deviation_vectors(n_ic, 6, 6, 2, "orthonormal")
    else:
        N = 8 if case.endswith("8") else 32
        sysid, prm, y0 = FPUT, W.fput_params(N, 1.0, 0.0, 1.0), W.fput_ics(n_ic, N, seed=2, E=0.125 * N)
        w0 = W.deviation_vectors(n_ic, 4, 2 * N, 3, "orthonormal")
    k = w0.shape[0]
    by, y, pad = _guarded(torch, y0.shape, y0)
    bw, w, _ = _guarded(torch, w0.shape, w0)
    bl, lg, _ = _guarded(torch, (k, n_ic), np.zeros((k, n_ic)))
    rep = chs.Report(n_ic, "cuda")
    if case == "c3_tile":
        lam = chs.lyap(sysid, prm, y, w, renorm_every=3, logsum=lg, report=rep, h=0.01, n_steps=50)
        assert torch.isfinite(lam).all().item()
        chs.lyap(sysid, prm, y, w, renorm_every=3, logsum=lg, adaptive=True, t_end=1.0, rtol=1e-9, atol=1e-9)
    elif case == "hh_thread":
        s = chs.sali(sysid, prm, y, w, renorm_every=1, sample_every=7, lognorm=lg, report=rep, h=0.01, n_steps=50)
        assert s.shape == (50 // 7 + 1, n_ic) and torch.isfinite(s).all().item()
        chs.sali(sysid, prm, y, w, renorm_every=1, lognorm=lg, adaptive=True, t_end=1.0, rtol=1e-9, atol=1e-9)
    else:
        g = chs.gali(sysid, prm, y, w, renorm_every=2, sample_every=5, lognorm=lg, report=rep, h=0.05, n_steps=40)
        assert g.shape == (20 // 5 + 1, n_ic) and torch.isfinite(g).all().item()
        chs.gali(sysid, prm, y, w, renorm_every=1, lognorm=lg, adaptive=True, t_end=2.0, rtol=1e-8, atol=1e-8)
    bf, f, _ = _guarded(torch, (n_ic,), np.zeros(n_ic))
    bb, b, _ = _guarded(torch, (n_ic,), np.zeros(n_ic))
    chs.ld(sysid, prm, y, 0.0, 0.01, 20, out_fwd=f, out_bwd=b)
    torch.cuda.synchronize()
    for buf in (by, bw, bl, bf, bb):
        assert _guards_intact(buf, pad)
    assert torch.isfinite(y).all().item() and torch.isfinite(w).all().item() and (f > 0).all().item()


# ---------------------------------------------------------------------------- double pendulum (generic kernel)
DP = W.SYS_DOUBLE_PENDULUM


@pytest.mark.parametrize("prm", [(1.0, 1.0), (0.5, 2.0)])
def test_double_pendulum_fixed(chs, orc, prm):
    """non-separable system through the generic first-order kernel."""
    y0 = W.double_pendulum_ics(333, seed=3)
    yo = y0.copy()
    orc.integrate_fixed(DP, prm, yo, 0.0, 0.01, 1000, precision="f80")
    yg = dev(y0)
    rep = chs.Report(333, "cuda")
    chs.integrate_fixed(DP, prm, yg, 0.0, 0.01, 1000, report=rep)
    assert (rep.status.cpu().numpy() == 0).all()
    # t = 10 is well inside 10 Lyapunov times for these energies
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-10
    # energy conservation on the GPU result (paper's level for Fig. 1: 1e-9)
    # (truncation error of the method itself at h = 0.01: the oracle drifts by the same amount)
    H0, H1 = orc.energy(DP, prm, y0), orc.energy(DP, prm, yg.cpu().numpy())
    Ho = orc.energy(DP, prm, yo)
    assert np.abs(H1 - H0).max() <= 1e-10 and np.abs(H1 - Ho).max() <= 1e-12
    # backward
    yo = y0.copy()
    orc.integrate_fixed(DP, prm, yo, 0.0, -0.01, 500, precision="f80")
    yg = dev(y0)
    chs.integrate_fixed(DP, prm, yg, 0.0, -0.01, 500)
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-10


def test_double_pendulum_adaptive(chs, orc):
    prm = (1.0, 1.0)
    y0 = W.double_pendulum_ics(200, seed=4)
    yo = y0.copy()
    ro = orc.integrate_adaptive(DP, prm, yo, 0.0, 15.0, 1e-11, 1e-11, precision="f80")
    yg = dev(y0)
    rep = chs.Report(200, "cuda")
    chs.integrate_adaptive(DP, prm, yg, 0.0, 15.0, 1e-11, 1e-11, report=rep)
    assert (rep.status.cpu().numpy() == 0).all() and (rep.t_final.cpu().numpy() == 15.0).all()
    lam_guard = rel_state(yg.cpu().numpy(), yo)
    assert np.median(lam_guard) <= 1e-9 and lam_guard.max() <= 1e-6     # chaotic orbits amplify the tolerance
    assert abs(rep.n_accepted.cpu().numpy().sum() / ro["n_accepted"].sum() - 1) <= 5e-3
    H0, H1 = orc.energy(DP, prm, y0), orc.energy(DP, prm, yg.cpu().numpy())
    assert np.abs(H1 - H0).max() <= 1e-9


def test_double_pendulum_unsupported_entry_points(chs):
    import torch
    y = dev(W.double_pendulum_ics(8))
    w = torch.zeros((2, 4, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(chs.ChaoticusError, match="no compiled kernel"):
        chs.gali(DP, (1.0, 1.0), y, w, adaptive=True, t_end=1.0, rtol=1e-9, atol=1e-9)   # adaptive GALI: not compiled
    with pytest.raises(chs.ChaoticusError):
        chs.integrate_fixed(DP, (1.0, -1.0), y, 0.0, 0.01, 10)    # alpha <= 0


def test_double_pendulum_ld(chs, orc):
    """LD of the non-separable system (no variational equations needed)."""
    prm = (0.5, 2.0)
    y0 = W.double_pendulum_ics(301, seed=6)
    fo, bo = orc.ld(DP, prm, y0, 0.0, 0.01, 800, precision="f80")
    f, b = chs.ld(DP, prm, dev(y0), 0.0, 0.01, 800)
    assert np.abs(f.cpu().numpy() / fo - 1).max() <= 1e-8 and np.abs(b.cpu().numpy() / bo - 1).max() <= 1e-8
    assert (fo > 0).all() and np.abs(fo - bo).max() > 1e-3        # the two directions really differ


@pytest.mark.parametrize("n_ic", [1, 3])
def test_tiny_ensembles_on_tile_layouts(chs, orc, n_ic):
    """One or three trajectories: most tiles of the only warp are padding that shadows the last
    trajectory (shuffles must stay convergent) and must not store anything."""
    cfg = W.config("C5", n_ic=n_ic)
    go = orc.gali(FPUT, cfg["params"], cfg["y"].copy(), cfg["w"].copy(), renorm_every=10, h=0.05, n_steps=300,
                  precision="f80")["series"]
    gg = chs.gali(FPUT, cfg["params"], dev(cfg["y"]), dev(cfg["w"]), renorm_every=10, h=0.05, n_steps=300)
    assert np.abs(gg.cpu().numpy() / go - 1).max() <= 1e-8
    cfg = W.config("C4", n_ic=n_ic)
    lo = orc.lyap(C3, cfg["params"], cfg["y"].copy(), cfg["w"].copy(), renorm_every=10, h=0.01, n_steps=300,
                  precision="f80")["lam"]
    lg = chs.lyap(C3, cfg["params"], dev(cfg["y"]), dev(cfg["w"]), renorm_every=10, h=0.01, n_steps=300)
    assert lam_err(lg.cpu().numpy(), lo, 3.0) <= 1e-8
    cfg = W.config("C1", n_ic=1)   # 1 x 1 grid through the 4-lane SALI tile
    so = orc.sali(HH, None, cfg["y"].copy(), cfg["w"].copy(), renorm_every=1, h=0.01, n_steps=300,
                  precision="f80")["series"]
    sg = chs.sali(HH, None, dev(cfg["y"]), dev(cfg["w"]), renorm_every=1, h=0.01, n_steps=300)
    assert np.abs(sg.cpu().numpy() / so - 1).max() <= 1e-8


def test_zero_length_runs(chs, orc):
    """n_steps = 0 and t_end = t0: nothing is integrated; vectors come back (ortho)normalised, the
    indicator is that of the entry vectors, lambda is NaN (no elapsed time), counters are zero."""
    y0 = W.hh_grid(0.125, 5, 4)
    w0 = W.deviation_vectors(20, 2, 4, 9, "raw")
    for kw in (dict(h=0.01, n_steps=0), dict(adaptive=True, t_end=0.0, rtol=1e-9, atol=1e-9)):
        yo, wo = y0.copy(), w0.copy()
        so = orc.sali(HH, None, yo, wo, renorm_every=1, precision="f80", **kw)["series"]
        yg, wg = dev(y0), dev(w0)
        rep = chs.Report(20, "cuda")
        sg = chs.sali(HH, None, yg, wg, renorm_every=1, report=rep, **kw).cpu().numpy()
        assert np.abs(sg / so - 1).max() <= 1e-13
        assert (yg.cpu().numpy() == y0).all() and np.abs(wg.cpu().numpy() - wo).max() <= 1e-15
        assert (rep.n_accepted.cpu().numpy() == 0).all() and (rep.status.cpu().numpy() == 0).all()
        lam = chs.lyap(HH, None, dev(y0), dev(w0), renorm_every=1, **kw).cpu().numpy()
        assert np.isnan(lam).all()


# ---------------------------------------------------------------------------- LD neighbours
@pytest.mark.parametrize("case", ["hh", "coupled3", "fput12", "fput100", "dp"])
def test_ld_neighbours(chs, orc, case):
    """the 2n axis neighbours x0 +- sigma e_i of every IC are generated on the device and
    integrated in the same LD launch as the centres; members' LDs element-wise against the oracle's plain
    loop over displaced ICs, raw differences |M(x0 +- sigma e_i) - M(x0)| to an absolute 1e-9 M."""
    if case == "hh":
        sysid, prm, y0, h, ns, sg = HH, None, W.hh_grid(0.125, 19, 7), 0.01, 1500, 1e-3     # 133 ICs, ragged
    elif case == "coupled3":
        sysid, prm, y0, h, ns, sg = C3, W.coupled3_params(0.1), W.coupled3_ics(70, seed=1), 0.01, 1000, 1e-2
    elif case == "fput12":     # padded in-warp tile: members displace particles of a 12-chain on a 16-slot tile
        sysid, prm, y0, h, ns, sg = FPUT, W.fput_params(12, 1.0, 0.1, 0.8), W.fput_ics(9, 12, seed=5, E=1.2), 0.05, 400, 1e-3
    elif case == "fput100":    # wide tile (one block per member)
        sysid, prm, y0, h, ns, sg = FPUT, W.fput_params(100, 1.0, 0.0, 1.0), W.fput_ics(2, 100, seed=6, E=10.0), 0.05, 200, 1e-3
    else:
        sysid, prm, y0, h, ns, sg = W.SYS_DOUBLE_PENDULUM, (1.0, 1.0), W.double_pendulum_ics(50, seed=3), 0.01, 800, 1e-3
    n, n_ic = y0.shape
    ro = orc.ld_neighbours(sysid, prm, y0, sg, 0.0, h, ns, precision="f80")
    rg = chs.ld_neighbours(sysid, prm, dev(y0), sg, 0.0, h, ns)
    for key in ("fwd", "bwd"):
        g, o = rg[key].cpu().numpy(), ro[key]
        assert g.shape == o.shape == (1 + 2 * n, n_ic)
        assert np.abs(g / o - 1).max() <= 1e-8, key
    for key, ctr in (("diff_fwd", "fwd"), ("diff_bwd", "bwd")):
        g, o = rg[key].cpu().numpy(), ro[key]
        assert g.shape == (2 * n, n_ic) and np.abs(g - o).max() <= 1e-9 * ro[ctr][0].max(), key
        assert o.max() > 0.0
    # the centre row is chaoticus_ld itself, bit for bit; one direction only; no differences
    f, b = chs.ld(sysid, prm, dev(y0), 0.0, h, ns)
    assert (rg["fwd"][0] == f).all().item() and (rg["bwd"][0] == b).all().item()
    r1 = chs.ld_neighbours(sysid, prm, dev(y0), sg, 0.0, h, ns, backward=False, diffs=False)
    assert r1["bwd"] is None and r1["diff_fwd"] is None and (r1["fwd"] == rg["fwd"]).all().item()


def test_ld_neighbours_host_and_errors(chs):
    import torch
    y0 = W.hh_grid(0.125, 6, 5)
    rg = chs.ld_neighbours(HH, None, dev(y0), 2e-3, 0.0, 0.01, 300)
    f, b, df, db = np.empty((9, 30)), np.empty((9, 30)), np.empty((8, 30)), np.empty((8, 30))
    chs.ld_neighbours_host(HH, None, y0, 2e-3, 0.0, 0.01, 300, f, b, df, db)
    assert (rg["fwd"].cpu().numpy() == f).all() and (rg["bwd"].cpu().numpy() == b).all()
    assert (rg["diff_fwd"].cpu().numpy() == df).all() and (rg["diff_bwd"].cpu().numpy() == db).all()
    z = chs.ld_neighbours(HH, None, dev(y0), 0.0, 0.0, 0.01, 300)       # sigma = 0: every member is the centre
    assert (z["fwd"] == z["fwd"][0]).all().item() and (z["diff_fwd"] == 0).all().item()
    with pytest.raises(chs.ChaoticusError):
        chs.ld_neighbours(HH, None, dev(y0), -1.0, 0.0, 0.01, 10)
    e = torch.empty((4, 0), dtype=torch.float64, device="cuda")
    assert chs.ld_neighbours(HH, None, e, 1e-3, 0.0, 0.01, 10)["fwd"].shape == (9, 0)


# ---------------------------------------------------------------------------- double pendulum, variational eqs
def test_double_pendulum_sali_gali_lyap(chs, orc):
    """Solvers 3-6 of PAPER.md:49-52 for the paper's first example system (non-separable, generic form,
    one column per lane): states 1e-10, vectors 1e-9, indicators / exponents 1e-8 against the oracle."""
    DP, prm = W.SYS_DOUBLE_PENDULUM, (1.0, 1.0)
    n_ic = 75                                             # ragged: tiles of 2, 4, 8 lanes
    y0 = W.double_pendulum_ics(n_ic, seed=3, theta_max=1.0, p_max=0.5)
    w4 = W.deviation_vectors(n_ic, 4, 4, 41, "orthonormal")
    w2 = np.ascontiguousarray(w4[:2])
    # SALI, fixed step, sampled
    yo, wo, lo = y0.copy(), w2.copy(), np.zeros((2, n_ic))
    so = orc.sali(DP, prm, yo, wo, renorm_every=3, sample_every=50, lognorm=lo, h=0.01, n_steps=1500, precision="f80")["series"]
    yg, wg, lg = dev(y0), dev(w2), dev(np.zeros((2, n_ic)))
    sg = chs.sali(DP, prm, yg, wg, renorm_every=3, sample_every=50, lognorm=lg, h=0.01, n_steps=1500).cpu().numpy()
    assert sg.shape == so.shape and so.min() > 1e-6
    assert np.abs(sg / so - 1).max() <= 1e-8
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-10
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9 and np.abs(lg.cpu().numpy() - lo).max() <= 1e-9
    # GALI_k
    for k in (2, 3, 4):
        wk = np.ascontiguousarray(w4[:k])
        go = orc.gali(DP, prm, y0.copy(), wk.copy(), renorm_every=5, sample_every=40, h=0.01, n_steps=1000, precision="f80")["series"]
        gg = chs.gali(DP, prm, dev(y0), dev(wk), renorm_every=5, sample_every=40, h=0.01, n_steps=1000).cpu().numpy()
        big = go > 1e-12
        assert np.abs(gg[big] / go[big] - 1).max() <= 1e-8, k
        assert np.abs(gg[~big] - go[~big]).max(initial=0.0) <= 1e-13, k
    # Lyapunov k = 1, 2, 4 (full spectrum: sum = 0)
    for k in (1, 2, 4):
        wk = np.ascontiguousarray(w4[:k])
        yo, wo = y0.copy(), wk.copy()
        ro = orc.lyap(DP, prm, yo, wo, renorm_every=10, h=0.01, n_steps=2005, precision="f80")["lam"]
        yg, wg = dev(y0), dev(wk)
        lam = chs.lyap(DP, prm, yg, wg, renorm_every=10, h=0.01, n_steps=2005).cpu().numpy()
        assert lam_err(lam, ro, 20.05) <= 1e-8, k
        assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
        if k == 4:
            assert np.abs(lam.sum(0)).max() <= 1e-11
    # bit-identical continuation with the carried words
    import torch
    a_y, a_w, b_y, b_w = dev(y0), dev(w2), dev(y0), dev(w2)
    sa = chs.sali(DP, prm, a_y, a_w, renorm_every=5, h=0.01, n_steps=600)
    rep = chs.Report(n_ic, "cuda", n=4)
    chs.sali(DP, prm, b_y, b_w, renorm_every=5, h=0.01, n_steps=250, report=rep)
    rep.resume = True
    sb = chs.sali(DP, prm, b_y, b_w, renorm_every=5, t0=2.5, h=0.01, n_steps=350, report=rep)
    assert torch.equal(a_y, b_y) and torch.equal(a_w, b_w) and torch.equal(sa, sb)


def test_double_pendulum_adaptive_and_classification(chs, orc):
    DP, prm = W.SYS_DOUBLE_PENDULUM, (1.0, 1.0)
    n_ic = 60
    y0 = W.double_pendulum_ics(n_ic, seed=4, theta_max=1.0, p_max=0.5)
    w4 = W.deviation_vectors(n_ic, 4, 4, 43, "orthonormal")
    w2 = np.ascontiguousarray(w4[:2])
    st = dict(adaptive=True, t_end=30.0, rtol=1e-11, atol=1e-11)
    yo, wo = y0.copy(), w2.copy()
    ro = orc.sali(DP, prm, yo, wo, renorm_every=2, precision="f80", **st)
    yg, wg, rep = dev(y0), dev(w2), chs.Report(n_ic, "cuda")
    sg = chs.sali(DP, prm, yg, wg, renorm_every=2, report=rep, **st).cpu().numpy()
    assert (rep.status.cpu().numpy() == 0).all() and (rep.t_final.cpu().numpy() == 30.0).all()
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-8
    reg = ro["series"][0] > 1e-4
    assert reg.sum() > 0.5 * n_ic and np.abs(sg[0][reg] / ro["series"][0][reg] - 1).max() <= 1e-5
    assert abs(rep.n_accepted.cpu().numpy().sum() / ro["n_accepted"].sum() - 1) <= 1e-2
    for k in (1, 4):
        wk = np.ascontiguousarray(w4[:k])
        lo = orc.lyap(DP, prm, y0.copy(), wk.copy(), renorm_every=3, precision="f80", **st)["lam"]
        lg = chs.lyap(DP, prm, dev(y0), dev(wk), renorm_every=3, **st).cpu().numpy()
        assert lam_err(lg, lo, 30.0) <= 1e-5, k
    # regular / chaotic classification over a long horizon on an ensemble that mixes both (energies from
    # libration to tumbling): class agreement with the oracle >= 99.9 % (here: all but none of 400)
    y1 = W.double_pendulum_ics(400, seed=9, theta_max=3.0, p_max=0.5)
    w1 = W.deviation_vectors(400, 2, 4, 45, "unit")
    so = orc.sali(DP, prm, y1.copy(), w1.copy(), renorm_every=1, h=0.01, n_steps=40000, precision="f64")["series"][0]
    sg = chs.sali(DP, prm, dev(y1), dev(w1), renorm_every=1, h=0.01, n_steps=40000).cpu().numpy()[0]
    cls_o, cls_g = so < 1e-8, sg < 1e-8
    assert 0.1 < cls_o.mean() < 0.9
    clear = (so < 1e-12) | (so > 1e-4)            # away from the threshold both sides must agree
    assert (cls_o[clear] == cls_g[clear]).all() and (cls_o == cls_g).mean() >= 0.99
    # the entry points that have no compiled kernel still say so
    with pytest.raises(chs.ChaoticusError):
        chs.gali(DP, prm, dev(y0), dev(w2), renorm_every=1, **st)


# ---------------------------------------------------------------------------- spectra on column blocks
@pytest.mark.parametrize("N,k", [(4, 8), (8, 8), (8, 16), (16, 8)])
def test_fput_spectrum_column_blocks(chs, orc, N, k):
    """Lyapunov spectra with more vectors than one lane holds: column blocks of 4 vectors on
    adjacent sub-tiles, each with its own bit-identical replica of the orbit; Gram-Schmidt across the
    blocks by shuffles.  Full spectra (k = 2N): exponents sum to zero and pair up."""
    n_ic = 37                                            # ragged
    prm = W.fput_params(N, 1.0, 0.1, 0.8)
    y0 = W.fput_ics(n_ic, N, seed=20 + N, E=0.3 * N)
    w0 = W.deviation_vectors(n_ic, k, 2 * N, 70 + N, "raw")      # not orthonormal: the entry MGS is exercised
    info = chs.kernel_info(FPUT, prm, chs.WHAT_LYAP, k=k, n_ic=n_ic)
    assert info["lanes"] == N * k // 4 and info["spill_bytes"] == 0
    yo, wo, so = y0.copy(), w0.copy(), np.zeros((k, n_ic))
    ro = orc.lyap(FPUT, prm, yo, wo, renorm_every=10, logsum=so, h=0.05, n_steps=1203, precision="f80")["lam"]
    yg, wg, sg = dev(y0), dev(w0), dev(np.zeros((k, n_ic)))
    lam = chs.lyap(FPUT, prm, yg, wg, renorm_every=10, logsum=sg, h=0.05, n_steps=1203).cpu().numpy()
    assert lam_err(lam, ro, 0.05 * 1203) <= 1e-8
    assert np.abs(sg.cpu().numpy() - so).max() <= 1e-9
    assert rel_state(yg.cpu().numpy(), yo).max() <= 1e-10
    assert np.abs(wg.cpu().numpy() - wo).max() <= 1e-9
    Wm = np.transpose(wg.cpu().numpy(), (2, 0, 1))       # orthonormal on return
    assert np.abs(Wm @ np.transpose(Wm, (0, 2, 1)) - np.eye(k)).max() <= 1e-13
    if k == 2 * N:
        assert np.abs(lam.sum(0)).max() <= 1e-11         # Liouville
    # the first 4 exponents are those of the k = 4 kernel (same Gram-Schmidt prefix)
    w4 = np.ascontiguousarray(w0[:4])
    lam4 = chs.lyap(FPUT, prm, dev(y0), dev(w4), renorm_every=10, h=0.05, n_steps=1203).cpu().numpy()
    assert np.abs(lam4 - lam[:4]).max() <= 1e-10
    # bit-identical continuation
    import torch
    b_y, b_w = dev(y0), dev(w0)
    rep = chs.Report(n_ic, "cuda", n=2 * N)
    chs.lyap(FPUT, prm, b_y, b_w, renorm_every=10, h=0.05, n_steps=500, report=rep)
    rep.resume = True
    chs.lyap(FPUT, prm, b_y, b_w, renorm_every=10, t0=25.0, h=0.05, n_steps=703, report=rep)
    a_y, a_w = dev(y0), dev(w0)
    chs.lyap(FPUT, prm, a_y, a_w, renorm_every=10, h=0.05, n_steps=1203)
    assert torch.equal(a_y, b_y)


# ------------------------------------------------------------------ adaptive Lagrangian descriptor (R21)
@pytest.mark.parametrize("case", ["hh", "coupled3", "fput8", "fput12_padded", "fput100_wide", "double_pendulum"])
def test_ld_adaptive(chs, orc, case):
    """chaoticus_ld_adaptive (augmented ODE (y, M), M' = |f|, M in the error norm) against the oracle's
    orc_ld_adaptive: two solutions to the same tolerance (R16), so values agree to 1e-8 relative and the
    accepted counts to 0.5 %; ragged ensemble sizes; both directions and each alone."""
    if case == "hh":
        sysid, prm, y0, tau = HH, None, W.hh_grid(1.0 / 6.0, 23, 19), 60.0
    elif case == "coupled3":
        cfg = W.config("C4", n_ic=333)
        sysid, prm, y0, tau = C3, cfg["params"], cfg["y"], 40.0
    elif case == "double_pendulum":          # generic first-order kernel
        sysid, prm, y0, tau = W.SYS_DOUBLE_PENDULUM, (0.5, 2.0), W.double_pendulum_ics(203, seed=11, theta_max=1.0), 25.0
    else:
        N = {"fput8": 8, "fput12_padded": 12, "fput100_wide": 100}[case]
        n_ic = 37 if N == 100 else 301
        sysid, prm, y0, tau = FPUT, W.fput_params(N, 1.0, 0.25, 1.0), W.fput_ics(n_ic, N, 7, 1.0), 15.0
    n_ic = y0.shape[1]
    tol = 1e-11
    ro = orc.ld_adaptive(sysid, prm, y0, 0.5, tau, rtol=tol, atol=tol, precision="f80")
    rep = chs.LdReport(n_ic, "cuda")
    yg = dev(y0)
    f, b = chs.ld_adaptive(sysid, prm, yg, 0.5, tau, rtol=tol, atol=tol, report=rep)
    f, b = f.cpu().numpy(), b.cpu().numpy()
    assert (rep.status.cpu().numpy() == 0).all() and (ro["status"] == 0).all()
    assert np.abs(f / ro["fwd"] - 1).max() <= 1e-8 and np.abs(b / ro["bwd"] - 1).max() <= 1e-8
    na = rep.n_accepted.cpu().numpy()
    assert abs(na.sum() / ro["n_accepted"].sum() - 1) <= 5e-3
    assert (rep.t_final.cpu().numpy() == 0.5 + tau).all()     # backward = forward pass of the reversed momenta
    assert np.array_equal(yg.cpu().numpy(), y0)                # y0 untouched
    # one direction alone gives the same bits, and leaves the other row of the report untouched
    rep1 = chs.LdReport(n_ic, "cuda")
    f1, none = chs.ld_adaptive(sysid, prm, yg, 0.5, tau, rtol=tol, atol=tol, backward=False, report=rep1)
    assert none is None and np.array_equal(f1.cpu().numpy(), f)
    assert (rep1.n_accepted[1] == 0).all() and torch_equal(rep1.n_accepted[0], rep.n_accepted[0])
    none, b1 = chs.ld_adaptive(sysid, prm, yg, 0.5, tau, rtol=tol, atol=tol, forward=False)
    assert none is None and np.array_equal(b1.cpu().numpy(), b)


def torch_equal(a, b):
    import torch
    return torch.equal(a, b)


def test_ld_adaptive_closed_form_status_and_host(chs):
    """Isotropic oscillator: M = tau sqrt(2E) whatever the steps; max_steps exhausted -> status 3 and NaN;
    tau = 0 -> 0; refill on/off bit-identical; host-buffer form equals the device form; error paths."""
    P = np.array([1.0, 1.0, 1.0, 0.0])
    y0 = np.random.default_rng(3).uniform(-0.5, 0.5, size=(6, 517))
    ref = 50.0 * np.sqrt((y0 ** 2).sum(0))
    yg = dev(y0)
    f, b = chs.ld_adaptive(C3, P, yg, 0.0, 50.0, rtol=1e-12, atol=1e-12)
    assert np.abs(f.cpu().numpy() / ref - 1).max() <= 1e-11 and np.abs(b.cpu().numpy() / ref - 1).max() <= 1e-11
    rep = chs.LdReport(517, "cuda")
    f2, b2 = chs.ld_adaptive(C3, P, yg, 0.0, 50.0, rtol=1e-12, atol=1e-12, max_steps=25, report=rep)
    assert (rep.status.cpu().numpy() == 3).all() and np.isnan(f2.cpu().numpy()).all() and np.isnan(b2.cpu().numpy()).all()
    assert ((rep.n_accepted + rep.n_rejected).cpu().numpy() == 25).all()
    f0, b0 = chs.ld_adaptive(C3, P, yg, 1.0, 0.0, rtol=1e-9, atol=1e-9)
    assert (f0 == 0).all().item() and (b0 == 0).all().item()
    try:
        chs.set_option("adaptive_refill", 0)
        f3, b3 = chs.ld_adaptive(C3, P, yg, 0.0, 50.0, rtol=1e-12, atol=1e-12)
    finally:
        chs.set_option("adaptive_refill", 1)
    assert torch_equal(f3, f) and torch_equal(b3, b)
    fh, bh = np.empty(517), np.empty(517)
    chs.ld_adaptive_host(C3, P, y0, 0.0, 50.0, fh, bh, rtol=1e-12, atol=1e-12)
    assert np.array_equal(fh, f.cpu().numpy()) and np.array_equal(bh, b.cpu().numpy())
    # the host form hands the report back too: the NaN entries of a run cut short come with their reason
    hrep = chs.HostLdReport(517)
    chs.ld_adaptive_host(C3, P, y0, 0.0, 50.0, fh, bh, rtol=1e-12, atol=1e-12, max_steps=25, report=hrep)
    assert np.isnan(fh).all() and np.isnan(bh).all() and (hrep.status == 3).all()
    assert np.array_equal(hrep.n_accepted, rep.n_accepted.cpu().numpy())
    assert np.array_equal(hrep.n_rejected, rep.n_rejected.cpu().numpy())
    assert np.array_equal(hrep.t_final, rep.t_final.cpu().numpy())
    with pytest.raises(ValueError):
        chs.ld_adaptive_host(C3, P, y0, 0.0, 50.0, fh, bh, rtol=1e-12, atol=1e-12, report=chs.HostReport(517))
    with pytest.raises(chs.ChaoticusError):
        chs.ld_adaptive(C3, P, yg, 0.0, -1.0, rtol=1e-9, atol=1e-9)          # tau < 0
    with pytest.raises(chs.ChaoticusError):
        chs.ld_adaptive(C3, P, yg, 0.0, 1.0, rtol=0.0, atol=1e-9)
    assert chs.kernel_info(HH, None, chs.WHAT_LD, adaptive=True, n_ic=1000)["spill_bytes"] == 0


def test_adaptive_status_words_match_the_oracle(chs, orc):
    """The controller's corner cases against the oracle on identical inputs (the kernels build 10 ulp(t) from
    integer instructions and take the accept decision without forming err, the oracle uses nextafter and pow):
    step-size underflow at t0 = 1e17 (10 ulp = 160: one rejected attempt, nothing accepted, t unchanged), at
    a negative t0 and backwards in time; max_steps hit at exactly the same attempt; blow-up time of an escaping
    orbit within the solver's resolution."""
    y0 = np.ascontiguousarray(W.hh_grid(0.125, 4, 4)[:, 5:8])
    for t0, t_end in ((1e17, 1e17 + 1e6), (-1e17, -1e17 + 1e6), (1e17, 1e17 - 1e6), (-4.0e16, -4.0e16 - 1e6)):
        yo = y0.copy()
        ro = orc.integrate_adaptive(HH, None, yo, t0, t_end, 1e-9, 1e-9, h0=160.0, precision="f64")
        yg, rep = dev(y0), chs.Report(3, "cuda")
        chs.integrate_adaptive(HH, None, yg, t0, t_end, 1e-9, 1e-9, h0=160.0, report=rep)
        assert (ro["status"] == chs.ST_UNDERFLOW).all()
        assert (rep.status.cpu().numpy() == ro["status"]).all()
        assert (rep.n_accepted.cpu().numpy() == ro["n_accepted"]).all() and (rep.n_rejected.cpu().numpy() == ro["n_rejected"]).all()
        assert (rep.t_final.cpu().numpy() == t0).all() and np.isnan(yg.cpu().numpy()).all()
    # max_steps: same count of attempts on both sides, same status
    y0 = W.hh_grid(0.125, 6, 6)
    yo = y0.copy()
    ro = orc.integrate_adaptive(HH, None, yo, 0.0, 100.0, 1e-10, 1e-10, max_steps=57, precision="f64")
    yg, rep = dev(y0), chs.Report(36, "cuda")
    chs.integrate_adaptive(HH, None, yg, 0.0, 100.0, 1e-10, 1e-10, max_steps=57, report=rep)
    assert (ro["status"] == chs.ST_MAXSTEPS).all() and (rep.status.cpu().numpy() == chs.ST_MAXSTEPS).all()
    assert ((rep.n_accepted + rep.n_rejected).cpu().numpy() == 57).all()
    assert np.abs(rep.t_final.cpu().numpy() - ro["t_final"]).max() <= 1e-6 * ro["t_final"].max()
    # escaping orbit: flagged at the same time
    y0 = W.hh_grid(0.125, 3, 3).copy()
    y0[:, 4] = [0.0, 3.0, 0.0, 5.0]
    yo = y0.copy()
    ro = orc.integrate_adaptive(HH, None, yo, 0.0, 50.0, 1e-10, 1e-10, max_steps=200000, precision="f64")
    yg, rep = dev(y0), chs.Report(9, "cuda")
    chs.integrate_adaptive(HH, None, yg, 0.0, 50.0, 1e-10, 1e-10, max_steps=200000, report=rep)
    st = rep.status.cpu().numpy()
    assert st[4] in (chs.ST_NONFINITE, chs.ST_UNDERFLOW) and ro["status"][4] in (chs.ST_NONFINITE, chs.ST_UNDERFLOW)
    assert abs(rep.t_final.cpu().numpy()[4] - ro["t_final"][4]) < 1e-3
    ok = np.delete(np.arange(9), 4)
    assert (st[ok] == 0).all() and rel_state(yg.cpu().numpy()[:, ok], yo[:, ok]).max() <= 1e-8


def test_adaptive_indicator_time_series_by_continuation(chs, orc):
    """An indicator time series of an ADAPTIVE run (sample_every must be 0 there: accepted times differ per
    trajectory) is taken by continuation: consecutive calls t_j -> t_{j+1} with resume = 1 (no entry
    normalisation; the last step of each call lands on the checkpoint).  Same protocol on the oracle; SALI at
    every checkpoint and the accumulated counts agree, on the tile and on the thread layout."""
    for side in (12, 68):                      # 144 ICs: 4-lane tile; 4624 ICs: one thread per trajectory
        y0 = W.hh_grid(0.125, side, side)
        n_ic = y0.shape[1]
        w0 = W.deviation_vectors(n_ic, 2, 4, 5, "unit")
        if side == 68:                         # oracle on a sample of the large ensemble
            idx = np.random.default_rng(2).choice(n_ic, 96, replace=False)
        else:
            idx = np.arange(n_ic)
        yo, wo = np.ascontiguousarray(y0[:, idx]), np.ascontiguousarray(w0[:, :, idx])
        yg, wg, rep = dev(y0), dev(w0), chs.Report(n_ic, "cuda")
        cps = [0.0, 40.0, 80.0, 120.0, 160.0]
        acc_g, acc_o = np.zeros(n_ic, dtype=np.int64), np.zeros(len(idx), dtype=np.int64)
        for j in range(len(cps) - 1):
            rep.resume = j > 0
            sg = chs.sali(HH, None, yg, wg, renorm_every=1, adaptive=True, t0=cps[j], t_end=cps[j + 1], rtol=1e-11,
                          atol=1e-11, report=rep).cpu().numpy()[0]
            ro = orc.sali(HH, None, yo, wo, renorm_every=1, adaptive=True, t0=cps[j], t_end=cps[j + 1], rtol=1e-11,
                          atol=1e-11, precision="f80")
            so = ro["series"][0]
            acc_g += rep.n_accepted.cpu().numpy()
            acc_o += ro["n_accepted"]
            assert (rep.status.cpu().numpy() == 0).all() and (rep.t_final.cpu().numpy() == cps[j + 1]).all()
            reg = so > 1e-4
            assert reg.sum() > 0.5 * len(idx) and np.abs(sg[idx][reg] / so[reg] - 1).max() <= 1e-6
            assert rel_state(yg.cpu().numpy()[:, idx], yo)[reg].max() <= 1e-8   # (chaotic orbits diverge: R16)
        assert abs(acc_g[idx].sum() / acc_o.sum() - 1) <= 5e-3


def test_adaptive_controller_clipping_matches_the_oracle(chs, orc):
    """The clipping range of the step-size factor (the kernels evaluate 0.9 err^(-1/8) in single precision
    from num^2 and den, the oracle with pow): err = 0 at an equilibrium -> factor 10 every step (same few
    accepted steps, none rejected); a hopeless first step h0 = 50 -> rejections with the factor clipped at
    0.2 until the step fits (same number of rejections); a tiny h0 -> growth by the cap 10 per step."""
    y0 = W.hh_grid(0.125, 5, 5)
    y0[:, 3] = 0.0                                   # the equilibrium at the origin: f = 0, err = 0
    for h0, t_end in ((0.0, 300.0), (50.0, 300.0), (1e-9, 5.0)):
        yo = y0.copy()
        ro = orc.integrate_adaptive(HH, None, yo, 0.0, t_end, 1e-10, 1e-10, h0=h0, precision="f64")
        yg, rep = dev(y0), chs.Report(25, "cuda")
        chs.integrate_adaptive(HH, None, yg, 0.0, t_end, 1e-10, 1e-10, h0=h0, report=rep)
        na, nr = rep.n_accepted.cpu().numpy(), rep.n_rejected.cpu().numpy()
        assert (rep.status.cpu().numpy() == 0).all() and (ro["status"] == 0).all()
        assert na[3] == ro["n_accepted"][3] and nr[3] == ro["n_rejected"][3] == 0 and na[3] <= 12
        assert (yg.cpu().numpy()[:, 3] == 0).all()
        assert (np.abs(na - ro["n_accepted"]) <= 2).all()
        if h0 == 50.0:                               # 50 -> 10 -> 2 -> 0.4 -> (0.08): at least three clipped rejections
            assert (nr >= 3)[np.arange(25) != 3].all() and (np.abs(nr - ro["n_rejected"]) <= 1).all()
        if h0 == 1e-9:                               # growth is capped at 10x per accepted step
            assert (na >= 8)[np.arange(25) != 3].all()
            ok = np.arange(25) != 3              # (states only here: at t = 300 chaotic orbits have diverged, R16)
            assert rel_state(yg.cpu().numpy()[:, ok], yo[:, ok]).max() <= 1e-8


def test_adaptive_calls_in_flight_on_many_streams(chs):
    """More adaptive calls in flight than the library has work counters (64 per device): every call owns its
    counter until its kernel has finished, and a call that finds none free runs without lane refill -- same
    results either way.  96 calls on 96 streams, enqueued back to back, all equal to the single-call result."""
    import torch
    y0 = W.hh_grid(1.0 / 6.0, 30, 20)
    w0 = W.deviation_vectors(600, 2, 4, 3, "unit")
    yr, wr = dev(y0), dev(w0)
    ref = chs.sali(HH, None, yr, wr, renorm_every=1, adaptive=True, t_end=120.0, rtol=1e-11, atol=1e-11)
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream() for _ in range(96)]
    ys = [dev(y0) for _ in streams]
    ws = [dev(w0) for _ in streams]
    torch.cuda.synchronize()
    outs = []
    for st, yg, wg in zip(streams, ys, ws):
        with torch.cuda.stream(st):
            outs.append(chs.sali(HH, None, yg, wg, renorm_every=1, adaptive=True, t_end=120.0, rtol=1e-11, atol=1e-11))
    torch.cuda.synchronize()
    for o, yg, wg in zip(outs, ys, ws):
        assert torch.equal(o, ref) and torch.equal(yg, yr) and torch.equal(wg, wr)


# ---------------------------------------------------------------------------- host-buffer forms: carry, pool
def test_host_adaptive_run_returns_a_clean_carry(chs):
    """The *_host forms stage rep->carry in device scratch that comes from a pool (recycled memory).  Adaptive
    runs of the separable systems carry no rounding words and never write that array, so a fresh run must hand
    back zeros -- not whatever the pool block held -- or a later fixed-step continuation with resume = 1 would
    add garbage to the orbit.  With resume = 1 the words that went in come back unchanged."""
    n_ic = 300
    y0 = np.ascontiguousarray(W.hh_grid(0.125, 20, 15))
    w0 = W.deviation_vectors(n_ic, 2, 4, 7, "orthonormal")
    # 1. dirty the pool: a fixed-step host run whose carry block is full of non-zero words, then freed
    y, w, out, rep = y0.copy(), w0.copy(), np.empty((1, n_ic)), chs.HostReport(n_ic, n=4)
    chs.sali_host(HH, None, y, w, out, renorm_every=5, h=0.01, n_steps=200, report=rep)
    assert np.abs(rep.carry).max() > 0.0
    # 2. fresh adaptive runs with a carry array full of junk on the host side
    for fn in ("integrate", "sali"):
        y, w, rep = y0.copy(), w0.copy(), chs.HostReport(n_ic, n=4)
        rep.carry[:] = 123.0
        if fn == "integrate":
            chs.integrate_host(HH, None, y, report=rep, adaptive=True, t0=0.0, t_end=5.0, rtol=1e-10, atol=1e-10)
        else:
            chs.sali_host(HH, None, y, w, out, renorm_every=5, report=rep, adaptive=True, t0=0.0, t_end=5.0,
                          rtol=1e-10, atol=1e-10)
        assert (rep.status == 0).all() and (rep.carry == 0.0).all(), fn
        # ... so that a fixed-step continuation from it is the fixed-step run from the same state, bit for bit
        ya, yb = y.copy(), y.copy()
        rep.resume = True
        chs.integrate_host(HH, None, ya, report=rep, h=0.01, n_steps=100)
        chs.integrate_host(HH, None, yb, h=0.01, n_steps=100)
        assert np.array_equal(ya, yb), fn
    # 3. resume = 1 on an adaptive run: the words pass through untouched
    y, w, rep = y0.copy(), w0.copy(), chs.HostReport(n_ic, n=4)
    rep.carry[:] = np.random.default_rng(1).normal(size=rep.carry.shape) * 1e-17
    keep = rep.carry.copy()
    rep.resume = True
    chs.sali_host(HH, None, y, w, out, renorm_every=5, report=rep, adaptive=True, t0=0.0, t_end=2.0, rtol=1e-10, atol=1e-10)
    assert np.array_equal(rep.carry, keep)


def test_host_forms_use_their_own_memory_pool(chs):
    """The scratch of the *_host forms comes from a pool the library owns: the release threshold of the device's
    DEFAULT pool (which torch's cudaMallocAsync backend or other libraries may use) stays what it was, and
    set_option("host_pool_trim", 0) gives the memory the library's pool kept back to the driver."""
    import ctypes
    import torch
    rt = ctypes.CDLL("libcudart.so.12")
    def default_threshold():
        pool, val = ctypes.c_void_p(), ctypes.c_uint64(12345)
        assert rt.cudaDeviceGetDefaultMemPool(ctypes.byref(pool), torch.cuda.current_device()) == 0
        assert rt.cudaMemPoolGetAttribute(pool, 4, ctypes.byref(val)) == 0      # cudaMemPoolAttrReleaseThreshold = 4
        return val.value
    before = default_threshold()
    n_ic = 1 << 20                                           # 32 MiB of states + 16 MiB of outputs
    y0 = np.ascontiguousarray(np.tile(W.hh_grid(0.125, 4, 4)[:, 5:6], (1, n_ic)))
    f, b = np.empty(n_ic), np.empty(n_ic)
    chs.ld_host(HH, None, y0, 0.0, 0.01, 2, f, b)
    assert default_threshold() == before
    torch.cuda.synchronize()
    held = torch.cuda.mem_get_info()[0]
    chs.set_option("host_pool_trim", 0)
    freed = torch.cuda.mem_get_info()[0] - held
    assert freed >= 40 * 2 ** 20, freed                      # the 48 MiB the call used went back
    f2, b2 = np.empty(n_ic), np.empty(n_ic)
    chs.ld_host(HH, None, y0, 0.0, 0.01, 2, f2, b2)          # and the pool refills on the next call
    assert np.array_equal(f, f2) and np.array_equal(b, b2)
    with pytest.raises(chs.ChaoticusError):
        chs.set_option("host_pool_trim", -1)
