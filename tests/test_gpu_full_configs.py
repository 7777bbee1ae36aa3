"""The five BASELINE.json configurations at FULL size, in the launch configuration bench.py
times, against the oracle (x86 long double) on sampled trajectories -- DESIGN.md "Parity
protocol":

  * states: per trajectory |dy|_2/|y|_2 <= 1e-10 at every checkpoint with t <= 10 T_L,
    T_L = 1/max(lambda1_hat, 10/T), lambda1_hat the oracle's finite-time mLE at the end;
  * indicators on regular orbits (oracle value >= 1e-4 at the end): relative 1e-8;
  * classification (chaotic iff indicator < 1e-8) over the full horizon: >= 99.9 % agreement;
  * never a log or a relative error of a value that may be 0.
Samples are drawn over the WHOLE index range (random + block/warp/tile boundary trajectories).
"""
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


def test_C1_full(chs, orc):
    """configs[0]: all 1024 ICs, 10^4 steps, SALI renormalised every step; 10 checkpoints."""
    cfg = W.config("C1")
    y0, w0 = cfg["y"], cfg["w"]
    n_ic, T, chunks = 1024, 100.0, 10
    yo, wo, lo = y0.copy(), w0.copy(), np.zeros((2, n_ic))
    yg, wg = dev(y0), dev(w0)
    ck = []
    for c in range(chunks):
        ro = orc.sali(HH, None, yo, wo, renorm_every=1, lognorm=lo, t0=c * T / chunks, h=0.01, n_steps=1000,
                      precision="f80")
        sg = chs.sali(HH, None, yg, wg, renorm_every=1, t0=c * T / chunks, h=0.01, n_steps=1000)
        ck.append(((c + 1) * T / chunks, rel_state(yg.cpu().numpy(), yo), sg.cpu().numpy()[0], ro["series"][0]))
    lam1 = lo[0] / T
    TL = 1.0 / np.maximum(lam1, 10.0 / T)
    regular = ck[-1][3] >= 1e-4
    assert regular.sum() > 0.5 * n_ic
    for t, err, sg, so in ck:
        inside = t <= 10 * TL
        assert inside.any() and err[inside].max() <= 1e-10, (t, err[inside].max())
        assert np.abs(sg[regular] / so[regular] - 1).max() <= 1e-8, t
    assert ((ck[-1][2] < 1e-8) == (ck[-1][3] < 1e-8)).mean() >= 0.999


def test_C2_full(chs, orc):
    """configs[1]: 1024 x 1024 grid, 5000 steps forward + backward; 512 sampled ICs vs the oracle;
    the mirror symmetry M-(y, py) = M+(y, -py) on the whole grid."""
    cfg = W.config("C2")
    y0 = cfg["y"]
    f, b = chs.ld(HH, None, dev(y0), 0.0, 0.01, 5000)
    f, b = f.cpu().numpy(), b.cpu().numpy()
    assert np.isfinite(f).all() and np.isfinite(b).all()
    idx = np.random.default_rng(0).choice(y0.shape[1], 512, replace=False)
    fo, bo = orc.ld(HH, None, np.ascontiguousarray(y0[:, idx]), 0.0, 0.01, 5000, precision="f80")
    assert np.abs(f[idx] / fo - 1).max() <= 1e-8 and np.abs(b[idx] / bo - 1).max() <= 1e-8
    F, B = f.reshape(1024, 1024), b.reshape(1024, 1024)
    assert np.abs(B - F[:, ::-1]).max() <= 1e-12
    # the LD is an arc length: bounded by tau * max|f| on the energy surface and > 0
    assert f.min() > 10.0 and f.max() < 50.0


def test_C3_full(chs, orc):
    """configs[2]: 512 x 512 grid, adaptive 1e-12, t = 1000, SALI; 2048 sampled ICs."""
    cfg = W.config("C3")
    y0, w0 = cfg["y"], cfg["w"]
    n = y0.shape[1]
    yg, wg = dev(y0), dev(w0)
    rep = chs.Report(n, "cuda")
    sg = chs.sali(HH, None, yg, wg, renorm_every=1, adaptive=True, t_end=1000.0, rtol=1e-12, atol=1e-12,
                  report=rep).cpu().numpy()[0]
    assert (rep.status.cpu().numpy() == 0).all() and (rep.t_final.cpu().numpy() == 1000.0).all()
    na, nr = rep.n_accepted.cpu().numpy(), rep.n_rejected.cpu().numpy()
    idx = np.random.default_rng(1).choice(n, 2048, replace=False)
    yo, wo = np.ascontiguousarray(y0[:, idx]), np.ascontiguousarray(w0[:, :, idx])
    ro = orc.sali(HH, None, yo, wo, renorm_every=1, adaptive=True, t_end=1000.0, rtol=1e-12, atol=1e-12,
                  precision="f80")
    so = ro["series"][0]
    agree = ((sg[idx] < 1e-8) == (so < 1e-8)).mean()
    print(f"C3: accepted {na.sum()} rejected {nr.sum()} ({100.0 * nr.sum() / (na.sum() + nr.sum()):.2f} %), "
          f"chaotic fraction {np.mean(sg < 1e-8):.4f}, undecided band {(np.mean((sg >= 1e-8) & (sg < 1e-4))):.4f}, "
          f"classification agreement on the sample {agree:.5f}")
    assert agree >= 0.999
    reg = so >= 1e-4
    if reg.any():   # adaptive: both are solutions to tolerance, not the same rounding sequence
        assert np.abs(sg[idx][reg] / so[reg] - 1).max() <= 1e-4
    assert abs(na[idx].sum() / ro["n_accepted"].sum() - 1) <= 5e-3
    # energy conservation on the whole grid (paper's own level: 1e-8)
    from oracle import chaos_oracle
    H = chaos_oracle.energy(HH, None, yg.cpu().numpy())
    assert np.abs(H - 1.0 / 6.0).max() <= 1e-10


def spread_sample(n, n_random, seed):
    """Indices spread over the WHOLE index range: n_random random ones plus the first and last
    trajectory and the trajectories on either side of warp, block and tile boundaries."""
    fixed = [0, 1, 3, 4, 7, 8, 15, 16, 31, 32, 63, 64, 127, 128, 255, 256, n // 2 - 1, n // 2, n - 129, n - 128,
             n - 33, n - 32, n - 2, n - 1]
    rnd = np.random.default_rng(seed).choice(n, n_random, replace=False)
    return np.unique(np.concatenate([np.array(fixed), rnd]))


def test_C4_full(chs, orc):
    """configs[3]: 65536 ICs, 10^5 steps, full Lyapunov spectrum (MGS every 10 steps); 488 random ICs
    + boundary ICs across the whole index range against the long-double oracle."""
    cfg = W.config("C4")
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    yg, wg = dev(y0), dev(w0)
    lam = chs.lyap(C3, prm, yg, wg, renorm_every=10, h=0.01, n_steps=100000).cpu().numpy()
    idx = spread_sample(y0.shape[1], 488, 4)
    assert idx.min() == 0 and idx.max() == 65535 and len(idx) >= 480
    yo, wo = np.ascontiguousarray(y0[:, idx]), np.ascontiguousarray(w0[:, :, idx])
    ro = orc.lyap(C3, prm, yo, wo, renorm_every=10, h=0.01, n_steps=100000, precision="f80")
    T = 1000.0
    den = np.maximum(np.abs(ro["lam"]).max(0), 1.0 / T)
    assert (np.abs(lam[:, idx] - ro["lam"]) / den).max() <= 1e-8
    # States are compared to 1e-10 where round-off is not amplified beyond it, lambda_1 T <= 10.  WHICH sampled
    # trajectories that leaves out is decided twice, from the oracle's lambda_1 and from the GPU's own, and the
    # two sets must be the same (a trajectory within 1e-6 of the threshold may fall either way); no flat quota.
    lam1, lam1_g = ro["lam"][0], lam[0, idx]
    inside = T <= 10.0 / np.maximum(lam1, 10.0 / T)
    inside_g = T <= 10.0 / np.maximum(lam1_g, 10.0 / T)
    clear = np.abs(lam1 - 10.0 / T) > 1e-6
    assert (inside == inside_g)[clear].all() and inside.any()
    ys = yg.cpu().numpy()[:, idx]
    assert np.isfinite(ys).all() and np.isfinite(yo).all()          # nobody escaped or blew up on either side
    assert rel_state(ys, yo)[inside].max() <= 1e-10
    # the left-out (chaotic) ones still follow the oracle as far as e^{lambda_1 T} allows
    if (~inside).any():
        assert (rel_state(ys, yo)[~inside] <= 1e-8 * np.exp(lam1[~inside] * T - 10.0)).all()
    # properties at any size: Liouville (sum = 0), pairing, two vanishing exponents
    assert np.abs(lam.sum(0)).max() <= 1e-12
    assert np.abs(lam + lam[::-1]).max() <= 2e-3
    assert np.isfinite(lam).all()


def test_C5_full(chs, orc):
    """configs[4]: 65536 ICs, FPUT-beta N = 8, GALI_4, 2 x 10^4 steps of h = 0.05; 1000 random ICs
    + boundary ICs across the whole index range against the long-double oracle."""
    cfg = W.config("C5")
    y0, w0, prm = cfg["y"], cfg["w"], cfg["params"]
    yg, wg, lg = dev(y0), dev(w0), dev(np.zeros((4, y0.shape[1])))
    g = chs.gali(FPUT, prm, yg, wg, renorm_every=10, lognorm=lg, h=0.05, n_steps=20000).cpu().numpy()[0]
    idx = spread_sample(y0.shape[1], 1000, 5)
    ns = len(idx)
    assert idx.min() == 0 and idx.max() == 65535 and ns >= 1000
    yo, wo, lo = np.ascontiguousarray(y0[:, idx]), np.ascontiguousarray(w0[:, :, idx]), np.zeros((4, ns))
    go = orc.gali(FPUT, prm, yo, wo, renorm_every=10, lognorm=lo, h=0.05, n_steps=20000, precision="f80")["series"][0]
    T = 1000.0
    regular = go >= 1e-4
    assert regular.any() and np.abs(g[idx][regular] / go[regular] - 1).max() <= 1e-8
    assert ((g[idx] < 1e-8) == (go < 1e-8)).mean() >= 0.999
    inside = T <= 10.0 / np.maximum(lo[0] / T, 10.0 / T)
    assert inside.any() and rel_state(yg.cpu().numpy()[:, idx], yo)[inside].max() <= 1e-10
    assert np.abs(lg.cpu().numpy()[:, idx][:, inside] - lo[:, inside]).max() <= 1e-7
    from oracle import chaos_oracle
    H = chaos_oracle.energy(FPUT, prm, yg.cpu().numpy())
    assert np.abs(H - 1.0).max() <= 1e-11
    assert (g >= 0).all() and (g <= 1.0 + 1e-12).all()
