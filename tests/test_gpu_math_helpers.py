"""GPU test of the device math helpers the step kernels inline instead of the CUDA library routines
(csrc/dop8_core.cuh fast_sqrt / fast_rsqrt / fast_rcp: MUFU seed + polynomial, no slow-path branch;
csrc/gen_kernels.cuh fast_sincos: three-constant reduction by pi/2 + Taylor polynomials).  The parity
tests bound their END-TO-END effect; this file bounds the helpers themselves, through a test-only entry of
libchaoticus_probe.so (not the product ABI), against the host's 80-bit long double over >= 10^7 seeded
arguments per function, edge values included.  Error unit: the spacing of doubles at the true value."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
N = 10_000_000


@pytest.fixture(scope="module")
def probe():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_00622_b200 import probe
    return probe


def _run(probe, name, x):
    import torch
    r = probe.math_probe(name, torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    return tuple(t.cpu().numpy() for t in r) if isinstance(r, tuple) else r.cpu().numpy()


def _ulp_err(got, ref_ld):
    """|got - ref| in units of the double spacing at |ref| (ref in long double)."""
    ref_d = ref_ld.astype(np.float64)
    sp = np.spacing(np.maximum(np.abs(ref_d), np.finfo(np.float64).tiny))
    return np.abs((got.astype(np.longdouble) - ref_ld) / sp.astype(np.longdouble)).astype(np.float64)


def _positive_arguments(seed):
    rng = np.random.default_rng(seed)
    x = np.empty(N)
    a, b, c = N // 2, N // 4, N // 8
    x[:a] = 10.0 ** rng.uniform(-300.0, 300.0, a)                    # the whole exponent range
    x[a:a + b] = rng.uniform(0.0, 4.0, b)                             # sums of squares of unit-size vectors
    x[a + b:a + b + c] = 2.0 ** rng.integers(-1000, 1000, c)          # exact powers of two
    x[a + b + c:] = np.ldexp(rng.uniform(1.0, 2.0, N - a - b - c), rng.integers(-1021, 1023, N - a - b - c))
    x[-8:] = [1e300, 1e-300, 2.2250738585072014e-308, 1.7976931348623157e308, 1.0, 4.0, 0.25, 3.0]
    return x


def test_fast_sqrt_rsqrt_rcp(probe):
    x = _positive_arguments(1)
    xl = x.astype(np.longdouble)
    e = _ulp_err(_run(probe, "fast_sqrt", x), np.sqrt(xl))
    assert e.max() <= 1.0, ("fast_sqrt", e.max(), x[e.argmax()])
    big = x < 1e300                                                   # 1/sqrt and 1/x of these stay normal numbers
    e = _ulp_err(_run(probe, "fast_rsqrt", x), 1.0 / np.sqrt(xl))[big]
    assert e.max() <= 1.5, ("fast_rsqrt", e.max())
    ok = (x > 1e-300) & (x < 1e300)
    e = _ulp_err(_run(probe, "fast_rcp", x), 1.0 / xl)[ok]
    assert e.max() <= 1.5, ("fast_rcp", e.max())
    # the documented edge values: zero and subnormals (.ftz seed): sqrt -> 0; rsqrt -> inf for a subnormal and
    # NaN for zero itself (0 * inf in the correction step): not finite either way
    z = np.array([0.0, 5e-324, 1e-310, 2.2250738585072009e-308])
    assert (_run(probe, "fast_sqrt", z) == 0.0).all()
    r = _run(probe, "fast_rsqrt", z)
    assert np.isnan(r[0]) and np.isinf(r[1:]).all()
    # exact where the true result is a double and the seed error is a pure rounding matter
    p2 = 2.0 ** np.arange(-600, 601, 2, dtype=np.float64)
    assert (_run(probe, "fast_sqrt", p2) == np.sqrt(p2)).all()
    assert (_run(probe, "fast_rcp", p2) == 1.0 / p2).all()


def test_fast_sincos(probe):
    """|x| up to 1e8 (a pendulum that has rotated 10^7 times).  The reduction r = x - k pi/2 runs in three fused
    multiply-adds against a three-double pi/2; the error is measured in ulps of the true sine / cosine of the
    double x, everywhere -- next to their zeros too (multiples of the double nearest pi/2 are in the sample)."""
    rng = np.random.default_rng(2)
    x = np.empty(N)
    a, b = N // 2, N // 4
    x[:a] = rng.uniform(-1e8, 1e8, a)
    x[a:a + b] = rng.uniform(-10.0, 10.0, b)
    x[a + b:] = np.sign(rng.uniform(-1, 1, N - a - b)) * 10.0 ** rng.uniform(-300.0, 8.0, N - a - b)
    k = np.arange(1, 1001, dtype=np.float64)
    x[-3000:-2000] = k * (np.pi / 2)                                  # next to the zeros of sin / cos
    x[-2000:-1000] = k * 1e5 * (np.pi / 2)
    x[-1000:] = [0.0, -0.0, 1e-300, -1e-300, 1e8, -1e8, np.pi, -np.pi] + [0.5] * 992
    sn, cs = _run(probe, "fast_sincos", x)
    xl = x.astype(np.longdouble)
    rs, rc = np.sin(xl), np.cos(xl)
    for got, ref, name in ((sn, rs, "sin"), (cs, rc, "cos")):
        e = _ulp_err(got, ref)
        assert e.max() <= 2.0, (name, e.max(), x[e.argmax()])        # also next to the zeros, also at |x| = 1e8
        small = np.abs(x) <= 10.0
        assert e[small].max() <= 2.0, (name, e[small].max())         # (1.54 measured: the bound is the polynomial's, not the reduction's)
    assert np.abs(sn * sn + cs * cs - 1.0).max() <= 4.5e-16
    assert sn[-1000] == 0.0 and cs[-1000] == 1.0 and sn[-998] == 1e-300
