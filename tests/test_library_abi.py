"""CPU-side checks of the CUDA path's host pieces (no GPU, no compute calls):
the C-ABI library loads and exports every symbol include/chaoticus.h declares, argument
validation, and the generated separable-form coefficients (csrc/dop8_coeffs.h) against order
conditions written for that form."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2507_00622_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "chaoticus.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(chaoticus_\w+)\s*\(", hdr)))
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in chaoticus.h but not exported"
    from paper_2507_00622_b200 import binding
    assert sorted(binding.EXPORTS) == declared


def test_header_compiles_as_c_and_cxx(tmp_path):
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "chaoticus.h"\nint main(void){chs_stepper s; s.adaptive = 0; return (int)sizeof(chs_problem) * 0 + s.adaptive;}\n')
    inc = os.path.join(ROOT, "include")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", inc, "-c", str(src), "-o", str(tmp_path / "t.o")], check=True)
    subprocess.run(["g++", "-std=c++17", "-Wall", "-Werror", "-x", "c++", "-I", inc, "-c", str(src), "-o", str(tmp_path / "t2.o")], check=True)


def test_host_logic_without_gpu(lib):
    from paper_2507_00622_b200 import binding as chs
    assert chs.version() == 220
    assert chs.dim(chs.SYS_HENON_HEILES) == 4 and chs.dim(chs.SYS_COUPLED3, [1, 2, 3, 0.1]) == 6
    assert chs.dim(chs.SYS_FPUT, [8, 1, 0, 1]) == 16 and chs.dim(chs.SYS_FPUT, [8.5, 1, 0, 1]) == -1
    assert chs.dim(chs.SYS_COUPLED3, [1.0]) == -1 and chs.dim(9) == -1
    # sampling rule (include/chaoticus.h): ceil(n_steps/m)/sample_every + 1
    assert chs.n_samples(10000, 1, 0) == 1
    assert chs.n_samples(10000, 1, 500) == 21
    assert chs.n_samples(1000, 7, 10) == 143 // 10 + 1
    assert chs.n_samples(2003, 10, 25) == 201 // 25 + 1


def test_package_reexports_the_whole_binding(lib):
    """Every public function / class of binding.py that wraps an entry point is reachable as
    paper_2507_00622_b200.<name> (the lazy re-export list once missed ld_adaptive and LdReport)."""
    import inspect
    import paper_2507_00622_b200 as pkg
    from paper_2507_00622_b200 import binding
    public = [n for n, o in vars(binding).items()
              if not n.startswith("_") and (inspect.isfunction(o) or inspect.isclass(o)) and o.__module__ == binding.__name__]
    assert {"ld_adaptive", "ld_adaptive_host", "LdReport", "HostLdReport", "ld_neighbour_diffs_noalloc"} <= set(public)
    for name in public:
        assert getattr(pkg, name) is getattr(binding, name), name
    with pytest.raises(AttributeError):
        pkg.no_such_entry_point


def test_n_samples_matches_oracle(orc):
    from paper_2507_00622_b200 import binding as chs
    for n_steps, m, se in [(0, 1, 1), (1, 1, 1), (999, 10, 3), (1000, 10, 3), (12345, 7, 11)]:
        assert chs.n_samples(n_steps, m, se) == orc.n_samples(n_steps, m, se)


# ---- the generated coefficient header -----------------------------------------------------------
def _parse_coeffs():
    txt = open(os.path.join(ROOT, "paper_2507_00622_b200", "csrc", "dop8_coeffs.h")).read()
    out = {}
    for name, dims, body in re.findall(r"constexpr double (\w+)((?:\[\d+\])+) = \{(.*?)\};", txt, flags=re.S):
        body = re.sub(r"/\*.*?\*/", "", body, flags=re.S).replace("{", "").replace("}", "")
        vals = [float.fromhex(v.strip()) if "x" in v else float(v) for v in body.split(",") if v.strip()]
        shape = [int(d) for d in re.findall(r"\[(\d+)\]", dims)]
        out[name] = np.array(vals).reshape(shape)
    return out


def test_separable_coefficients_order_conditions():
    """Conditions specific to the second-order (Nystrom-like) form the kernels use:
    sum_l A2_il c_l^k = c_i^(k+2)/((k+1)(k+2)) cannot hold for every stage, but the WEIGHTS must
    integrate x'' = t^k exactly: sum_l BQ_l c_l^k = 1/((k+1)(k+2)), sum_l B_l c_l^k = 1/(k+1),
    k = 0..6 / 0..7, and the embedded weights must annihilate low-degree polynomials."""
    c = _parse_coeffs()
    A, A2, CS, B, BQ = c["A"], c["A2"], c["CS"], c["B"], c["BQ"]
    assert np.abs(A @ A - A2).max() <= 1e-13   # float matmul vs the exact rational product
    assert np.abs(A.sum(1) - CS).max() <= 1e-14
    assert (np.triu(A) == 0).all() and (np.triu(A2, -1) == 0).all()
    assert np.count_nonzero(A) == 50 and np.count_nonzero(A2) == 48
    assert np.count_nonzero(B) == 8 and np.count_nonzero(BQ) == 7
    for k in range(8):
        assert abs(B @ CS ** k - 1.0 / (k + 1)) <= 1e-14, k
    for k in range(7):
        assert abs(BQ @ CS ** k - 1.0 / ((k + 1) * (k + 2))) <= 1e-14, k
    # b^T A = b (1 - c) (simplifying assumption D(1)), hence the structural zeros of BQ
    assert np.abs(BQ - B * (1 - CS)).max() <= 1e-14
    E5, E3, E5Q, E3Q = c["E5"], c["E3"], c["E5Q"], c["E3Q"]
    assert abs(E5.sum()) <= 1e-15 and abs(E3.sum()) <= 2e-15
    assert np.abs(E5 @ A - E5Q).max() <= 1e-14 and np.abs(E3 @ A - E3Q).max() <= 1e-14
    for k in range(5):
        assert abs(E5 @ CS ** k) <= 1e-14
    assert abs(E5 @ CS ** 5) > 1e-5
    for k in range(3):
        assert abs(E3 @ CS ** k) <= 1e-14
    assert abs(E3 @ CS ** 3) > 1e-3


def test_separable_form_equals_generic_form_on_cpu(orc):
    """The rearrangement itself, checked with numpy against the oracle's generic step: for
    H = p^2/2 + V(q) the separable combination of the 12 forces gives the same y+ (round-off)."""
    c = _parse_coeffs()
    A2, CS, B, BQ = c["A2"], c["CS"], c["B"], c["BQ"]
    y = np.array([0.05, 0.1, 0.35, -0.2])
    h = 0.1
    q, p = y[:2].copy(), y[2:].copy()

    def force(Q):
        x, yy = Q
        return np.array([-x - 2 * x * yy, -yy - x * x + yy * yy])

    F = np.zeros((12, 2))
    for i in range(12):
        Q = q + CS[i] * h * p + h * h * (A2[i] @ F)
        F[i] = force(Q)
    qn = q + h * p + h * h * (BQ @ F)
    pn = p + h * (B @ F)
    Y, K, _ = orc.step(0, None, y, h)
    assert np.abs(np.concatenate([qn, pn]) - Y).max() <= 5e-16
    assert np.abs(F - K[:, 2:]).max() <= 1e-15   # the stored stage forces are the p-half of k_i


def test_missing_library_fails_loudly(tmp_path, monkeypatch):
    """No CPU fallback: the binding refuses to import without the shared library."""
    import importlib.util
    src = os.path.join(ROOT, "paper_2507_00622_b200", "binding.py")
    dst = tmp_path / "binding_copy.py"
    dst.write_text(open(src).read())
    spec = importlib.util.spec_from_file_location("binding_copy", str(dst))
    mod = importlib.util.module_from_spec(spec)
    with pytest.raises(ImportError):
        spec.loader.exec_module(mod)


def test_compute_call_without_device_is_an_error(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2507_00622_b200 import binding as chs
    with pytest.raises(chs.ChaoticusError):
        chs.kernel_info(chs.SYS_HENON_HEILES, None, chs.WHAT_LD)


def test_every_kernel_is_spill_free(lib):
    """north_star: zero register spills.  The build keeps ptxas -v output per translation unit."""
    from paper_2507_00622_b200 import build
    rep = build.spill_report()
    if not rep.strip():   # library was up to date and the logs are gone: rebuild to get them
        build.build(force=True)
        rep = build.spill_report()
    lines = [l for l in rep.splitlines() if l.strip()]
    assert len(lines) >= 60
    for l in lines:
        assert "spill_st=0 spill_ld=0" in l, l
        regs = int(re.search(r"regs=\s*(\d+)", l).group(1))
        assert regs <= 255, l
    import subprocess
    sass = subprocess.run(["cuobjdump", "-sass", build.LIB], capture_output=True, text=True).stdout
    assert len(sass) > 1_000_000
    # no local-memory instruction in ANY kernel (the double pendulum's kernels use fast_sincos, not the CUDA
    # library's sincos(), whose huge-argument slow path keeps an array on the stack), and no stack frame
    funcs = re.split(r"\n\s*Function : ", sass)
    assert len(funcs) >= 160
    for f in funcs[1:]:
        name = f.split("\n", 1)[0]
        assert not re.search(r"\b(STL|LDL)\b", f), name
    logs = "".join(open(os.path.join(build.BUILD, f"ptxas_{u}.log")).read() for u in build.UNITS)
    frames = re.findall(r"(\d+) bytes stack frame", logs)
    assert len(frames) >= 160 and all(int(x) == 0 for x in frames)
    assert "DFMA" in sass and "SHFL" in sass


def test_backward_ld_is_forward_ld_of_reversed_momenta(orc):
    """The LD kernel runs the backward pass as the forward pass of (q, -p): for
    H even in p this is exact, bit for bit -- checked here on the oracle, which integrates the
    backward pass literally with step -h."""
    from paper_2507_00622_b200 import workloads as W
    y0 = W.hh_grid(0.125, 7, 6)
    _, b = orc.ld(0, None, y0, 0.0, 0.01, 300, forward=False, precision="f64")
    yr = y0.copy()
    yr[2:] *= -1.0
    f, _ = orc.ld(0, None, yr, 0.0, 0.01, 300, backward=False, precision="f64")
    assert (f == b).all()
    prm = W.fput_params(8, 1.0, 0.3, 1.0)
    y0 = W.fput_ics(9, 8, seed=4)
    _, b = orc.ld(2, prm, y0, 0.0, 0.05, 100, forward=False, precision="f64")
    yr = y0.copy()
    yr[8:] *= -1.0
    f, _ = orc.ld(2, prm, yr, 0.0, 0.05, 100, backward=False, precision="f64")
    assert (f == b).all()
