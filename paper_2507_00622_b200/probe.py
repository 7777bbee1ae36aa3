"""FP64 FMA peak probe (measurement aid for bench.py).

A register-only DFMA microbenchmark in its own small library, libchaoticus_probe.so -- it is not
part of the product C ABI (include/chaoticus.h).  mode 0: fixed register operands (the pipe's
ceiling); mode 1: multiplier from the constant bank, as the step kernels read the tableau;
mode 2: three distinct register operands per DFMA (register-file bandwidth included).
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchaoticus_probe.so")
_lib = None


def _load():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2507_00622_b200.build`")
        _lib = C.CDLL(LIB_PATH)
        _lib.chs_probe_dfma.argtypes = [C.c_int, C.c_longlong, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        _lib.chs_probe_math.argtypes = [C.c_int, C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    return _lib


def dfma_probe(iters, n_blocks, n_threads=256, mode=0):
    """Launches the probe on the current stream; returns (FP64 flop it performs, output tensor)."""
    out = torch.empty(n_blocks * n_threads, dtype=torch.float64, device="cuda")
    rc = _load().chs_probe_dfma(mode, int(iters), n_blocks, n_threads, out.data_ptr(),
                                torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError(f"chs_probe_dfma rc={rc}")
    return 2.0 * 16.0 * iters * n_blocks * n_threads, out


MATH_FNS = {"fast_sqrt": 0, "fast_rsqrt": 1, "fast_rcp": 2, "fast_sincos": 3}


def math_probe(name, x):
    """The kernels' own math helper `name` (csrc/dop8_core.cuh, csrc/gen_kernels.cuh) applied to every element
    of the CUDA float64 tensor x: returns one tensor, or (sin, cos) for fast_sincos.  Test aid."""
    out1 = torch.empty_like(x)
    out2 = torch.empty_like(x) if name == "fast_sincos" else None
    rc = _load().chs_probe_math(MATH_FNS[name], x.numel(), x.data_ptr(), out1.data_ptr(),
                                out2.data_ptr() if out2 is not None else None, torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError(f"chs_probe_math rc={rc}")
    return (out1, out2) if out2 is not None else out1
