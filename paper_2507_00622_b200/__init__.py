"""paper_2507_00622_b200 -- B200-native (sm_100a, FP64) ensemble DOP8 integrator with chaos
indicators (the hot path of arXiv 2507.00622).

    binding    ctypes binding of libchaoticus.so (C ABI: include/chaoticus.h); loaded lazily,
               raises ImportError if the library has not been built (no CPU fallback)
    workloads  seeded synthetic input generators (no arithmetic of the method)
    build      in-tree nvcc build of the library
"""
import importlib

_API = ("integrate_fixed", "integrate_adaptive", "sali", "gali", "ld", "ld_adaptive", "ld_neighbours",
        "ld_neighbour_diffs_noalloc", "lyap", "ld_host", "ld_adaptive_host", "ld_neighbours_host", "sali_host",
        "gali_host", "lyap_host", "integrate_host", "Report", "HostReport", "LdReport", "HostLdReport", "kernel_info",
        "dim", "n_samples", "version", "set_option", "ChaoticusError")


def __getattr__(name):
    if name in ("binding", "workloads", "build"):
        return importlib.import_module(f"{__name__}.{name}")
    if name in _API:
        return getattr(importlib.import_module(f"{__name__}.binding"), name)
    raise AttributeError(name)
