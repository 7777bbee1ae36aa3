"""Builds paper_2507_00622_b200/libchaoticus.so (the product) and libchaoticus_probe.so (the
bench-only DFMA peak probe) in-tree with nvcc for sm_100a.

    python -m paper_2507_00622_b200.build [--force]

One object per translation unit, compiled in parallel; -Xptxas -v output of each is kept in
build/ptxas_<name>.log (register counts and spill bytes: the spill-free evidence).
"""
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libchaoticus.so")
PROBE_LIB = os.path.join(HERE, "libchaoticus_probe.so")
UNITS = ["chaoticus", "inst_hh", "inst_hh_ind", "inst_hh_adapt", "inst_hh_adapt2", "inst_c3", "inst_c3_lyap",
         "inst_c3_more", "inst_dp", "inst_fput", "inst_fput_adapt", "inst_fput_spec",
         "inst_fput_n4", "inst_fput_n8", "inst_fput_n16", "inst_fput_n32", "inst_fput_n64",
         "inst_fput_pad4", "inst_fput_pad8", "inst_fput_pad16", "inst_fput_pad32", "inst_fput_pad64",
         "inst_fput_wide64", "inst_fput_wide128", "inst_fput_wide256"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xptxas", "-v",
              "-Xcompiler", "-fPIC"]


def _deps():
    return [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h", ".cu"))] + \
           [os.path.join(os.path.dirname(HERE), "include", "chaoticus.h")]


def _compile(unit):
    src = os.path.join(CSRC, unit + ".cu")
    obj = os.path.join(BUILD, unit + ".o")
    r = subprocess.run(["nvcc", *NVCC_FLAGS, "-c", src, "-o", obj], capture_output=True, text=True)
    with open(os.path.join(BUILD, f"ptxas_{unit}.log"), "w") as f:
        f.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {unit}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force=False, verbose=False):
    os.makedirs(BUILD, exist_ok=True)
    deps = _deps()
    newest = max(os.path.getmtime(d) for d in deps)
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest and os.path.exists(PROBE_LIB)
            and os.path.getmtime(PROBE_LIB) >= newest):
        return LIB
    with cf.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(_compile, UNITS + ["probe"]))
    for lib, members in ((LIB, objs[:-1]), (PROBE_LIB, objs[-1:])):
        r = subprocess.run(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib, *members,
                            "-lcudart"], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(spill_report())
    return LIB


def spill_report():
    """One line per kernel: registers and spill bytes, from the kept ptxas logs."""
    import re
    out = []
    for unit in UNITS:
        p = os.path.join(BUILD, f"ptxas_{unit}.log")
        if not os.path.exists(p):
            continue
        txt = open(p).read()
        for m in re.finditer(r"Compiling entry function '(\S+)'.*?(\d+) bytes spill stores, (\d+) bytes spill loads"
                             r".*?Used (\d+) registers", txt, re.S):
            out.append(f"{unit:14s} regs={int(m.group(4)):3d} spill_st={m.group(2)} spill_ld={m.group(3)}  {m.group(1)}")
    return "\n".join(out)


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print("built", LIB)
