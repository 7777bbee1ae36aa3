#!/usr/bin/env python3
"""bench.py -- throughput of the hot path on the workloads of BASELINE.json.

Headline (BASELINE.json configs[1], "C2", the configuration the metric is quoted on): Henon-Heiles
arc-length Lagrangian descriptor, E = 1/8, 1024 x 1024 energy-fitted grid of (y, py) on the x = 0
section, forward and backward fixed-step DOP8, h = 0.01, |t| = 50 (5000 steps per direction), FP64.
One "step" of the benchmark = one pass of the whole hot path over that batch = 2 * 1048576 * 5000
RK-steps, one kernel launch.  Metric: trajectory RK-steps/sec.

The same JSON line carries `per_config`: all five BASELINE configs (C1..C5, the four with variational
equations included) plus C1sat (the C1 kernel on a saturating ensemble), each timed the same way
(CUDA events on the launching stream, L2 flushed, >= 5 runs after warm-up), with its roofline fraction,
kernel launch shape, end-to-end number (host buffers through the C ABI) and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C2|...]

--gpus N > 1 without a torchrun environment re-launches itself under torch.distributed.run with N
ranks; every rank integrates its own 1024 x 1024 block of rows of a (1024 N) x 1024 grid (weak
scaling, no data-path collective: trajectories are independent).
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line on rank 0.
"""
import argparse
import csv
import json
import os
import socket
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "trajectory RK-steps/sec (FP64, incl. variational eqs)"
UNIT = "RK-steps/s"
# algorithmic FP64 flop per RK-step of the formulation that runs
FLOP_PER_STEP = {"C1": 1216.0, "C2": 640.0, "C1sat": 1216.0, "C3": 1692.0, "C4": 4213.0, "C5": 8492.0, "F3": None,
                 "F1": None, "LDN": 640.0, "LDA": None}
WORKLOAD_LABEL = {
    "C1": "C1: Henon-Heiles E=1/8, 32x32 grid (1024 ICs), fixed DOP8 h=0.01, 1e4 steps, SALI renormalised every step",
    "C2": "C2: Henon-Heiles Lagrangian descriptor (arc length), E=1/8, 1024x1024 grid per GPU, fixed DOP8 h=0.01, 5000 steps forward + 5000 backward",
    "C1sat": "C1sat: Henon-Heiles fixed-step SALI kernel of configs[0] (h=0.01, renormalised every step) on a --sali-side^2 grid, --sali-steps steps",
    "C3": "C3: Henon-Heiles adaptive DOP8(5) rtol=atol=1e-12, 512x512 grid at E=1/6, t=1000, SALI (RK-step = attempted step)",
    "C4": "C4: 3-DoF coupled oscillators, 65536 ICs, full Lyapunov spectrum (6 vectors, MGS every 10 steps), h=0.01, 1e5 steps",
    "C5": "C5: FPUT-beta N=8, 65536 ICs, GALI_4 (renormalised every 10 steps), h=0.05, 2e4 steps",
    "F1": "F1 (shape of PAPER.md Fig. 1): dimensionless double pendulum (sigma = alpha = 1), random ICs, t = 1000, fixed h = 0.01 or adaptive rtol = atol = 1e-9",
    "F3": "F3 (shape of PAPER.md Fig. 3): FPUT-beta chain, random ICs, GALI_4, adaptive DOP8(5) rtol=atol=1e-8, t=1000",
    "LDA": "LDA: the C2 grid with the ADAPTIVE solver (chaoticus_ld_adaptive: augmented ODE (y, M), rtol=atol=1e-10), tau = h * --n-steps forward + backward (RK-step = attempted step)",
    "LDN": "LDN: LD of every IC of the C2 grid and of its 2n axis neighbours x0 +- sigma e_i, generated on the device (PAPER.md:57-58), fixed DOP8 h=0.01, --n-steps steps forward + backward",
}
PER_CONFIG = ["C1", "C1sat", "C2", "C3", "C4", "C5"]
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12  # 37.2
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "kernel_traffic.csv")


def parse(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=list(WORKLOAD_LABEL))
    ap.add_argument("--configs", default=",".join(PER_CONFIG),
                    help="per_config entries of the headline line (comma list, '' = none)")
    ap.add_argument("--config-steps", type=int, default=5, help="timed runs of each per_config entry")
    ap.add_argument("--f1-adaptive", action="store_true", help="F1: adaptive DOP8(5) instead of fixed step")
    ap.add_argument("--shrink", type=int, default=1, help="C3/C4/C5/F3: divide the horizon (profiling runs)")
    ap.add_argument("--shrink-ic", type=int, default=1, help="C3/C4/C5: divide the ensemble (profiling runs)")
    ap.add_argument("--side", type=int, default=1024, help="grid side per rank (C2)")
    ap.add_argument("--n-steps", type=int, default=5000, help="DOP8 steps per direction (C2)")
    ap.add_argument("--sali-side", type=int, default=512, help="C1sat: grid side per rank")
    ap.add_argument("--sali-steps", type=int, default=2000, help="C1sat: DOP8 steps")
    ap.add_argument("--fput-n", type=int, default=8, help="F3: chain length (1..256)")
    ap.add_argument("--n-ic", type=int, default=1000, help="F3: ensemble size (PAPER.md:129: 10^3 random ICs)")
    ap.add_argument("--ldn-sigma", type=float, default=1e-3, help="LDN: neighbour displacement")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweeps", action="store_true", help="skip the FPUT DoF and ensemble-size sweeps of the headline line")
    return ap.parse_args(argv)


# ------------------------------------------------------------------------------------ launch plan
def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_plan(gpus, env, argv):
    """How this process takes part in an N-GPU run.  Returns
    ("run", rank, local_rank, world)  run the benchmark as that rank (world = 1: no process group);
    ("spawn", cmd)                    --gpus N > 1 outside torchrun: re-launch under torch.distributed.run;
    ("error", message)                --gpus N contradicts the torchrun environment.
    bench.py never reports n_gpus other than the number of ranks that ran."""
    if gpus < 1:
        return ("error", f"--gpus {gpus}: need >= 1")
    ws = env.get("WORLD_SIZE")
    if ws is None:
        if gpus == 1:
            return ("run", 0, 0, 1)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__), *argv]
        return ("spawn", cmd)
    world = int(ws)
    if world != gpus:
        return ("error", f"--gpus {gpus} but WORLD_SIZE={world}: launch with --nproc-per-node {gpus}")
    return ("run", int(env.get("RANK", "0")), int(env.get("LOCAL_RANK", "0")), world)


def rank_max(x, world, device=None):
    """max over ranks of a python float (the device-timed duration); identity at world = 1."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(rk_steps_per_rank, world, steps, t_max):
    """whole-job throughput: the units all ranks processed / the max-over-ranks time (weak scaling)."""
    return rk_steps_per_rank * world * steps / t_max


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md): ONE
    nvidia-smi process looping every 200 ms, started before and killed after the region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.out = index, None, ""

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            time.sleep(0.3)   # let it take its first sample before the region starts
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.out = self.proc.communicate(timeout=5)[0]
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0, set()
        for line in self.out.splitlines():
            r = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def kernel_traffic(workload):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the workload's kernel from
    the tracked ncu --set full captures (profiles/kernel_traffic.csv), or None if not captured."""
    try:
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                if row["workload"] == workload:
                    return int(float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]))
    except Exception:
        pass
    return None


def workload_inputs(args, rank, world):
    from paper_2507_00622_b200 import workloads as W
    if args.workload in ("C2", "LDN", "LDA"):
        side = args.side
        y0 = W.hh_grid(0.125, side * world, side, i_range=(rank * side, (rank + 1) * side))
        return dict(y0=y0, h=0.01, n_steps=args.n_steps, rk_steps=2.0 * y0.shape[1] * args.n_steps)
    # C1sat: the fixed-step SALI kernel of configs[0] on a saturating ensemble
    side = args.sali_side
    y0 = W.hh_grid(0.125, side * world, side, i_range=(rank * side, (rank + 1) * side))
    w0 = W.deviation_vectors(y0.shape[1], 2, 4, 0, "unit")
    return dict(y0=y0, w0=w0, h=0.01, n_steps=args.sali_steps, rk_steps=1.0 * y0.shape[1] * args.sali_steps)


# ------------------------------------------------------------------------------------ CPU oracle leg
def _oracle_call(orc, name, args, y, w, prec="f64", threads=None, frac=1.0):
    """One oracle pass of workload `name` over the ICs (y, w) with the horizon scaled by frac.
    Returns the RK-steps it performed."""
    from paper_2507_00622_b200 import workloads as W
    kw = dict(precision=prec, threads=threads)
    n = y.shape[1]
    if name == "C2":
        ns = max(1, int(round(args.n_steps * frac)))
        orc.ld(0, None, y, 0.0, 0.01, ns, **kw)
        return 2.0 * n * ns
    if name in ("C1", "C1sat"):
        ns = max(1, int(round((10_000 if name == "C1" else args.sali_steps) * frac)))
        orc.sali(0, None, y, w, renorm_every=1, h=0.01, n_steps=ns, **kw)
        return 1.0 * n * ns
    if name == "C3":
        r = orc.sali(0, None, y, w, renorm_every=1, adaptive=True, t_end=1000.0 * frac, rtol=1e-12, atol=1e-12, **kw)
        return float(r["n_accepted"].sum() + r["n_rejected"].sum())
    if name == "C4":
        ns = max(10, int(round(100_000 * frac)))
        orc.lyap(1, W.coupled3_params(0.1), y, w, renorm_every=10, h=0.01, n_steps=ns, **kw)
        return 1.0 * n * ns
    if name == "C5":
        ns = max(10, int(round(20_000 * frac)))
        orc.gali(2, W.fput_params(8, 1.0, 0.0, 1.0), y, w, renorm_every=10, h=0.05, n_steps=ns, **kw)
        return 1.0 * n * ns
    raise ValueError(name)


def _oracle_ics(name, args, n_ic):
    """n_ic initial conditions spread over the workload's ensemble (strided subsample)."""
    from paper_2507_00622_b200 import workloads as W
    if name in ("C1", "C1sat", "C2", "C3"):
        side = {"C1": 32, "C1sat": args.sali_side, "C2": args.side, "C3": 512}[name]
        E = 1.0 / 6.0 if name == "C3" else 0.125
        sub = max(1, min(side, int(round(np.sqrt(n_ic)))))
        idx = np.unique(np.linspace(0, side - 1, sub).round().astype(int))
        rows = [W.hh_grid(E, side, side, i_range=(int(i), int(i) + 1))[:, idx] for i in idx]
        y = np.ascontiguousarray(np.concatenate(rows, axis=1))
        w = W.deviation_vectors(y.shape[1], 2, 4, 0, "unit") if name != "C2" else None
        return y, w, f"{len(idx)}x{len(idx)} sub-grid of the {side}x{side} grid"
    cfg = W.config(name)
    idx = np.unique(np.linspace(0, cfg["y"].shape[1] - 1, n_ic).round().astype(int))
    return (np.ascontiguousarray(cfg["y"][:, idx]), np.ascontiguousarray(cfg["w"][:, :, idx]),
            f"{len(idx)} ICs spread evenly over the 65536")


def size_sample(orc, name, args, target_s):
    """A sample of the workload's ensemble (full horizon) sized from a short calibration run so that the
    oracle, as it stands, needs about target_s seconds on it.  Returns (y, w, description, cores)."""
    cores = orc.default_threads()
    full = {"C1": 1024, "C1sat": args.sali_side ** 2, "C2": args.side ** 2, "C3": 512 * 512, "C4": 65536, "C5": 65536}[name]
    n_cal = min(full, 16 * cores)           # the oracle hands out ICs in chunks of 16 per thread
    yc, wc, _ = _oracle_ics(name, args, n_cal)
    fc = {"C1": 0.05, "C1sat": 0.1, "C2": 0.05, "C3": 0.02, "C4": 0.004, "C5": 0.01}[name]
    _oracle_call(orc, name, args, yc[:, :16].copy(), None if wc is None else wc[:, :, :16].copy(), threads=cores,
                 frac=fc / 4)   # thread start-up
    t = time.perf_counter()
    rk = _oracle_call(orc, name, args, yc.copy(), None if wc is None else wc.copy(), threads=cores, frac=fc)
    rate = rk / (time.perf_counter() - t)
    per_ic = rk / fc / yc.shape[1]           # RK-steps of one IC over the full horizon
    n_ic = int(max(16 * cores, min(full, rate * target_s / per_ic)))
    if n_ic < full:
        n_ic = max(16 * cores, (n_ic // (16 * cores)) * 16 * cores)
    y, w, what = _oracle_ics(name, args, n_ic)
    return y, w, what, cores


def cpu_baseline(orc, name, args, target_s):
    """The oracle as it stands (double, gcc -O2, OpenMP over ICs, all host cores) on a BOUNDED sample of
    the workload with the FULL horizon."""
    y, w, what, cores = size_sample(orc, name, args, target_s)
    t = time.perf_counter()
    rk = _oracle_call(orc, name, args, y, w, threads=cores, frac=1.0)
    dt = time.perf_counter() - t
    return {"value": rk / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{what} ({y.shape[1]} ICs), full horizon, {dt:.1f} s"}


def run_reference(args):
    """The CPU oracle, as it stands, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import chaos_oracle as orc
    orc.build()
    y0, _, what, cores = size_sample(orc, "C2", args, target_s=120.0 / max(1, args.steps + args.warmup))
    times = []
    for it in range(args.warmup + args.steps):
        t = time.perf_counter()
        orc.ld(0, None, y0, 0.0, 0.01, args.n_steps, precision="f64", threads=cores)
        dt = time.perf_counter() - t
        if it >= args.warmup:
            times.append(dt)
    rk = 2.0 * y0.shape[1] * args.n_steps
    val = rk * len(times) / sum(times)
    sample = f"{what}, full horizon ({args.n_steps} steps x 2 directions)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "C2: Henon-Heiles LD, E=1/8, fixed DOP8 h=0.01, fwd+bwd (CPU oracle on a bounded sample)",
                   "n_ic_sample": int(y0.shape[1]), "n_steps_per_direction": args.n_steps},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------------ GPU workloads
def make_workload(chs, torch, args, rank, world, name=None):
    """Device-resident inputs + the two step closures (device pointers / host buffers) of a workload."""
    from paper_2507_00622_b200 import workloads as W
    HH = chs.SYS_HENON_HEILES
    name = name or args.workload
    if name == "F1":
        # shape of the paper's Fig. 1: double pendulum, tau = 10^3, fixed vs adaptive
        DPS, prm = chs.SYS_DOUBLE_PENDULUM, (1.0, 1.0)
        y0_host = torch.from_numpy(W.double_pendulum_ics(args.n_ic, seed=3)).pin_memory()
        y0 = y0_host.cuda()
        n_ic = y0.shape[1]
        yb, yh = torch.empty_like(y0), torch.empty_like(y0_host).pin_memory()
        t_end = 1000.0 / args.shrink
        if args.f1_adaptive:
            rep = chs.Report(n_ic, "cuda")
            call = lambda: chs.integrate_adaptive(DPS, prm, yb, 0.0, t_end, 1e-9, 1e-9, report=rep)
            host = lambda: chs.integrate_host(DPS, prm, yh, adaptive=True, t_end=t_end, rtol=1e-9, atol=1e-9)
            wl = dict(rk_steps=None, report=rep)
        else:
            ns = int(round(t_end / 0.01))
            call = lambda: chs.integrate_fixed(DPS, prm, yb, 0.0, 0.01, ns)
            host = lambda: chs.integrate_host(DPS, prm, yh, h=0.01, n_steps=ns)
            wl = dict(rk_steps=1.0 * n_ic * ns)

        def step_e2e():
            yh.copy_(y0_host)
            host()

        return dict(wl=wl, n_ic=n_ic, h2d=y0_host.numel() * 8, d2h=y0_host.numel() * 8,
                    kinfo=chs.kernel_info(DPS, prm, chs.WHAT_INTEGRATE, adaptive=args.f1_adaptive, n_ic=n_ic),
                    step_dev=call, step_e2e=step_e2e, prepare=lambda: yb.copy_(y0))
    if name in ("C2", "LDN", "LDA"):
        wl = workload_inputs(args, rank, world)
        y0_host = torch.from_numpy(wl["y0"]).pin_memory()
        y0 = y0_host.cuda()
        n_ic = y0.shape[1]
    if name == "C2":
        f = torch.empty(n_ic, dtype=torch.float64, device="cuda")
        b = torch.empty(n_ic, dtype=torch.float64, device="cuda")
        f_host = torch.empty(n_ic, dtype=torch.float64).pin_memory()
        b_host = torch.empty(n_ic, dtype=torch.float64).pin_memory()
        return dict(wl=wl, n_ic=n_ic, h2d=y0_host.numel() * 8, d2h=2 * n_ic * 8,
                    kinfo=chs.kernel_info(HH, None, chs.WHAT_LD, n_ic=n_ic),
                    step_dev=lambda: chs.ld(HH, None, y0, 0.0, wl["h"], wl["n_steps"], out_fwd=f, out_bwd=b),
                    step_e2e=lambda: chs.ld_host(HH, None, y0_host, 0.0, wl["h"], wl["n_steps"], f_host, b_host))
    if name == "LDA":
        tau = wl["h"] * wl["n_steps"]
        rep = chs.LdReport(n_ic, "cuda")
        f_host = torch.empty(n_ic, dtype=torch.float64).pin_memory()
        b_host = torch.empty(n_ic, dtype=torch.float64).pin_memory()
        wl = dict(wl, rk_steps=None, report=rep)
        return dict(wl=wl, n_ic=n_ic, h2d=y0_host.numel() * 8, d2h=2 * n_ic * 8,
                    kinfo=chs.kernel_info(HH, None, chs.WHAT_LD, adaptive=True, n_ic=n_ic),
                    step_dev=lambda: chs.ld_adaptive(HH, None, y0, 0.0, tau, rtol=1e-10, atol=1e-10, report=rep),
                    step_e2e=lambda: chs.ld_adaptive_host(HH, None, y0_host, 0.0, tau, f_host, b_host, rtol=1e-10, atol=1e-10))
    if name == "LDN":
        nn = 1 + 2 * 4
        f = torch.empty((nn, n_ic), dtype=torch.float64, device="cuda")
        b = torch.empty((nn, n_ic), dtype=torch.float64, device="cuda")
        f_host = torch.empty((nn, n_ic), dtype=torch.float64).pin_memory()
        b_host = torch.empty((nn, n_ic), dtype=torch.float64).pin_memory()
        wl["rk_steps"] *= nn
        sg = args.ldn_sigma
        return dict(wl=wl, n_ic=n_ic, h2d=y0_host.numel() * 8, d2h=2 * nn * n_ic * 8,
                    kinfo=chs.kernel_info(HH, None, chs.WHAT_LD, n_ic=n_ic * nn),
                    step_dev=lambda: chs.ld_neighbours(HH, None, y0, sg, 0.0, wl["h"], wl["n_steps"], out_fwd=f, out_bwd=b),
                    step_e2e=lambda: chs.ld_neighbours_host(HH, None, y0_host, sg, 0.0, wl["h"], wl["n_steps"], f_host, b_host))
    # the other workloads advance y, w in place: every step starts from a fresh device copy made
    # OUTSIDE the timed events (prepare), so only the library's kernel is timed
    if name in ("C1", "C1sat"):
        if name == "C1":
            cfg = W.config("C1")
            wl = dict(y0=cfg["y"], w0=cfg["w"], h=0.01, n_steps=10_000, rk_steps=1024.0 * 10_000)
        else:
            a2 = argparse.Namespace(**vars(args))
            a2.workload = "C1sat"
            wl = workload_inputs(a2, rank, world)
        y0_host = torch.from_numpy(wl["y0"]).pin_memory()
        y0 = y0_host.cuda()
        n_ic = y0.shape[1]
        sysid, prm, w0_np, k = HH, None, wl["w0"], 2
        call = lambda y, w: chs.sali(HH, None, y, w, renorm_every=1, h=wl["h"], n_steps=wl["n_steps"])
        host = lambda y, w, o: chs.sali_host(HH, None, y, w, o, renorm_every=1, h=wl["h"], n_steps=wl["n_steps"])
        out_rows, what, adaptive = 1, chs.WHAT_SALI, False
    elif name == "F3":
        # shape of the paper's Fig. 3: FPUT, 10^3 random ICs, GALI_4, adaptive
        # solver, atol = 1e-8, tau = 10^3, as a function of the number of degrees of freedom
        N = args.fput_n
        sysid, prm = chs.SYS_FPUT, W.fput_params(N, 1.0, 0.0, 1.0)
        y0_host = torch.from_numpy(W.fput_ics(args.n_ic, N, seed=2, E=0.125 * N)).pin_memory()
        y0 = y0_host.cuda()
        n_ic = y0.shape[1]
        w0_np = W.deviation_vectors(n_ic, 4, 2 * N, 102, "orthonormal")
        k = 4
        rep = chs.Report(n_ic, "cuda")
        t_end = 1000.0 / args.shrink
        call = lambda y, w: chs.gali(sysid, prm, y, w, renorm_every=1, adaptive=True, t_end=t_end, rtol=1e-8,
                                     atol=1e-8, report=rep)
        host = lambda y, w, o: chs.gali_host(sysid, prm, y, w, o, renorm_every=1, adaptive=True, t_end=t_end,
                                             rtol=1e-8, atol=1e-8)
        out_rows, what, adaptive = 1, chs.WHAT_GALI, True
        wl = dict(rk_steps=None, report=rep)
    else:
        n_full = {"C3": 512 * 512, "C4": 65536, "C5": 65536}[name]
        cfg = W.config(name, n_ic=max(1024, n_full // args.shrink_ic) if args.shrink_ic > 1 else None)
        sysid, prm, w0_np = cfg["system"], cfg["params"], cfg["w"]
        k = w0_np.shape[0]
        y0_host = torch.from_numpy(cfg["y"]).pin_memory()
        y0 = y0_host.cuda()
        n_ic = y0.shape[1]
        ns = max(10, cfg.get("n_steps", 0) // args.shrink)
        if name == "C3":
            t_end = cfg["t_end"] / args.shrink
            rep = chs.Report(n_ic, "cuda")
            call = lambda y, w: chs.sali(sysid, prm, y, w, renorm_every=1, adaptive=True, t_end=t_end, rtol=1e-12,
                                         atol=1e-12, report=rep)
            host = lambda y, w, o: chs.sali_host(sysid, prm, y, w, o, renorm_every=1, adaptive=True, t_end=t_end,
                                                 rtol=1e-12, atol=1e-12)
            out_rows, what, adaptive = 1, chs.WHAT_SALI, True
            wl = dict(rk_steps=None, report=rep)
        elif name == "C4":
            call = lambda y, w: chs.lyap(sysid, prm, y, w, renorm_every=10, h=cfg["h"], n_steps=ns)
            host = lambda y, w, o: chs.lyap_host(sysid, prm, y, w, o, renorm_every=10, h=cfg["h"], n_steps=ns)
            out_rows, what, adaptive = k, chs.WHAT_LYAP, False
            wl = dict(rk_steps=1.0 * n_ic * ns)
        else:
            call = lambda y, w: chs.gali(sysid, prm, y, w, renorm_every=10, h=cfg["h"], n_steps=ns)
            host = lambda y, w, o: chs.gali_host(sysid, prm, y, w, o, renorm_every=10, h=cfg["h"], n_steps=ns)
            out_rows, what, adaptive = 1, chs.WHAT_GALI, False
            wl = dict(rk_steps=1.0 * n_ic * ns)
    w0_host = torch.from_numpy(w0_np).pin_memory()
    w0 = w0_host.cuda()
    yb, wb = torch.empty_like(y0), torch.empty_like(w0)
    yh, wh = torch.empty_like(y0_host).pin_memory(), torch.empty_like(w0_host).pin_memory()
    oh = torch.empty((out_rows, n_ic), dtype=torch.float64).pin_memory()

    def prepare():
        yb.copy_(y0)
        wb.copy_(w0)

    def step_e2e():
        yh.copy_(y0_host)
        wh.copy_(w0_host)
        host(yh, wh, oh)

    return dict(wl=wl, n_ic=n_ic, h2d=(y0_host.numel() + w0_host.numel()) * 8,
                d2h=(y0_host.numel() + w0_host.numel() + out_rows * n_ic) * 8,
                kinfo=chs.kernel_info(sysid, prm, what, k=k, adaptive=adaptive, n_ic=n_ic),
                step_dev=lambda: call(yb, wb), step_e2e=step_e2e, prepare=prepare)


def timed(torch, flush, wk, n):
    """n runs, each bracketed by CUDA events on the launching stream, L2 flushed between."""
    ms = []
    for _ in range(n):
        flush.fill_(1)
        if "prepare" in wk:
            wk["prepare"]()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        wk["step_dev"]()
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    return ms


def resolve_rk_steps(wl):
    if wl["rk_steps"] is None:   # adaptive: one RK-step = one ATTEMPTED step (accepted + rejected), counted by the kernel
        rp = wl["report"]
        wl["accepted"], wl["rejected"] = int(rp.n_accepted.sum().item()), int(rp.n_rejected.sum().item())
        wl["rk_steps"] = float(wl["accepted"] + wl["rejected"])
    return wl["rk_steps"]


def roofline_entry(name, wl, ms, dfma_tflops, full_size=True):
    flop = FLOP_PER_STEP.get(name)
    achieved = (flop * wl["rk_steps"] / (np.mean(ms) * 1e-3) / 1e12) if flop else None
    return {
        "bound": "alu", "achieved": achieved, "peak": NOMINAL_FP64_TFLOPS, "unit": "TFLOP/s",
        "frac": (achieved / NOMINAL_FP64_TFLOPS) if achieved else None,
        # DRAM bytes per launch of this kernel at this size from the tracked ncu --set full capture
        "traffic": kernel_traffic(name) if full_size else None,
        "peak_source": "nominal: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz (DESIGN.md Roofline)",
        "measured_dfma_tflops": dfma_tflops, "frac_of_measured_dfma": (achieved / dfma_tflops) if achieved else None,
        "flop_per_rk_step": flop, "kernel_ms": float(np.mean(ms)),
    }


def measure_config(chs, torch, flush, args, name, dfma_tflops, orc):
    """One per_config entry: device-timed kernel, roofline, e2e through host buffers, CPU oracle."""
    a2 = argparse.Namespace(**vars(args))
    a2.workload, a2.shrink, a2.shrink_ic = name, 1, 1
    wk = make_workload(chs, torch, a2, 0, 1, name)
    for _ in range(2):
        if "prepare" in wk:
            wk["prepare"]()
        wk["step_dev"]()
    torch.cuda.synchronize()
    ms = timed(torch, flush, wk, max(1, args.config_steps))
    wl = wk["wl"]
    rk = resolve_rk_steps(wl)
    med = float(np.median(ms))
    wk["step_e2e"]()
    t0 = time.perf_counter()
    n_e2e = 3
    for _ in range(n_e2e):
        wk["step_e2e"]()
    torch.cuda.synchronize()
    t_e2e = (time.perf_counter() - t0) / n_e2e
    ent = {
        "workload": WORKLOAD_LABEL[name], "n_ic": int(wk["n_ic"]), "rk_steps": rk, "ms": med,
        "ms_each": [round(x, 3) for x in ms], "ns_per_step_per_trajectory": 1e6 * med / (rk / wk["n_ic"]),
        "rk_steps_per_s": rk / (med * 1e-3), "flop_per_rk_step": FLOP_PER_STEP[name],
        "roofline": roofline_entry(name, wl, [med], dfma_tflops), "kernel": wk["kinfo"],
        "e2e": {"value": rk / t_e2e, "unit": UNIT, "ms": 1e3 * t_e2e, "h2d_bytes_per_step": int(wk["h2d"]),
                "d2h_bytes_per_step": int(wk["d2h"])},
    }
    if "accepted" in wl:
        ent["accepted_steps"], ent["rejected_steps"] = wl["accepted"], wl["rejected"]
    if orc is not None:
        ent["cpu_baseline"] = cpu_baseline(orc, name, a2, target_s=8.0)
    del wk
    torch.cuda.empty_cache()
    return ent


def run_sweeps(chs, torch, flush, args):
    """Shapes of the paper's figures, driver-timed (one warm-up + 2 timed runs each, median):
    fput_dof      PAPER.md:113, 129 (Fig. 3): FPUT-beta, GALI_4, adaptive DOP8(5) rtol = atol = 1e-8 on a
                  SATURATING ensemble (65536 ICs, t = 100) as a function of the chain length N -- the
                  "linear trend" in the number of degrees of freedom; N spans every tile class (exact and
                  padded in-warp tiles, wide tiles);
    ensemble_size PAPER.md:94, 125 (Fig. 2): the fixed-step SALI kernel, time per IC against the number of
                  simultaneously integrated ICs;
    ensemble_size_adaptive  the same curve with the adaptive solver (the solver of the paper's Fig. 2)."""
    out = {"fput_dof": [], "ensemble_size": [], "ensemble_size_adaptive": []}
    for N in (4, 8, 12, 16, 32, 48, 64, 128):
        a2 = argparse.Namespace(**vars(args))
        a2.workload, a2.fput_n, a2.n_ic, a2.shrink, a2.shrink_ic = "F3", N, 65536, 10, 1
        wk = make_workload(chs, torch, a2, 0, 1, "F3")
        wk["prepare"]()
        wk["step_dev"]()
        ms = timed(torch, flush, wk, 2)
        rk = resolve_rk_steps(wk["wl"])
        med = float(np.median(ms))
        out["fput_dof"].append({"N": N, "n_ic": 65536, "t_end": 100.0, "ms": med, "ms_per_dof": med / N,
                                "accepted": wk["wl"]["accepted"], "rejected": wk["wl"]["rejected"],
                                "attempts_per_s": rk / (med * 1e-3), "lanes": wk["kinfo"]["lanes"],
                                "regs": wk["kinfo"]["regs"], "spill_bytes": wk["kinfo"]["spill_bytes"]})
        del wk
        torch.cuda.empty_cache()
    for side, ns in ((32, 10000), (64, 10000), (128, 10000), (256, 10000), (512, 2000), (1024, 2000)):
        a2 = argparse.Namespace(**vars(args))
        a2.workload, a2.sali_side, a2.sali_steps = "C1sat", side, ns
        wk = make_workload(chs, torch, a2, 0, 1, "C1sat")
        wk["prepare"]()
        wk["step_dev"]()
        ms = timed(torch, flush, wk, 2)
        med = float(np.median(ms))
        rk = wk["wl"]["rk_steps"]
        out["ensemble_size"].append({"n_ic": side * side, "n_steps": ns, "ms": med,
                                     "ns_per_ic_per_step": 1e6 * med / rk, "rk_steps_per_s": rk / (med * 1e-3),
                                     "frac_of_fp64_peak": FLOP_PER_STEP["C1sat"] * rk / (med * 1e-3) / 1e12 / NOMINAL_FP64_TFLOPS,
                                     "lanes": wk["kinfo"]["lanes"]})
        del wk
        torch.cuda.empty_cache()
    # the same curve with the ADAPTIVE solver (the solver of the paper's Fig. 2): Henon-Heiles E = 1/8, SALI,
    # rtol = atol = 1e-12, t = 100
    from paper_2507_00622_b200 import workloads as W
    for side in (32, 64, 128, 256, 512):
        y0 = torch.from_numpy(W.hh_grid(0.125, side, side)).cuda()
        n_ic = y0.shape[1]
        w0 = torch.from_numpy(W.deviation_vectors(n_ic, 2, 4, 0, "unit")).cuda()
        yb, wb, rep = torch.empty_like(y0), torch.empty_like(w0), chs.Report(n_ic, "cuda")

        def prepare():
            yb.copy_(y0)
            wb.copy_(w0)
        wk = dict(prepare=prepare, step_dev=lambda: chs.sali(chs.SYS_HENON_HEILES, None, yb, wb, renorm_every=1, adaptive=True,
                                                             t_end=100.0, rtol=1e-12, atol=1e-12, report=rep))
        prepare()
        wk["step_dev"]()
        ms = timed(torch, flush, wk, 2)
        med = float(np.median(ms))
        att = int(rep.n_accepted.sum().item()) + int(rep.n_rejected.sum().item())
        out["ensemble_size_adaptive"].append({
            "n_ic": n_ic, "t_end": 100.0, "ms": med, "us_per_ic": 1e3 * med / n_ic, "attempts": att,
            "attempts_per_s": att / (med * 1e-3),
            "lanes": chs.kernel_info(chs.SYS_HENON_HEILES, None, chs.WHAT_SALI, k=2, adaptive=True, n_ic=n_ic)["lanes"]})
        del wk, y0, w0, yb, wb
        torch.cuda.empty_cache()
    return out


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    args = parse(argv)
    if args.impl == "reference":
        return run_reference(args)
    plan = launch_plan(args.gpus, os.environ, argv)
    if plan[0] == "error":
        raise SystemExit("bench.py: " + plan[1])
    if plan[0] == "spawn":
        raise SystemExit(subprocess.call(plan[1]))
    _, rank, local, world = plan

    import torch
    import torch.distributed as dist
    from paper_2507_00622_b200 import binding as chs  # raises if the library is missing
    from paper_2507_00622_b200 import probe

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    if local >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} needs GPU {local} but only {torch.cuda.device_count()} are visible")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    wk = make_workload(chs, torch, args, rank, world)
    wl, step_dev, step_e2e, h2d, d2h, kinfo = wk["wl"], wk["step_dev"], wk["step_e2e"], wk["h2d"], wk["d2h"], wk["kinfo"]
    n_ic = wk["n_ic"]
    launches_per_step = 1

    # FP64 FMA peak of this device, measured live (register-only DFMA chains)
    probe.dfma_probe(1000, 148 * 8)
    torch.cuda.synchronize()
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record()
    probe_flop, _ = probe.dfma_probe(400000, 148 * 8)
    pe1.record()
    torch.cuda.synchronize()
    dfma_tflops = probe_flop / (pe0.elapsed_time(pe1) * 1e-3) / 1e12

    with ClockSampler(local) as cs:   # sampling starts before the warm-up so the GPU never idles before the timed region
        for _ in range(max(args.warmup, 0)):
            if "prepare" in wk:
                wk["prepare"]()
            step_dev()
        barrier()
        t_wall = time.perf_counter()
        ms = timed(torch, flush, wk, args.steps)
        barrier()
        t_wall = time.perf_counter() - t_wall
    clocks = cs.summary()
    t_dev = rank_max(sum(ms) * 1e-3, world, "cuda")
    resolve_rk_steps(wl)
    value = aggregate(wl["rk_steps"], world, args.steps, t_dev)

    # end to end: host buffers through the C ABI's host entry point, copies inside the timed region
    for _ in range(max(args.warmup, 1)):
        step_e2e()
    barrier()
    e2e_ms = []
    t0 = time.perf_counter()
    for _ in range(args.steps):
        t1 = time.perf_counter()
        step_e2e()
        e2e_ms.append(1e3 * (time.perf_counter() - t1))
    torch.cuda.synchronize()
    t_e2e = rank_max(time.perf_counter() - t0, world, "cuda")
    e2e_value = aggregate(wl["rk_steps"], world, args.steps, t_e2e)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    label = WORKLOAD_LABEL[args.workload]
    if args.workload == "C2":
        label = ("C2: Henon-Heiles Lagrangian descriptor (arc length), E=1/8, %dx%d grid per GPU, fixed DOP8 h=0.01, "
                 "%d steps forward + %d backward" % (args.side, args.side, wl["n_steps"], wl["n_steps"]))
    full_size = (world == 1 and args.shrink == 1 and args.shrink_ic == 1 and
                 (args.workload != "C2" or (args.side == 1024 and args.n_steps == 5000)))
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {
            "workload": label + (" (shrink %d)" % args.shrink if args.shrink > 1 else ""),
            "n_ic_per_gpu": int(n_ic), "rk_steps_per_step": wl["rk_steps"] * world,
            "fput_n": args.fput_n if args.workload == "F3" else None,
            "l2": "flushed between timed iterations (256 MiB write)",
            "kernel": kinfo,
        },
        "roofline": roofline_entry(args.workload, wl, ms, dfma_tflops, full_size),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step_each": [round(x, 3) for x in e2e_ms]},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
        "wall_s_timed_region": t_wall,
    }
    if "accepted" in wl:
        out["config"]["accepted_steps"], out["config"]["rejected_steps"] = wl["accepted"], wl["rejected"]
    orc = None
    if not args.no_cpu_baseline and world == 1:
        from oracle import chaos_oracle as orc
        orc.build()
        if args.workload in PER_CONFIG:
            out["cpu_baseline"] = cpu_baseline(orc, args.workload, args, target_s=15.0)
    # the other configs, each measured the same way (single GPU, headline workload only)
    names = [c for c in args.configs.split(",") if c]
    if world == 1 and args.workload == "C2" and full_size and names:
        del wk
        torch.cuda.empty_cache()
        per = {}
        with ClockSampler(local) as cs2:
            for name in names:
                if name == "C2":      # the headline itself: same numbers, same shape of entry
                    per[name] = {
                        "workload": label, "n_ic": int(n_ic), "rk_steps": wl["rk_steps"], "ms": float(np.median(ms)),
                        "ms_each": [round(x, 3) for x in ms],
                        "ns_per_step_per_trajectory": 1e6 * float(np.median(ms)) / (2.0 * wl["n_steps"]),
                        "rk_steps_per_s": wl["rk_steps"] / (float(np.median(ms)) * 1e-3),
                        "flop_per_rk_step": FLOP_PER_STEP["C2"],
                        "roofline": roofline_entry("C2", wl, [float(np.median(ms))], dfma_tflops), "kernel": kinfo,
                        "e2e": dict(out["e2e"], ms=float(np.mean(e2e_ms))),
                    }
                    if "cpu_baseline" in out:
                        per[name]["cpu_baseline"] = out["cpu_baseline"]
                    continue
                per[name] = measure_config(chs, torch, flush, args, name, dfma_tflops, orc)
            if not args.no_sweeps:
                out["sweeps"] = run_sweeps(chs, torch, flush, args)
                # the widened rows of SURVEY 8(f), driver-timed in the same line: f-2 LD of neighbouring ICs and
                # the adaptive LD on the C2 grid, f-3 the double pendulum (Fig. 1 shape)
                a3 = argparse.Namespace(**vars(args))
                a3.config_steps = 2
                out["widened"] = {n: measure_config(chs, torch, flush, a3, n, dfma_tflops, None)
                                  for n in ("LDN", "LDA", "F1")}
        out["per_config"] = per
        out["per_config_clocks"] = cs2.summary()
        out["gpu_launches_total"] = (out["gpu_launches"] + sum(2 + args.config_steps + 4 for n in names if n != "C2")
                                     + (0 if args.no_sweeps else 3 * (2 + 2 + 4)))
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
