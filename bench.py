#!/usr/bin/env python3
"""bench.py -- throughput of the hot path on the workload BASELINE.json's metric is quoted on.

Workload (BASELINE.json configs[1], "C2"): Henon-Heiles arc-length Lagrangian descriptor,
E = 1/8, 1024 x 1024 energy-fitted grid of (y, py) on the x = 0 section, forward and backward
fixed-step DOP8, h = 0.01, |t| = 50 (5000 steps per direction), FP64.  One "step" of this
benchmark = one pass of the whole hot path over that batch = 2 * 1048576 * 5000 RK-steps,
one kernel launch.  Metric: trajectory RK-steps/sec.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C2|C1sat]

N > 1 (torchrun): every rank integrates its own 1024 x 1024 block of rows of a (1024 N) x 1024
grid (weak scaling, no data-path collective: trajectories are independent).
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "trajectory RK-steps/sec (FP64, incl. variational eqs)"
UNIT = "RK-steps/s"
# algorithmic FP64 flop per RK-step of the formulation that runs
FLOP_PER_STEP = {"C2": 640.0, "C1sat": 1216.0, "C3": 1812.0, "C4": 4213.0, "C5": 8492.0, "F3": None, "F1": None}
WORKLOAD_LABEL = {
    "C1sat": "C1sat: Henon-Heiles fixed-step SALI kernel of configs[0] (h=0.01, renormalised every step) on a --sali-side^2 grid, --sali-steps steps",
    "C3": "C3: Henon-Heiles adaptive DOP8(5) rtol=atol=1e-12, 512x512 grid at E=1/6, t=1000, SALI (RK-step = attempted step)",
    "C4": "C4: 3-DoF coupled oscillators, 65536 ICs, full Lyapunov spectrum (6 vectors, MGS every 10 steps), h=0.01, 1e5 steps",
    "C5": "C5: FPUT-beta N=8, 65536 ICs, GALI_4 (renormalised every 10 steps), h=0.05, 2e4 steps",
    "F1": "F1 (shape of PAPER.md Fig. 1): dimensionless double pendulum (sigma = alpha = 1), random ICs, t = 1000, fixed h = 0.01 or adaptive rtol = atol = 1e-9",
    "F3": "F3 (shape of PAPER.md Fig. 3): FPUT-beta chain, random ICs, GALI_4, adaptive DOP8(5) rtol=atol=1e-8, t=1000",
}
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12  # 37.2


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=["C2", "C1sat", "C3", "C4", "C5", "F3", "F1"])
    ap.add_argument("--f1-adaptive", action="store_true", help="F1: adaptive DOP8(5) instead of fixed step")
    ap.add_argument("--shrink", type=int, default=1, help="C3/C4/C5/F3: divide the horizon (profiling runs)")
    ap.add_argument("--shrink-ic", type=int, default=1, help="C3/C4/C5: divide the ensemble (profiling runs)")
    ap.add_argument("--side", type=int, default=1024, help="grid side per rank (C2)")
    ap.add_argument("--n-steps", type=int, default=5000, help="DOP8 steps per direction (C2)")
    ap.add_argument("--sali-side", type=int, default=512, help="C1sat: grid side per rank")
    ap.add_argument("--sali-steps", type=int, default=2000, help="C1sat: DOP8 steps")
    ap.add_argument("--fput-n", type=int, default=8, help="F3: chain length (4, 8, 16, 32)")
    ap.add_argument("--n-ic", type=int, default=1000, help="F3: ensemble size (PAPER.md:129: 10^3 random ICs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tune", type=int, default=0, help="development: kernel variant knob (chaoticus_set_option)")
    return ap.parse_args()


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


def workload_inputs(args, rank, world):
    from paper_2507_00622_b200 import workloads as W
    if args.workload == "C2":
        side = args.side
        y0 = W.hh_grid(0.125, side * world, side, i_range=(rank * side, (rank + 1) * side))
        return dict(y0=y0, h=0.01, n_steps=args.n_steps, rk_steps=2.0 * y0.shape[1] * args.n_steps)
    # C1sat: the fixed-step SALI kernel of configs[0] on a saturating ensemble
    side = args.sali_side
    y0 = W.hh_grid(0.125, side * world, side, i_range=(rank * side, (rank + 1) * side))
    w0 = W.deviation_vectors(y0.shape[1], 2, 4, 0, "unit")
    return dict(y0=y0, w0=w0, h=0.01, n_steps=args.sali_steps, rk_steps=1.0 * y0.shape[1] * args.sali_steps)


def oracle_sample(orc, args, target_s):
    """A sub-grid of the C2 grid (every k-th row and column, full horizon) sized from a short
    calibration run so that the oracle, as it stands, needs about target_s seconds on it."""
    from paper_2507_00622_b200 import workloads as W
    cores = orc.default_threads()
    yc = W.hh_grid(0.125, 64, 64)
    orc.ld(0, None, yc[:, :64].copy(), 0.0, 0.01, 10, precision="f64", threads=cores)  # thread start-up
    t = time.perf_counter()
    orc.ld(0, None, yc, 0.0, 0.01, 300, precision="f64", threads=cores)
    rate = 2.0 * 4096 * 300 / (time.perf_counter() - t)
    sub = int(np.sqrt(max(rate * target_s / (2.0 * args.n_steps), 256.0)))
    sub = max(16, min(sub, args.side))
    idx = np.unique(np.linspace(0, args.side - 1, sub).round().astype(int))
    rows = [W.hh_grid(0.125, args.side, args.side, i_range=(int(i), int(i) + 1))[:, idx] for i in idx]
    return np.ascontiguousarray(np.concatenate(rows, axis=1)), len(idx), cores


def run_reference(args):
    """The CPU oracle, as it stands, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import chaos_oracle as orc
    from paper_2507_00622_b200 import workloads as W
    orc.build()
    y0, sub, cores = oracle_sample(orc, args, target_s=120.0 / max(1, args.steps + args.warmup))
    n_steps = args.n_steps
    times = []
    for it in range(args.warmup + args.steps):
        t = time.perf_counter()
        orc.ld(0, None, y0, 0.0, 0.01, n_steps, precision="f64", threads=cores)
        dt = time.perf_counter() - t
        if it >= args.warmup:
            times.append(dt)
    rk = 2.0 * y0.shape[1] * n_steps
    val = rk * len(times) / sum(times)
    sample = f"{sub}x{sub} sub-grid of the {args.side}x{args.side} grid, full horizon ({n_steps} steps x 2 directions)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "C2: Henon-Heiles LD, E=1/8, fixed DOP8 h=0.01, fwd+bwd (CPU oracle on a bounded sample)",
                   "n_ic_sample": int(y0.shape[1]), "n_steps_per_direction": n_steps},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def make_workload(chs, torch, args, rank, world):
    """Device-resident inputs + the two step closures (device pointers / host buffers) of a workload."""
    from paper_2507_00622_b200 import workloads as W
    HH = chs.SYS_HENON_HEILES
    name = args.workload
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
    if name in ("C2", "C1sat"):
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
    # the other workloads advance y, w in place: every step starts from a fresh device copy made
    # OUTSIDE the timed events (prepare), so only the library's kernel is timed
    if name == "C1sat":
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


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2507_00622_b200 import binding as chs  # raises if the library is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.tune:
        chs.set_option("tune", args.tune)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    wk = make_workload(chs, torch, args, rank, world)
    wl, step_dev, step_e2e, h2d, d2h, kinfo = wk["wl"], wk["step_dev"], wk["step_e2e"], wk["h2d"], wk["d2h"], wk["kinfo"]
    n_ic = wk["n_ic"]
    launches_per_step = 1

    def timed(fn, n):
        """n iterations, each bracketed by CUDA events on the launching stream, L2 flushed between."""
        ms = []
        for _ in range(n):
            flush.fill_(1)
            if "prepare" in wk:
                wk["prepare"]()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        return ms

    # FP64 FMA peak of this device, measured live (register-only DFMA chains)
    from paper_2507_00622_b200 import probe
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
        ms = timed(step_dev, args.steps)
        barrier()
        t_wall = time.perf_counter() - t_wall
    clocks = cs.summary()
    t_dev = sum(ms) * 1e-3
    if world > 1:
        tt = torch.tensor([t_dev], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_dev = tt.item()
    if wl["rk_steps"] is None:   # adaptive: one RK-step = one ATTEMPTED step (accepted + rejected), counted by the kernel
        rp = wl["report"]
        wl["rk_steps"] = float((rp.n_accepted.sum() + rp.n_rejected.sum()).item())
        wl["accepted"], wl["rejected"] = int(rp.n_accepted.sum().item()), int(rp.n_rejected.sum().item())
    value = wl["rk_steps"] * world * args.steps / t_dev

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
    t_e2e = time.perf_counter() - t0
    if world > 1:
        tt = torch.tensor([t_e2e], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_e2e = tt.item()
    e2e_value = wl["rk_steps"] * world * args.steps / t_e2e

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    flop = FLOP_PER_STEP[args.workload]
    achieved = (flop * wl["rk_steps"] / (np.mean(ms) * 1e-3) / 1e12) if flop else None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {
            "workload": ("C2: Henon-Heiles Lagrangian descriptor (arc length), E=1/8, %dx%d grid per GPU, "
                         "fixed DOP8 h=0.01, %d steps forward + %d backward" % (args.side, args.side, wl["n_steps"], wl["n_steps"]))
            if args.workload == "C2" else WORKLOAD_LABEL[args.workload] + (" (shrink %d)" % args.shrink if args.shrink > 1 else ""),
            "n_ic_per_gpu": int(n_ic), "rk_steps_per_step": wl["rk_steps"] * world,
            "fput_n": args.fput_n if args.workload == "F3" else None,
            "l2": "flushed between timed iterations (256 MiB write)",
            "kernel": kinfo,
        },
        "roofline": {
            "bound": "alu", "achieved": achieved, "peak": NOMINAL_FP64_TFLOPS, "unit": "TFLOP/s",
            "frac": (achieved / NOMINAL_FP64_TFLOPS) if achieved else None,
            # DRAM bytes per launch from the ncu --set full capture of this kernel at this size
            # (profiles/r01_ld_kernel_ncu.md: 33.70 MB read + 0.06 MB written; algorithmic 48 MiB, the
            # 16 MiB of results were still in L2 when the kernel ended); other workloads: not captured
            "traffic": 33752832 if (args.workload == "C2" and args.side == 1024 and world == 1) else None,
            "peak_source": "nominal: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz (DESIGN.md Roofline)",
            "measured_dfma_tflops": dfma_tflops, "frac_of_measured_dfma": (achieved / dfma_tflops) if achieved else None,
            "flop_per_rk_step": flop, "kernel_ms": float(np.mean(ms)),
        },
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step_each": [round(x, 3) for x in e2e_ms]},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
        "wall_s_timed_region": t_wall,
    }
    if "accepted" in wl:
        out["config"]["accepted_steps"], out["config"]["rejected_steps"] = wl["accepted"], wl["rejected"]
    if not args.no_cpu_baseline and world == 1 and args.workload == "C2":
        from oracle import chaos_oracle as orc
        orc.build()
        ys, sub, cores = oracle_sample(orc, args, target_s=15.0)
        t0 = time.perf_counter()
        orc.ld(0, None, ys, 0.0, 0.01, wl["n_steps"], precision="f64", threads=cores)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {
            "value": 2.0 * ys.shape[1] * wl["n_steps"] / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{sub}x{sub} sub-grid of the same grid, full horizon, {dt:.1f} s"}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
