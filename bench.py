#!/usr/bin/env python
"""bench.py -- grid-point RK3 steps per second of the ocfd hot path on B200 (one process per GPU).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A "step" is one production step of the whole hot path on one synthetic workload: Lambda by
ocfd_max_wavespeed (row a9, with its device-to-host read), dt = CFL / Lambda, then one TVD-RK3 step (3 x [ghost fill,
viscous flux + sensor, inviscid x, y, z sweeps, viscous divergence + RK update] + a final ghost fill).  `value_fixed_dt`
is the same K steps without row a9, with one fixed dt (what rounds 1 and 2 reported as `value`).  The default workload is
BASELINE.json's configs[4], the >=100M-point Mach 2.9 ramp grid that north_star's target names; it fits one GPU.
N > 1 runs N independent replicas (north_star: no domain decomposition), value = sum over replicas.
Prints ONE JSON line on rank 0 (contract: see the task statement; extra keys: roofline, cpu_baseline, kernels).
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2209_15333_b200 import workloads as W  # noqa: E402

METRIC = "grid_point_rk3_steps_per_sec"
UNIT = "grid-point RK3 steps/s"

def _with(case, **kw):
    for k, v in kw.items():
        setattr(case, k, v)
    return case


# name -> (generator for the GPU workload, generator for the bounded CPU sample of the same workload, note)
WORKLOADS = {
    "ramp2048x300x256_hybrid": (lambda: W.ramp(), lambda: W.ramp(nx=512, ny=76, nz=32), "BASELINE configs[4]"),
    "plate1024x128x128_weno7": (lambda: W.flat_plate(), lambda: W.flat_plate(nx=256, ny=64, nz=32), "BASELINE configs[3]"),
    "hit256_hybrid": (lambda: W.hit(256, Mt=1.0, seed=20223, scheme="hybrid", nsteps=50),
                      lambda: W.hit(64, Mt=1.0, seed=20223, scheme="hybrid", nsteps=50), "BASELINE configs[2]"),
    "hit128_weno7": (lambda: W.hit(128), lambda: W.hit(64), "BASELINE configs[1]"),
    "tgv32_weno7": (lambda: W.tgv(32), lambda: W.tgv(32), "BASELINE configs[0]"),
    "ramp2048x300x256_weno7": (lambda: W.ramp(scheme="weno7"), lambda: W.ramp(nx=512, ny=76, nz=32, scheme="weno7"),
                               "configs[4] grid with WENO7 everywhere (ALU-bound variant)"),
    "ramp2048x300x256_hybrid_visc8": (lambda: _with(W.ramp(), visc_order=8),
                                      lambda: _with(W.ramp(nx=512, ny=76, nz=32), visc_order=8),
                                      "configs[4] grid with the 8th-order central viscous scheme (SURVEY 8(f) NEXT #3)"),
    "ramp2048x300x256_hybrid_closure": (lambda: _with(W.ramp(), bc_closure=1),
                                        lambda: _with(W.ramp(nx=512, ny=76, nz=32), bc_closure=1),
                                        "configs[4] with the paper's inviscid boundary scheme (SURVEY 8(f) NEXT #1)"),
    "ramp2048x300x256_hybrid_char": (lambda: _with(W.ramp(), char_recon=1),
                                     lambda: _with(W.ramp(nx=512, ny=76, nz=32), char_recon=1),
                                     "configs[4] with reconstruction in characteristic variables (SURVEY 8(f) NEXT #2)"),
    "ramp2048x300x256_weno7_char": (lambda: _with(W.ramp(scheme="weno7"), char_recon=1),
                                    lambda: _with(W.ramp(nx=512, ny=76, nz=32, scheme="weno7"), char_recon=1),
                                    "configs[4] grid, WENO7 everywhere in characteristic variables (ALU-bound)"),
    "ramp2048x300x256_ud7": (lambda: W.ramp(scheme="ud7"), lambda: W.ramp(nx=512, ny=76, nz=32, scheme="ud7"),
                             "configs[4] grid with the linear 7th-order scheme everywhere (no sensor, no flags)"),
    # the hybrid scheme at the flagged fraction the paper quotes ("more than 90 %" linear, i.e. up to 10 %
    # not) and with the three-level thresholds of PAPER.md:L303 (theta2 = 0.1): config-5 grid with a train of 15 weak
    # oblique fronts ahead of the ramp shock (6.3 % of the interfaces flagged: 5.2 % WENO7 + 1.1 % WENO5 with theta2 = 0.1)
    "ramp2048x300x256_hybrid_shocktrain": (lambda: W.ramp(nshocks=16), lambda: W.ramp(nx=512, ny=76, nz=32, nshocks=16),
                                           "configs[4] grid, two-level hybrid, 6.3 % of the interfaces flagged"),
    "ramp2048x300x256_hybrid3_shocktrain": (lambda: W.ramp(nshocks=16, theta2=0.1),
                                            lambda: W.ramp(nx=512, ny=76, nz=32, nshocks=16, theta2=0.1),
                                            "configs[4] grid, three-level hybrid (theta2 = 0.1), 6.3 % flagged"),
    "ramp2048x300x256_hybrid3": (lambda: W.ramp(theta2=0.1), lambda: W.ramp(nx=512, ny=76, nz=32, theta2=0.1),
                                 "configs[4] with the three-level thresholds of PAPER.md:L303"),
    "hit256_hybrid3": (lambda: W.hit(256, Mt=1.0, seed=20223, scheme="hybrid", nsteps=50, theta2=0.1),
                       lambda: W.hit(64, Mt=1.0, seed=20223, scheme="hybrid", nsteps=50, theta2=0.1),
                       "BASELINE configs[2] with the three-level thresholds (SURVEY 8(d))"),
    "shocked256_hybrid3": (lambda: W.shocked_periodic(256, steep=36.0), lambda: W.shocked_periodic(64, steep=9.0),
                           "periodic 256^3 box with steep fronts, three-level hybrid, about 7 % flagged"),
    # the paper's own timing grids (section 5.3: 280^3 per GPU; L642-651 Table 7: 200^3), periodic, WENO7
    # (the paper times WENO-SYMBO, whose constants are not in the container: context, not a like-for-like comparison)
    "periodic200_weno7": (lambda: W.hit(200, nsteps=10), lambda: W.hit(64), "PAPER.md Table 7 grid (200^3), WENO7"),
    "periodic280_weno7": (lambda: W.hit(280, nsteps=10), lambda: W.hit(64), "PAPER.md section 5.3 grid (280^3), WENO7"),
    "periodic280_hybrid": (lambda: W.hit(280, Mt=1.0, seed=20223, scheme="hybrid", nsteps=10),
                           lambda: W.hit(64, Mt=1.0, seed=20223, scheme="hybrid"), "280^3, hybrid scheme"),
    "ramp512x76x32_hybrid": (lambda: W.ramp(nx=512, ny=76, nz=32), lambda: W.ramp(nx=512, ny=76, nz=32), "small twin"),
    "ramp1024x152x64_hybrid": (lambda: W.ramp(nx=1024, ny=152, nz=64), lambda: W.ramp(nx=512, ny=76, nz=32),
                               "mid-size twin (ncu captures)"),
    "ramp1024x152x64_weno7": (lambda: W.ramp(nx=1024, ny=152, nz=64, scheme="weno7"),
                              lambda: W.ramp(nx=512, ny=76, nz=32, scheme="weno7"), "mid-size twin, WENO7 everywhere"),
}
DEFAULT_WORKLOAD = "ramp2048x300x256_hybrid"

# Peaks: HBM from MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback; fp64 from the committed
# DFMA probe (profiles/fp64_peak_r01.md): 34.2 TFLOP/s sustained on this pool's B200 (nominal 148 SM x 64 lanes x 2 x
# 1.965 GHz = 37.2).  MEASURED_PEAKS.json has no fp64 entry, so every fp64 fraction is also quoted against the nominal
# figure and against 148 x 64 x 2 x the SM clock sampled during the timed region.
FP64_PEAK_TFLOPS = 34.2
FP64_NOMINAL_TFLOPS = 37.2
FP64_FLOPS_PER_CLOCK = 148 * 64 * 2
HBM_FALLBACK_GBS = 6650.0


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback"


# ----------------------------------------------------------------------------------------------------------
# Algorithmic work per interior point and launch of each kernel class.  Bytes count every
# field the kernel must read or write once; flops follow the operation counts of the formulas.
def algorithmic(case, flag_hist=None):
    hyb = case.scheme == "hybrid"
    met3d = case.grid_kind == "curvilinear" and case.metrics[0].shape[0] > 1
    P = float(np.prod(case.padded_shape)) / case.npoints            # padded / interior points
    rec = {"ud7": 13.0, "weno7": 146.0, "weno5": 74.0}
    if hyb:
        h = np.array(flag_hist if flag_hist is not None else [1.0, 0.0, 0.0], dtype=float)
        h = h / h.sum()
        fl_rec = h[0] * rec["ud7"] + h[1] * rec["weno7"] + h[2] * rec["weno5"]
    else:
        fl_rec = rec[case.scheme]
    prim_flops = 30.0                   # row a2 inside a consumer: 1/rho, u, v, w, p, c (or T)
    inv_flops = 10 * fl_rec + 5 + 140 + 15 + prim_flops
    th = 8 if hyb else 0
    m_inv = 40 if met3d else 0          # k1, k2, k3, sigma, J of one direction (z-extruded grids: L2-resident planes)
    state = 40                          # the five conserved fields (no primitive field exists in HBM)
    out = {
        "ghost_fill": (0.0, 0.0),
        "shock_sensor": (40.0 + 8.0, 25.0 + prim_flops),      # stand-alone form (runs without viscous terms)
        # one launch per direction: x writes dU, y / z add into it
        # (TMA reduce at the L2: dU still crosses HBM in and out)
        "inviscid_x": (state + th + m_inv + 40, inv_flops),
        "inviscid_y": (state + th + m_inv + 80, inv_flops),
        "inviscid_z": (state + th + m_inv + 80, inv_flops),
        # a6 (+ a3 for the hybrid scheme: theta is written by this kernel, its inputs are already staged)
        "viscous_flux": (40 + 96 + th + (80 if met3d else 0), 240.0 + prim_flops + (25.0 if hyb else 0.0)),
        # a7 + a8 fused (inside ocfd_rk3_step), rotating state buffers: R Fv 96 + dU 40 + U 40 (+ U^n 40 in stages 2 and
        # 3), W U 40: 216 B in stage 1, 256 B in stages 2 and 3; the figure is the mean over the three launches of a step
        "viscous_div": ((216.0 + 256.0 + 256.0) / 3.0 + (8 if met3d else 0), 125.0 + 20.0),
        "rk3_update": (160.0, 20.0),
        "max_wavespeed": (40.0 + (80 if met3d else 0), 45.0),
        "check_state": (40.0, 12.0),
    }
    return out


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU during the timed region (NVML)."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_steps(case, nsteps, warmup):
    """Time the CPU oracle, as it stands, on `case`: returns (points*steps/s, seconds, threads)."""
    from oracle.oracle import Oracle
    o = Oracle(case)
    U = o.fill_ghosts(case.U0.copy())
    dt = case.cfl / o.max_wavespeed(U)
    for _ in range(warmup):
        o.rk3_step(U, dt)
    t0 = time.perf_counter()
    for _ in range(nsteps):                 # the same production step the CUDA arm times: row a9, dt = CFL/Lambda, RK3
        dt = case.cfl / o.max_wavespeed(U)
        o.rk3_step(U, dt)
    t = time.perf_counter() - t0
    threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return case.npoints * nsteps / t, t, threads


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    gen, twin, note = WORKLOADS[args.workload]
    case = twin()
    n_warm = min(args.warmup, 1)            # the oracle needs no warm-up beyond one step (page faults, OpenMP pool)
    val, t, threads = oracle_steps(case, args.steps, n_warm)
    sample = f"{case.name} twin of {args.workload}, {args.steps} production steps (max wavespeed + RK3), full oracle path"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": n_warm, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "note": note, "sample": sample, "warmup_requested": args.warmup},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(x, world, device="cpu"):
    """Max of a per-rank scalar over all ranks (NCCL on the GPU box, gloo in the CPU tests); identity for one rank."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(seconds_local, points_per_rank, steps, world, device="cpu"):
    """Replicas only: every rank advances its own copy of the workload, no data-path collective;
    the job's throughput is all ranks' grid-point steps over the slowest rank's time."""
    return world * points_per_rank * steps / max_over_ranks(seconds_local, world, device)


def sensor_decisions(th_ref, fl_ref, fl_gpu, theta1, theta2, band=1e-12):
    """Per-interface scheme decisions of the CUDA path against the reference's: fl_*[d] are padded byte fields whose entry
    at point s is the scheme of interface s+1/2 along direction d (s = -1 .. n-1 on interior lines); Theta of an
    interface is the larger theta of its two points.  Returns (mismatches farther than `band` from a threshold,
    interfaces within `band` of one, interfaces, histogram of the reference's decisions)."""
    ng = 4
    bad = near = total = 0
    hist = np.zeros(3, dtype=np.int64)
    for d in range(3):
        left = [slice(ng, -ng)] * 3
        right = [slice(ng, -ng)] * 3
        left[2 - d] = slice(ng - 1, -ng)
        right[2 - d] = slice(ng, -ng + 1)
        left, right = tuple(left), tuple(right)
        Th = np.maximum(th_ref[left], th_ref[right])
        close = np.abs(Th - theta1) <= band
        if np.isfinite(theta2):
            close |= np.abs(Th - theta2) <= band
        differ = fl_gpu[d][left] != fl_ref[d][left]
        bad += int((differ & ~close).sum())
        near += int(close.sum())
        total += differ.size
        hist += np.bincount(fl_ref[d][left].ravel(), minlength=3)[:3]
    return bad, near, total, hist


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2209_15333_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gen, twin, note = WORKLOADS[args.workload]
    t_gen = time.perf_counter()
    case = gen()
    t_gen = time.perf_counter() - t_gen
    s = B.Solver(case, device=f"cuda:{local}")
    for kv in args.tune:
        k, v = kv.split("=")
        s.set_tuning(k, int(v))
    U0_host = torch.from_numpy(case.U0)
    U = U0_host.to(s.device)
    s.fill_ghosts(U)
    lam = s.max_wavespeed(U)
    dt = case.cfl / lam
    flag_hist = None
    if case.scheme == "hybrid":
        _, fl = s.debug_sensor(U)
        flag_hist = torch.bincount(fl[fl < 3].flatten().to(torch.int64), minlength=3).cpu().numpy()
        del fl

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        s.rk3_step(U, dt)
    barrier()
    # ---- K steps with one fixed dt (rows a1-a8 only: the quantity rounds 1 and 2 reported as `value`), kept as
    # `value_fixed_dt` for continuity
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(s.stream)
    for _ in range(args.steps):
        s.rk3_step(U, dt)
    f1.record(s.stream)
    barrier()
    ms_fixed = f0.elapsed_time(f1)
    # ---- timed region: K PRODUCTION steps -- row a9 every step (Lambda by ocfd_max_wavespeed, its device-to-host read
    # and stream synchronisation included), dt = CFL / Lambda, then rows a1-a8; CUDA events on the launch stream,
    # per-kernel events inside the library
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s.timing(True)
    n0 = s.launch_count()
    with ClockSampler(local) as clk:
        e0.record(s.stream)
        for _ in range(args.steps):
            dt = case.cfl / s.max_wavespeed(U)
            s.rk3_step(U, dt)
        e1.record(s.stream)
        barrier()
    ms = e0.elapsed_time(e1)
    launches = s.launch_count() - n0
    per_kernel = s.timing_read()
    s.timing(False)
    finite = bool(torch.isfinite(U).all().item())
    flag_hist_end = None
    if case.scheme == "hybrid":     # after the warm-up and timed steps (outside the timed region)
        _, fl = s.debug_sensor(U)
        flag_hist_end = torch.bincount(fl[fl < 3].flatten().to(torch.int64), minlength=3).cpu().numpy()
        del fl
    ms_all = max_over_ranks(ms, world, s.device)
    value = whole_job_value(ms * 1e-3, case.npoints, args.steps, world, s.device)
    value_fixed = whole_job_value(ms_fixed * 1e-3, case.npoints, args.steps, world, s.device)
    ms_fixed_all = max_over_ranks(ms_fixed, world, s.device)

    # ---- end to end through the C ABI with HOST buffers: H2D + step + D2H inside the timed region, every step
    n_e2e = max(1, args.steps)
    Uh = torch.empty(U0_host.shape, dtype=torch.float64, pin_memory=True)
    Uh.copy_(U.cpu())
    s.rk3_steps_host(Uh, U, dt, 1)          # warm-up of the copy path
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        s.rk3_steps_host(Uh, U, dt, 1)      # synchronises the stream before returning
    barrier()
    t_e2e = time.perf_counter() - t0
    e2e_value = whole_job_value(t_e2e, case.npoints, n_e2e, world, s.device)
    nbytes = int(Uh.numel() * 8)

    # ---- optional: the same fixed-dt steps replayed from a CUDA graph (one graph launch per step instead of 27 kernel
    # launches), in a second context on a stream of its own (the legacy default stream cannot be captured)
    graph = None
    if args.graph:
        gstream = torch.cuda.Stream()
        with torch.cuda.stream(gstream):
            sg = B.Solver(case, device=f"cuda:{local}", stream=gstream)
            V = U.clone()
            for _ in range(3):
                sg.rk3_step(V, dt)
            gstream.synchronize()
            cg = torch.cuda.CUDAGraph()
            with torch.cuda.graph(cg, stream=gstream):
                sg.rk3_step(V, dt)
            for _ in range(3):
                cg.replay()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gstream)
            for _ in range(args.steps):
                cg.replay()
            g1.record(gstream)
            gstream.synchronize()
            ms_graph = g0.elapsed_time(g1)
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(gstream)
            for _ in range(args.steps):
                sg.rk3_step(V, dt)
            p1.record(gstream)
            gstream.synchronize()
            ms_plain = p0.elapsed_time(p1)
            sg.close()
        graph = {"ms_per_step_graph_replay": ms_graph / args.steps, "ms_per_step_plain_launches": ms_plain / args.steps,
                 "value_graph_replay": case.npoints * args.steps / (ms_graph * 1e-3), "unit": UNIT,
                 "note": "fixed dt, rows a1-a8, one CUDA-graph launch per step; this rank only"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, from the library's per-launch CUDA events over the timed region
    hbm_peak, peak_src = peaks()
    alg = algorithmic(case, flag_hist)
    tot_kernel_ms = sum(v[0] for k, v in per_kernel.items())
    clk_mhz = clk.summary()["sm_mhz"]
    kern = {}
    for name, (kms, n) in per_kernel.items():
        if n == 0:
            continue
        by, fl = alg[name]
        per_launch_ms = kms / n
        gbs = by * case.npoints / (per_launch_ms * 1e-3) / 1e9
        tfl = fl * case.npoints / (per_launch_ms * 1e-3) / 1e12
        kern[name] = {"ms_per_launch": per_launch_ms, "launches_per_step": n / args.steps, "share": kms / tot_kernel_ms,
                      "alg_GBs": gbs, "alg_TFLOPs": tfl, "frac_hbm": gbs / hbm_peak, "frac_fp64": tfl / FP64_PEAK_TFLOPS,
                      "frac_fp64_nominal": tfl / FP64_NOMINAL_TFLOPS,
                      "frac_fp64_at_sampled_clock": (tfl / (FP64_FLOPS_PER_CLOCK * clk_mhz * 1e-6)) if clk_mhz else None}
    top = max(kern, key=lambda k: kern[k]["share"])
    kt = kern[top]
    if kt["frac_fp64"] > kt["frac_hbm"]:
        roof = {"kernel": top, "bound": "alu", "achieved": kt["alg_TFLOPs"], "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": kt["frac_fp64"], "frac_nominal_37.2": kt["frac_fp64_nominal"],
                "frac_at_sampled_clock": kt["frac_fp64_at_sampled_clock"],
                "peak_source": "fp64 DFMA probe (profiles/fp64_peak_r01.md)"}
    else:
        roof = {"kernel": top, "bound": "hbm", "achieved": kt["alg_GBs"], "peak": hbm_peak, "unit": "GB/s",
                "frac": kt["frac_hbm"], "peak_source": f"MEASURED_PEAKS.json ({peak_src})"}
    roof["traffic"] = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        try:
            roof["traffic"] = json.load(open(tpath)).get(args.workload, {}).get(top)
        except Exception:
            pass

    # ---- the oracle timed on this box's host cores, bounded sample of the same workload
    cpu = None
    sensor_parity = None
    if world == 1 and not args.no_cpu_baseline:
        tw = twin()
        from oracle.oracle import Oracle  # noqa: F401  (cpu_baseline leg: the one place bench.py may run the oracle)
        rate, _, threads = oracle_steps(tw, 1, 1)
        nst = int(max(1, min(50, round(12.0 * rate / tw.npoints))))
        rate, tsec, threads = oracle_steps(tw, nst, 0)
        cpu = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"{tw.name} (twin of the workload, same generator), {nst} production steps (max wavespeed + RK3), {tsec:.1f} s"}
        if case.scheme == "hybrid":
            # north_star: sensor decisions of the CUDA path against the oracle's on the WHOLE grid of this workload;
            # interfaces within 1e-12 of a threshold are counted and reported, the others must agree
            o = Oracle(case)
            U0 = o.fill_ghosts(case.U0.copy())
            th_ref = o.sensor(U0)
            fl_ref = [o.flags(th_ref, d) for d in range(3)]
            _, fl = s.debug_sensor(s.to_device(U0))
            bad, inband, total, hist = sensor_decisions(th_ref, fl_ref, fl.cpu().numpy(), case.theta1, case.theta2)
            sensor_parity = {"interfaces": total, "mismatches_outside_1e-12_band": bad, "within_1e-12_of_a_threshold": inband,
                             "oracle_hist_ud7_weno7_weno5": [int(v) for v in hist], "state": "initial field, ghosts filled"}
            del fl, th_ref, fl_ref, U0

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_all / args.steps, "higher_is_better": True, "scaling": "weak",
        "step": "production step: ocfd_max_wavespeed + dt = CFL/Lambda + ocfd_rk3_step, every step",
        "value_fixed_dt": value_fixed, "ms_per_step_fixed_dt": ms_fixed_all / args.steps,
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "note": note, "grid": [case.nx, case.ny, case.nz], "points": case.npoints,
                   "scheme": case.scheme, "grid_kind": case.grid_kind, "dt": dt, "cfl": case.cfl,
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas",
                   "cache": "inputs larger than L2 (state 5 fields x %.0f MB)" % (np.prod(case.padded_shape) * 8 / 1e6),
                   "hybrid_flag_hist_ud7_weno7_weno5": None if flag_hist is None else [int(v) for v in flag_hist],
                   "hybrid_flag_hist_after_steps": None if flag_hist_end is None else [int(v) for v in flag_hist_end],
                   "input_generation_s": t_gen, "finite": finite},
        "clocks": clk.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "steps": n_e2e, "api": "ocfd_rk3_steps_host (pinned host buffer)"},
        "gpu_launches": int(launches),
        "roofline": roof,
        "cpu_baseline": cpu,
        "sensor_parity": sensor_parity,
        "graph": graph,
        "kernels": kern,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--graph", action="store_true",
                    help="also time the fixed-dt steps replayed from a CUDA graph (extra key `graph`; for launch-bound grids)")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="launch-shape knob passed to ocfd_set_tuning (A/B measurements)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
