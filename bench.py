#!/usr/bin/env python
"""bench.py -- FP64 pressure-projection throughput on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W]            this repo's CUDA path
  python bench.py --impl reference [--gpus N] [--steps K] ...    the CPU oracle on the host cores

A "step" is one pass of the whole hot path (divergence -> x/y transforms -> z Thomas solve -> inverse
transforms -> gradient correction) on the C5 workload of BASELINE.json: the 1024x768x512 channel grid,
periodic x/y, Neumann z, tanh-stretched z (a = 1.6), seeded synthetic k^-5/3 + Poiseuille velocity
fields (recipe: DESIGN.md "Synthetic inputs"; stands in for the paper's turbulent-channel data).
One JSON line is printed by rank 0.  For N > 1 every rank runs an independent replica
("replicas only": the path has no exchange step on one GPU).

Order of the run: W warm-up steps; a K-step burst on the cool board (`burst`); SUSTAINED_SECONDS of back-to-back steps
with their own clock record (`sustained`); then EXACTLY K timed steps (`value`, `ms_per_step`, `roofline`), which
therefore sit in the sustained regime a time loop lives in.  `roofline` is the whole step against SURVEY 8(d)'s
112 B/cell; `roofline_kernel` the dominant kernel against its own bytes.  `cpu_baseline` is the oracle on a
1024x768xNZ_SAMPLE slab (the slab `--impl reference` times); `cpu_fft_baseline` the same slab through scipy.fft.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64_projection_throughput"
UNIT = "Gcells/s"
WORKLOAD = "C5: projection step 1024x768x512, PP/PP/NN, tanh z (a=1.6), dt=1e-4"

# algorithmic HBM bytes per cell of each kernel of the current launch sequence
KERNEL_BYTES_PER_CELL = {
    "x_fwd_div": 32.0,     # read u, v, w (24) + write f~ (8)
    "x_fwd": 16.0,
    "y_fwd": 16.0,
    "z_solve": 16.0,
    "y_inv": 16.0,
    "x_inv": 16.0,
    "grad_correct": 56.0,  # read Phi (8) + u, v, w (24), write u, v, w (24)
    "grad_correct_pacc": 72.0,   # the same kernel also doing eq. 2d: + read and write p_acc (16)
    "chkdt": 24.0,         # read u, v, w once
    "face_correct": 0.0,   # O(N^(2/3)) boundary planes
    "z_setup": 0.5,        # writes the N/16 segment-start pivots
}
STEP_MIN_BYTES_PER_CELL = {"projection": 112.0, "poisson": 48.0}   # structural minimum, SURVEY.md 8(d)
NZ_SAMPLE = 64            # planes of the C5 slab both CPU legs time (cpu_baseline of this arm and --impl reference)
SUSTAINED_SECONDS = 5.0   # length of the back-to-back window that precedes the timed steps


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            with open(path) as fh:
                mp = json.load(fh)
            return float(mp["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock / throttle-reason sampler running during the timed region: NVML polled from a thread every ~5 ms
    (nvidia_ml_py), or -- if NVML cannot be loaded -- `nvidia-smi -lms 20` read from a pipe."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []          # (arrival time, sm MHz, max MHz, power W, set of reasons)
        self.t_begin = None
        self.t_end = None
        self.stop_flag = False
        self.source = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            visible = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = self.index
            if visible:
                try:
                    idx = int(visible.split(",")[self.index])
                except Exception:
                    idx = self.index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.nv = pynvml
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.source = "nvml"
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.source = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi"
            self.thread = threading.Thread(target=self._read_smi, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _poll_nvml(self):
        nv = self.nv
        bits = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self.stop_flag:
            try:
                sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                mask = int(get_reasons(self.h))
                self.lines.append((time.time(), sm, self.smax, pw, {n for n, b in bits.items() if mask & b}))
            except Exception:
                pass
            time.sleep(0.005)

    def _read_smi(self):
        for line in self.proc.stdout:
            parts = [p.strip() for p in line.strip().split(",")]
            if len(parts) < 8:
                continue
            try:
                self.lines.append((time.time(), float(parts[1]), float(parts[2]), float(parts[3]),
                                   {n for n, v in zip(self.NAMES, parts[4:8]) if v.lower().startswith("active")}))
            except ValueError:
                continue

    def mark_begin(self):
        self.t_begin = time.time()

    def mark_end(self):
        self.t_end = time.time()

    def stop(self):
        self.stop_flag = True
        if self.source is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no clock source (NVML and nvidia-smi unavailable)"]}
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        slack = 0.02 if self.source == "nvidia-smi" else 0.0
        inside = [l for l in self.lines
                  if self.t_begin is None or (self.t_begin <= l[0] <= (self.t_end or l[0]) + slack)]
        sm = sorted(l[1] for l in inside)
        reasons = set()
        for l in inside:
            reasons |= l[4]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_min_mhz": sm[0] if sm else None,
                "sm_max_mhz": inside[-1][2] if inside else None, "reasons": sorted(reasons), "samples": len(sm),
                "power_w_max": max((l[3] for l in inside), default=None), "source": self.source}


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [d.get("num_threads", 1) for d in threadpool_info() if d.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count() or 1


def time_oracle_sample(nz_sample: int, repeats: int):
    """The CPU oracle, as it stands, on a bounded sample of C5: same nx, ny, domain, bc and stretching
    recipe with nz_sample planes.  Returns (Gcells/s, seconds per step, cells)."""
    import numpy as np
    from oracle import cans_oracle as orc
    from paper_2001_05234_b200 import workloads
    w = workloads.make_workload("C5", device="cpu", n_override=(1024, 768, nz_sample))
    u, v, ww = (w.fields[c].numpy() for c in "uvw")
    dzc, dzf = w.dzc.numpy(), w.dzf.numpy()
    times = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        orc.projection(u, v, ww, w.dt, *w.lengths, w.bc, dzc, dzf)
        times.append(time.perf_counter() - t0)
    return w.cells, times


def cpu_fft_projection(u, v, w, dt, lx, ly, lz, dzc, dzf, workers=-1):
    """A competent CPU restatement of the C5 projection step (PP/PP/NN) -- scipy.fft real transforms over all cores,
    one Thomas sweep vectorised over the (kx, ky) modes -- timed next to the oracle so that the GPU/CPU ratio can also be
    read against an O(n log n) program (the oracle's dense-matrix transforms are O(n^2) on purpose).  Bench tooling: not
    the oracle (tests/test_bench_cpu.py checks it against the oracle) and not the product.
    eq. 2b -> eq. 6 -> eq. 2c; returns (u, v, w, Phi)."""
    import numpy as np
    import scipy.fft as sfft
    nz, ny, nx = u.shape
    dx, dy = lx / nx, ly / ny
    dzf3, dzc_up = dzf[:, None, None], dzc[1:, None, None]
    wlow = np.concatenate([np.zeros((1, ny, nx)), w[:-1]], axis=0)                  # w on the lower wall face is 0
    f = ((u - np.roll(u, 1, axis=2)) / dx + (v - np.roll(v, 1, axis=1)) / dy + (w - wlow) / dzf3) / dt
    fh = sfft.rfft2(f, axes=(1, 2), workers=workers)
    lam_x = -4.0 * np.sin(np.pi * np.arange(nx // 2 + 1) / nx) ** 2 / dx ** 2
    lam_y = -4.0 * np.sin(np.pi * np.arange(ny) / ny) ** 2 / dy ** 2
    lam = lam_y[:, None] + lam_x[None, :]
    a = 1.0 / (dzc[:-1] * dzf); a[0] = 0.0                                          # Neumann: no coupling through a wall
    c = 1.0 / (dzc[1:] * dzf); c[-1] = 0.0
    b = -(a + c)
    lam00 = lam.copy(); lam00[0, 0] = 1.0                                            # the singular mode is solved apart
    cp = np.empty((nz, ny, nx // 2 + 1))
    den = b[0] + lam00
    cp[0] = c[0] / den
    fh[0] /= den
    for k in range(1, nz):
        den = b[k] + lam00 - a[k] * cp[k - 1]
        cp[k] = c[k] / den
        fh[k] = (fh[k] - a[k] * fh[k - 1]) / den
    for k in range(nz - 2, -1, -1):
        fh[k] -= cp[k] * fh[k + 1]
    # kx = ky = 0: singular (pure Neumann column); last unknown pinned to 0, then the dzf-weighted mean removed
    col = (f.sum(axis=(1, 2))).astype(np.float64)
    m = nz - 1
    cc, dd = np.zeros(m), np.zeros(m)
    cc[0], dd[0] = c[0] / b[0], col[0] / b[0]
    for k in range(1, m):
        den = b[k] - a[k] * cc[k - 1]
        cc[k], dd[k] = c[k] / den, (col[k] - a[k] * dd[k - 1]) / den
    x = np.zeros(nz)
    x[m - 1] = dd[m - 1]
    for k in range(m - 2, -1, -1):
        x[k] = dd[k] - cc[k] * x[k + 1]
    x -= np.sum(x * dzf) / np.sum(dzf)
    fh[:, 0, 0] = x
    phi = sfft.irfft2(fh, s=(ny, nx), axes=(1, 2), workers=workers)
    un = u - dt * (np.roll(phi, -1, axis=2) - phi) / dx
    vn = v - dt * (np.roll(phi, -1, axis=1) - phi) / dy
    phiup = np.concatenate([phi[1:], phi[-1:]], axis=0)                             # mirror ghost above the top wall
    wn = w - dt * (phiup - phi) / dzc_up
    return un, vn, wn, phi


def time_cpu_fft_sample(nz_sample: int, repeats: int):
    """cpu_fft_projection on the same slab as time_oracle_sample.  Returns (cells, [seconds])."""
    from paper_2001_05234_b200 import workloads
    w = workloads.make_workload("C5", device="cpu", n_override=(1024, 768, nz_sample))
    u, v, ww = (w.fields[c].numpy() for c in "uvw")
    dzc, dzf = w.dzc.numpy(), w.dzf.numpy()
    times = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        cpu_fft_projection(u, v, ww, w.dt, *w.lengths, dzc, dzf)
        times.append(time.perf_counter() - t0)
    return w.cells, times


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    nz_sample = NZ_SAMPLE
    cells, times = time_oracle_sample(nz_sample, args.warmup + args.steps)
    timed = times[args.warmup:]
    total = sum(timed)
    value = cells * len(timed) / total / 1e9
    sample = (f"oracle.projection on a {1024}x{768}x{nz_sample} slab of the C5 workload per step "
              f"(same domain, bc, tanh recipe; {cells} cells)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(timed),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def time_poisson_config(binding, workloads, torch, name, steps=10, warmup=3):
    """Poisson-only timing of a BASELINE.json config (RHS values do not affect the timing)."""
    w = workloads.make_workload(name, device="cuda", with_fields=False)
    nx, ny, nz = w.n
    plan = binding.plan_for(w)
    f = torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda")
    p = torch.empty_like(f)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for _ in range(warmup):
        p.copy_(f)
        plan.poisson_solve(p)
    for i in range(steps):
        p.copy_(f)
        ev[i][0].record()
        plan.poisson_solve(p)
        ev[i][1].record()
    torch.cuda.synchronize()
    ms = sorted(a.elapsed_time(b) for a, b in ev)
    plan.close()
    med = ms[len(ms) // 2]
    cells = nx * ny * nz
    return {"config": name, "grid": f"{nx}x{ny}x{nz}", "bc": w.bc_str, "ms_median": med, "ms_min": ms[0],
            "gcells_per_s": cells / med / 1e6, "min_bytes": 48.0 * cells}


PAIRS = ("PP", "NN", "DD", "ND", "DN")


def bc_sweep(binding, workloads, torch, steps=5, warmup=2):
    """Every supported boundary-condition combination on the C5 grid (BASELINE.json: "for every supported
    boundary-condition combination"): Poisson solve and projection step for all 5 x 5 x 5 pairs {PP,NN,DD,ND,DN}^3
    (lower 'D' sides with a registered face plane).  Median ms per call, CUDA events."""
    w = workloads.make_workload("C5", device="cuda", with_fields=False)
    nx, ny, nz = w.n
    lx, ly, lz = w.lengths
    f = torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda")
    bufs = [torch.empty_like(f) for _ in range(4)]
    out = {"grid": f"{nx}x{ny}x{nz}", "poisson_ms": {}, "projection_ms": {}}

    def med(fn, reset):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for _ in range(warmup):
            reset(); fn()
        for a, b in ev:
            reset(); a.record(); fn(); b.record()
        torch.cuda.synchronize()
        ms = sorted(a.elapsed_time(b) for a, b in ev)
        return ms[len(ms) // 2]

    for px in PAIRS:
        for py in PAIRS:
            for pz in PAIRS:
                bc = (tuple(px), tuple(py), tuple(pz))
                plan = binding.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, w.dzc, w.dzf)
                key = f"{px}/{py}/{pz}"
                out["poisson_ms"][key] = med(lambda: plan.poisson_solve(bufs[3]), lambda: bufs[3].copy_(f))
                # lower 'D' sides carry a registered face plane (kept alive in `planes` while registered)
                shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
                planes = {d: torch.zeros(shapes[d], dtype=torch.float64, device="cuda")
                          for d, pr in enumerate((px, py, pz)) if pr[0] == "D"}
                for d, t in planes.items():
                    plan.set_lower_face(d, t)

                def reset():
                    for b in bufs[:3]:
                        b.copy_(f)
                out["projection_ms"][key] = med(
                    lambda: plan.projection(bufs[0], bufs[1], bufs[2], bufs[3], 1e-4), reset)
                plan.close()
    pv, jv = list(out["poisson_ms"].values()), list(out["projection_ms"].values())
    out["combinations"] = len(pv)
    out["poisson_ms_min_max"] = [min(pv), max(pv)]
    out["projection_ms_min_max"] = [min(jv), max(jv)]
    # the paper's own GPU transform set (DFT, DCT-II/III, DST-II/III) separately from the mixed pairs
    core = [k for k in out["projection_ms"] if all(p in ("PP", "NN", "DD") for p in k.split("/")[:2])]
    out["projection_ms_min_max_without_mixed_xy"] = [min(out["projection_ms"][k] for k in core),
                                                     max(out["projection_ms"][k] for k in core)]
    return out


def time_step_variants(binding, torch, plan, w, fields, steps=5, warmup=2):
    """The calls around the projection in a time loop, on the C5 workload: cans_projection_step with eq. 2d fused into the
    correction kernel and the chkdt reduction; cans_helmholtz_solve (eq. 3b) with a channel-DNS shift.  Median ms."""
    u0, v0, w0, u, v, ww, p = fields
    pacc = torch.zeros_like(p)
    dti = torch.zeros((1,), dtype=torch.float64, device="cuda")

    def med(fn, reset):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for _ in range(warmup):
            reset(); fn()
        for a, b in ev:
            reset(); a.record(); fn(); b.record()
        torch.cuda.synchronize()
        ms = sorted(a.elapsed_time(b) for a, b in ev)
        return ms[len(ms) // 2]

    def restore():
        u.copy_(u0); v.copy_(v0); ww.copy_(w0)

    out = {}
    out["projection_step_pacc_chkdt_ms"] = med(lambda: plan.projection_step(u, v, ww, p, w.dt, p_acc=pacc, dti=dti), restore)
    out["projection_step_pacc_ms"] = med(lambda: plan.projection_step(u, v, ww, p, w.dt, p_acc=pacc), restore)
    out["projection_step_eq3e_ms"] = med(lambda: plan.projection_step(u, v, ww, p, w.dt, p_acc=pacc, nu_dt_half=4.4e-8), restore)
    out["chkdt_ms"] = med(lambda: plan.chkdt(u, v, ww, dti), lambda: None)
    out["chkdt_gbs"] = 24.0 * w.cells / (out["chkdt_ms"] * 1e-3) / 1e9
    alpha = -2.0 / (0.5 * 1.77e-4 * 1e-3)          # -2/(gamma nu dt): gamma ~ 1/2, nu = 1/5640, dt = 1e-3
    out["helmholtz_solve_ms"] = med(lambda: plan.helmholtz_solve(p, alpha), lambda: p.copy_(u0))
    plan.poisson_solve(p)                           # back to the alpha = 0 pivot table
    torch.cuda.synchronize()
    out["helmholtz_alpha"] = alpha
    del pacc
    return out


def time_paper_grid(binding, workloads, torch, steps=3, warmup=2):
    """Context line: the paper's own grid 1536 x 768 x 576, projection step, same bc / stretching as C5.
    nx = 1536 runs the 3-pass shared-memory transforms (no warp-level kernel for that length)."""
    nx, ny, nz = 1536, 768, 576
    w = workloads.make_workload("C5", device="cuda", with_fields=False, n_override=(nx, ny, nz))
    plan = binding.plan_for(w)
    f = torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda")
    bufs = [torch.empty_like(f) for _ in range(4)]
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for i in range(warmup + steps):
        for b in bufs[:3]:
            b.copy_(f)
        if i >= warmup:
            ev[i - warmup][0].record()
        plan.projection(bufs[0], bufs[1], bufs[2], bufs[3], 1e-4)
        if i >= warmup:
            ev[i - warmup][1].record()
    torch.cuda.synchronize()
    ms = sorted(a.elapsed_time(b) for a, b in ev)
    plan.close()
    med = ms[len(ms) // 2]
    cells = nx * ny * nz
    return {"grid": f"{nx}x{ny}x{nz}", "cells": cells, "projection_ms": med, "gcells_per_s": cells / med / 1e6,
            "note": "paper: 0.1404 s per RK3 step (3 projections + momentum) on 16 V100 (P:L280); context only"}


def max_over_ranks(total_ms, world, device):
    """Replicas only: every rank times its own independent replica; the job time is
    the slowest rank's (all-reduce MAX; NCCL on GPUs, gloo in the CPU test)."""
    if world <= 1:
        return total_ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([total_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gcells_per_s(cells, steps, world, total_ms):
    """Weak scaling: `world` replicas of `cells` cells each, `steps` steps in `total_ms` (max over ranks)."""
    return world * cells * steps / (total_ms * 1e-3) / 1e9


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    from paper_2001_05234_b200 import binding, workloads   # raises if libcans_poisson.so is missing

    peak_gbs, peak_src = load_peaks()
    w = workloads.make_workload("C5", device="cuda")
    nx, ny, nz = w.n
    cells = w.cells
    plan = binding.plan_for(w)
    u0, v0, w0 = (w.fields[c] for c in "uvw")
    u, v, ww = torch.empty_like(u0), torch.empty_like(u0), torch.empty_like(u0)
    p = torch.empty_like(u0)

    def restore():
        u.copy_(u0); v.copy_(v0); ww.copy_(w0)

    # ---- warm-up: W steps, a K-step burst on the still cool board, then SUSTAINED_SECONDS of back-to-back steps ----
    for _ in range(max(args.warmup, 3)):
        restore()
        plan.projection(u, v, ww, p, w.dt)
    torch.cuda.synchronize()
    burst_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in burst_ev:
        restore()
        a.record(); plan.projection(u, v, ww, p, w.dt); b.record()
    torch.cuda.synchronize()
    burst_ms = sorted(a.elapsed_time(b) for a, b in burst_ev)
    burst = {"steps": args.steps, "ms_mean": sum(burst_ms) / len(burst_ms), "ms_median": burst_ms[len(burst_ms) // 2],
             "ms_min": burst_ms[0], "note": "the K steps right after the W warm-up steps, board not yet under sustained load"}
    sustained = None
    if not args.no_sustained:
        # a time loop lives here: steps enqueued back to back (no restore: the projection of a projected field costs the
        # same), one event pair per step, until the window is full; its clock record goes with it
        s_sampler = ClockSampler(local_rank)
        s_sampler.start()
        per = max(burst["ms_median"], 1e-3)
        n_s = int(SUSTAINED_SECONDS * 1e3 / per) + 1
        s_ev = [torch.cuda.Event(enable_timing=True) for _ in range(n_s + 1)]
        torch.cuda.synchronize()
        s_sampler.mark_begin()
        s_ev[0].record()
        for i in range(n_s):
            plan.projection(u, v, ww, p, w.dt)
            s_ev[i + 1].record()
        torch.cuda.synchronize()
        s_sampler.mark_end()
        s_ms = sorted(s_ev[i].elapsed_time(s_ev[i + 1]) for i in range(n_s))
        s_tail = sorted(s_ev[i].elapsed_time(s_ev[i + 1]) for i in range(n_s - max(n_s // 5, 1), n_s))
        sustained = {"steps": n_s, "seconds": s_ev[0].elapsed_time(s_ev[n_s]) * 1e-3, "ms_median": s_ms[n_s // 2],
                     "ms_min": s_ms[0], "ms_max": s_ms[-1], "ms_median_last_fifth": s_tail[len(s_tail) // 2],
                     "clocks": s_sampler.stop()}
        sustained["gcells_per_s_median"] = cells / sustained["ms_median"] / 1e6
        sustained["roofline_frac_median"] = (STEP_MIN_BYTES_PER_CELL["projection"] * cells / (sustained["ms_median"] * 1e-3)
                                             / 1e9 / peak_gbs)

    # ---- timed region: EXACTLY K steps, right behind the sustained window (the board stays in that regime), CUDA events
    #      on the launching stream, per-kernel events inside ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    plan.set_profiling(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kernel_ms = {}
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.mark_begin()
    for i in range(args.steps):
        restore()                      # inputs (12.9 GB) are far larger than L2 (126 MB): every step starts cold
        ev[i][0].record()
        plan.projection(u, v, ww, p, w.dt)
        ev[i][1].record()
        for name, ms in plan.kernel_times():     # waits for this step's kernels only
            kernel_ms.setdefault(name, []).append(ms)
    torch.cuda.synchronize()
    sampler.mark_end()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    plan.set_profiling(False)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    total_ms = max_over_ranks(total_ms, world, "cuda")
    ms_per_step = total_ms / args.steps
    value = whole_job_gcells_per_s(cells, args.steps, world, total_ms)

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (largest share of the step) ----
    kavg = {k: sum(vv) / len(vv) for k, vv in kernel_ms.items()}
    dom = max(kavg, key=kavg.get)
    dom_bytes = KERNEL_BYTES_PER_CELL[dom] * cells
    dom_gbs = dom_bytes / (kavg[dom] * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")     # per-launch DRAM bytes from the committed ncu capture
    if os.path.exists(tpath):
        try:
            with open(tpath) as fh:
                traffic = json.load(fh).get(dom)
        except Exception:
            traffic = None
    roofline_kernel = {"bound": "hbm", "kernel": dom, "achieved": dom_gbs, "peak": peak_gbs, "unit": "GB/s",
                       "frac": dom_gbs / peak_gbs, "traffic": traffic, "peak_source": peak_src,
                       "algorithmic_bytes_per_launch": dom_bytes, "kernel_ms": kavg[dom],
                       "note": "the kernel with the largest share of the step against ITS OWN algorithmic bytes (a kernel-"
                               "quality figure); the SURVEY 8(d) quantity is `roofline`"}
    step_gbs = STEP_MIN_BYTES_PER_CELL["projection"] * cells / (ms_per_step * 1e-3) / 1e9
    step_traffic = None
    if os.path.exists(tpath):
        try:
            with open(tpath) as fh:
                tj = json.load(fh)
            step_traffic = sum(tj[k] for k in kavg if k in tj) if all(k in tj for k in kavg) else None
        except Exception:
            step_traffic = None
    # the whole step against its structural minimum of 112 B/cell (every field read and written once per
    # direction change that cannot be fused away), all kernels of one cans_projection call taken together
    roofline = {"bound": "hbm", "kernel": "whole step: " + " + ".join(kavg), "achieved": step_gbs, "peak": peak_gbs,
                "unit": "GB/s", "frac": step_gbs / peak_gbs, "frac_of_nominal_8TBs": step_gbs / 8000.0,
                "traffic": step_traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": STEP_MIN_BYTES_PER_CELL["projection"] * cells,
                "min_bytes_per_cell": STEP_MIN_BYTES_PER_CELL["projection"],
                "traffic_over_algorithmic": (step_traffic / (STEP_MIN_BYTES_PER_CELL["projection"] * cells)) if step_traffic else None,
                "note": "achieved = 112 B/cell x cells / ms_per_step of the K timed steps (which follow the sustained window); "
                        "traffic = sum over the step's kernels of dram__bytes_read+write from the committed ncu --set full "
                        "captures (profiles/traffic.json), not measured in this run; the dominant kernel alone is roofline_kernel"}
    kernels = {k: {"ms": kavg[k], "share": kavg[k] / sum(kavg.values()),
                   "achieved_gbs": KERNEL_BYTES_PER_CELL[k] * cells / (kavg[k] * 1e-3) / 1e9} for k in kavg}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        n_e2e = min(args.steps, 3)
        hu, hv, hw = (t.cpu().pin_memory() for t in (u0, v0, w0))
        hu0 = hu.clone()
        hp = torch.empty(u0.shape, dtype=torch.float64).pin_memory()
        plan.projection_host(hu, hv, hw, hp, w.dt)          # warm-up (allocates the plan's device buffers)
        t_e2e = 0.0
        for _ in range(n_e2e):
            hu.copy_(hu0)                                     # host-side restore of one field, outside the timing
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            plan.projection_host(hu, hv, hw, hp, w.dt)       # H2D of u,v,w + kernels + D2H of u,v,w,Phi + sync
            t_e2e += time.perf_counter() - t0
        e2e = {"value": cells * n_e2e / t_e2e / 1e9, "unit": UNIT, "h2d_bytes_per_step": 3 * 8 * cells,
               "d2h_bytes_per_step": 4 * 8 * cells, "steps": n_e2e, "ms_per_step": 1e3 * t_e2e / n_e2e,
               "api": "cans_projection_host (pinned host buffers)",
               "note": "PCIe-bound: 22.5 GB cross the host link per step, the kernels are 2-3 % of it"}
        del hu, hv, hw, hp, hu0

    # ---- measured denominators: FP64 FMA rate, HBM rate of the y / z tile access patterns (bare TMA copies) ----
    probes = None
    variants = None
    paper_grid = None
    if not args.no_extra:
        fma = binding.probe_fp64_fma()
        zc = plan.probe_tile_copy(p, 0)
        yc = plan.probe_tile_copy(p, 1)
        zw = plan.probe_tile_copy(p, 2)
        probes = {"fp64_fma_per_s": fma, "fp64_tflops": 2.0 * fma / 1e12,
                  "z_tile_copy_gbs": 16.0 * cells / (zc * 1e-3) / 1e9, "z_tile_copy_ms": zc,
                  "y_tile_copy_gbs": 16.0 * cells / (yc * 1e-3) / 1e9, "y_tile_copy_ms": yc,
                  "z_view_32col_tile_copy_gbs": 16.0 * cells / (zw * 1e-3) / 1e9, "z_view_32col_tile_copy_ms": zw,
                  "note": "bare TMA in/out copy of the field (two buffers, store drained before the refill: a conservative "
                          "ceiling) with the z-solve tiles (16 columns x 512 rows: 128-byte rows, each in another 2 MB page), "
                          "the y-transform tiles (16 doubles x 768 rows, 8 KB apart) and 32-column tiles of the z view "
                          "(256-byte rows): to be read next to the z_solve / y_fwd / y_inv achieved_gbs"}
        variants = time_step_variants(binding, torch, plan, w, (u0, v0, w0, u, v, ww, p))

    # ---- Poisson-only timings of the other configs (context; parity-test cases, not bench lines) ----
    poisson = []
    sweep = None
    if not args.no_extra:
        del u, v, ww, p
        torch.cuda.empty_cache()
        for name in ("C2", "C3", "C4", "C5"):
            r = time_poisson_config(binding, workloads, torch, name)
            r["frac_of_peak"] = r["min_bytes"] / (r["ms_median"] * 1e-3) / 1e9 / peak_gbs
            poisson.append(r)
        sweep = bc_sweep(binding, workloads, torch)
        w.fields.clear()
        del u0, v0, w0
        torch.cuda.empty_cache()
        paper_grid = time_paper_grid(binding, workloads, torch)

    # ---- CPU baseline: the oracle on a bounded sample, host cores of this box ----
    cpu_baseline = None
    cpu_fft = None
    if world == 1 and not args.no_cpu:
        nz_sample = NZ_SAMPLE
        reps = 4
        ccells, times = time_oracle_sample(nz_sample, reps)
        tot = sum(times)
        cpu_baseline = {"value": ccells * reps / tot / 1e9, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                        "method": "numpy + BLAS matmul, naive O(n^2) transforms (the parity oracle as it stands; cores = BLAS threads)",
                        "sample": f"oracle.projection on a 1024x768x{nz_sample} slab of C5 (same domain, bc, tanh recipe; the "
                                  f"slab --impl reference times), {ccells} cells, {reps} calls, {tot:.1f} s wall"}
        # the same slab through an O(n log n) CPU program (scipy.fft on all cores + vectorised Thomas): the fairer CPU figure
        try:
            fcells, ftimes = time_cpu_fft_sample(nz_sample, 5)
            ft = sum(ftimes[1:])
            cpu_fft = {"value": fcells * (len(ftimes) - 1) / ft / 1e9, "unit": UNIT, "cores": os.cpu_count() or 1,
                       "kind": "scipy_fft", "method": "bench.cpu_fft_projection: scipy.fft rfft2/irfft2 (workers = all cores) + "
                       "Thomas vectorised over modes; checked against the oracle in tests/test_bench_cpu.py",
                       "sample": f"the same 1024x768x{nz_sample} slab, {len(ftimes) - 1} calls after one warm-up, {ft:.1f} s wall"}
        except Exception as exc:                    # scipy missing: report, do not fail the GPU line
            cpu_fft = {"unavailable": repr(exc)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "ms_per_step_median": sorted(step_ms)[len(step_ms) // 2],
        "ms_per_step_min": min(step_ms), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "cells": cells, "l2_policy": "inputs (12.9 GB) larger than L2; "
                   "u,v,w restored by device copies between timed steps", "parallelism": f"replicas x{world}"},
        "roofline": roofline,
        "roofline_kernel": roofline_kernel,
        "burst": burst,
        "sustained": sustained,
        "kernels": kernels,
        "cpu_baseline": cpu_baseline,
        "cpu_fft_baseline": cpu_fft,
        "e2e": e2e,
        "gpu_launches": plan.launches_per_projection * args.steps,
        "clocks": clocks,
        "probes": probes,
        "step_variants": variants,
        "poisson_configs": poisson,
        "bc_sweep": sweep,
        "paper_grid": paper_grid,
        "paper_context": "PAPER.md Table 1 (P:L274-284): 0.1404 s per full RK3 time step (3 projections + momentum), "
                         "1536x768x576, 16x V100 DGX-2 -- whole time step on other hardware, not this metric",
    }
    print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the CPU-oracle baseline leg")
    ap.add_argument("--no-extra", action="store_true", help="skip the Poisson-only timings of C2..C5")
    ap.add_argument("--no-sustained", action="store_true", help="skip the back-to-back window before the timed steps")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
