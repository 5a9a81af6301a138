#!/usr/bin/env python
"""bench.py -- Mcell/s per fp64 pressure projection (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

A step = one whole projection (divergence -> x/y transforms -> z tridiagonal -> inverse
transforms -> velocity/pressure correction) through the C ABI
of libfsei.so on one batch of seeded synthetic input.  At N = 1 the workload is BASELINE.json
configs[3] (1024x1024x768, the size the north-star target is quoted on; it fits one GPU).
The path is single-GPU ("replicas only"): for N > 1 every rank runs an
independent replica and `value` is the sum over ranks / max-over-ranks time.

`--impl reference` times the CPU oracle (as it stands, `double` build) on the same full-size
workload (at most 3 timed projections of ~12 s each); rank 0 only.

Prints ONE JSON line.
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

METRIC = "Mcell/s per fp64 pressure projection"
UNIT = "Mcell/s"
# algorithmic bytes per cell per launch of each kernel = the bytes that launch has to MOVE:
# fields read + fields written + the reciprocal-pivot table where a kernel streams it.  `achieved` figures are
# computed from these, so they can never exceed the copy bandwidth; the unfused 7-kernel yardstick of SURVEY.md
# sec. 8(d) (184 B/cell) is reported separately as `unfused_equivalent_GBps`.
ALGO_BYTES_PER_CELL = {
    "divergence": 32.0, "x_forward": 16.0, "div_x_forward": 32.0, "y_forward": 16.0, "z_direct": 36.0,
    "z_paired": 32.0, "y_inverse": 16.0, "x_inverse": 16.0, "project": 72.0, "z_gauge": 0.0,
    # fused path: spectrum in + out (16) + one reciprocal pivot per complex element (4; 8 on Neumann grids)
    "yz_forward": 20.0, "yz_backward": 20.0,
    # fluid substep: u,v,w,p + 3 Hprev in, 3 H + 3 rhs out; generic sweeps in place,
    # forward + backward pass each (the z sweep also reads and writes the velocity component)
    "explicit_terms": 104.0, "visc_x": 32.0, "visc_y": 32.0, "visc_z": 40.0, "visc_factor": 0.0,
    # fast viscous family, three components per launch: rhs -> d' in place (3 x 16); d' + q in, q out (3 x 24)
    "visc_xz": 48.0, "visc_zy": 72.0, "ib_mls": 0.0, "ib_apply": 0.0,
}
A_REF = 184.0          # unfused reference accounting of one projection, B/cell
SLAB_NY = 64           # single-thread CPU leg: the workload's grid with ny cut to this many rows


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def _ncu_traffic(cfg: int, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the newest committed
    `ncu --set full` capture (profiles/*_traffic.csv; the .md beside it names the command)."""
    import glob
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        with open(path) as f:
            for line in f.read().splitlines()[1:]:
                c = line.split(",")
                if len(c) >= 4 and c[0] == f"cfg{cfg}" and c[1] == kernel:
                    best = float(c[2]) + float(c[3])
    return best


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.th = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.2] or [r for _, r in self.rows]
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(ms: float, device=None) -> float:
    """Device time of the slowest rank (the contract's max over ranks); identity on one rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(cells: int, world: int, ms_step: float) -> float:
    """Whole-job Mcell/s of `world` independent replicas ("replicas only")."""
    return world * cells / (ms_step * 1e-3) / 1e6


def _mem_available_gb() -> float:
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable"):
                    return int(line.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def _workload_name(case) -> str:
    return (f"configs[{case.cfg - 1}] {case.nx}x{case.ny}x{case.nz} fp64, "
            f"bc=({'PN'[case.bc_x]},{'PN'[case.bc_y]}), tanh-stretched z, Neumann phi in z, alpha*dt=1e-3")


# ------------------------------------------------------------------------------------------------
# CPU legs: the oracle (double build, as it stands) on a bounded sample of the workload
# ------------------------------------------------------------------------------------------------
def _cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _oracle_time(cfg: int, shape, reps: int, warm: int = 0, fields=None):
    """Times `reps` oracle projections (double build, as it stands) on the config's recipe at `shape`.
    Returns (Mcell/s, seconds per projection)."""
    import numpy as np
    from paper_2103_15187_b200 import inputs
    from oracle import Oracle
    if fields is None:
        case = inputs.make_case(cfg, shape=shape)
        u, v, w = case.u, case.v, case.w
    else:
        case = inputs.make_case(cfg, shape=shape, fields=False)
        u, v, w = fields
    orc = Oracle("d")
    p = np.zeros_like(u)
    for _ in range(warm):
        orc.pressure_projection(case.grid, u, v, w, p, case.alpha_dt, 0.0)
    t0 = time.perf_counter()
    for _ in range(reps):
        orc.pressure_projection(case.grid, u, v, w, p, case.alpha_dt, 0.0)
    dt = (time.perf_counter() - t0) / reps
    return case.cells / dt / 1e6, dt


def _oracle_single_thread(cfg: int):
    """One oracle projection with OMP_NUM_THREADS=1 on a slab of the workload (ny cut to SLAB_NY), in a child
    process (the OpenMP runtime reads the variable once).  Returns (Mcell/s, sample description) or (None, why)."""
    from paper_2103_15187_b200 import inputs
    nx, ny, nz = inputs.CONFIGS[cfg]["shape"]
    shape = (nx, min(ny, SLAB_NY), nz)
    code = ("import sys, json; sys.path.insert(0, %r); import bench; "
            "print(json.dumps(bench._oracle_time(%d, %r, 1)))" % (ROOT, cfg, shape))
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
        val, dt = json.loads(out.stdout.strip().splitlines()[-1])
    except Exception as e:  # noqa: BLE001 -- reported, not fatal
        return None, f"single-thread leg failed: {e}"
    return val, (f"1 oracle projection of a {shape[0]}x{shape[1]}x{shape[2]} slab of the workload grid (ny cut to {shape[1]}; "
                 f"the full grid would take ~{dt * ny / shape[1]:.0f} s on one thread), OMP_NUM_THREADS=1")


def _cpu_baseline(cfg: int, reps: int, warm: int = 0, fields=None, single: bool = True) -> dict:
    """The oracle on the box's host cores at the FULL benchmark configuration (all cores), plus a single-thread
    figure on a stated slab."""
    from paper_2103_15187_b200 import inputs
    shape = inputs.CONFIGS[cfg]["shape"]
    cores = int(os.environ.get("OMP_NUM_THREADS", 0)) or len(os.sched_getaffinity(0))
    need = 8 * shape[0] * shape[1] * shape[2] * (7 if fields is not None else 10) / 1e9
    if _mem_available_gb() < need + 4:
        return {"value": None, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": _cpu_model(),
                "sample": f"skipped: the full-size oracle needs ~{need:.0f} GB of host memory, {_mem_available_gb():.0f} GB available"}
    val, dt = _oracle_time(cfg, shape, reps, warm, fields)
    out = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": _cpu_model(), "s_per_projection": dt,
           "sample": (f"{reps} oracle projection(s) of the FULL {shape[0]}x{shape[1]}x{shape[2]} workload (double build, "
                      f"OpenMP over lines/columns, {cores} threads)")}
    if single:
        v1, s1 = _oracle_single_thread(cfg)
        out["threads1"] = {"value": v1, "unit": UNIT, "sample": s1}
    return out


def run_reference(args) -> dict:
    from paper_2103_15187_b200 import inputs
    case = inputs.make_case(args.config, fields=False)
    cpu = _cpu_baseline(args.config, args.steps, args.warmup, single=False)
    val = cpu["value"]
    return {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": cpu.get("s_per_projection", 0.0) * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_name(case), "cells": case.cells},
        "cpu_baseline": cpu,
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# ------------------------------------------------------------------------------------------------
# GPU leg
# ------------------------------------------------------------------------------------------------
def _config_table(main_cfg, dev, peak, steps_small=20):
    """Device-resident projection time of the OTHER BASELINE.json configs (compact: ms, Mcell/s, moved GB/s, kernel
    family), so that the one JSON line covers all five.  Inputs: N(0,1) fields generated on the device (the method is
    direct: its cost does not depend on the data; parity of these configs is the tests' job, with the seeded recipe)."""
    import torch
    from paper_2103_15187_b200 import inputs
    from paper_2103_15187_b200.binding import Plan
    fam = {0: "generic", 1: "fast", 2: "fused", 6: "fused+twisted"}
    out = {}
    for cfg in (1, 2, 3, 5):
        if cfg == main_cfg:
            continue
        case = inputs.make_case(cfg, fields=False)
        free, _ = torch.cuda.mem_get_info()
        if free < 8.0 * case.cells * 8:
            out[f"configs[{cfg - 1}]"] = {"skipped": "not enough device memory"}
            continue
        shp = (case.nz, case.ny, case.nx)
        g = torch.Generator(device=dev).manual_seed(cfg)
        u, v, w = (torch.randn(shp, dtype=torch.float64, device=dev, generator=g) for _ in range(3))
        w[0] = 0
        if case.bc_x:
            u[:, :, 0] = 0
        if case.bc_y:
            v[:, 0, :] = 0
        p, phi = torch.zeros_like(u), torch.empty_like(u)
        plan = Plan.from_grid(case.grid)
        steps = steps_small if case.cells < 3e8 else 5
        for _ in range(3):
            plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, 0.0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, 0.0)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps                       # timed WITHOUT the per-launch event pairs ...
        plan.profile(True)                                     # ... which cost a few microseconds per launch on the small grids
        for _ in range(steps):
            plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, 0.0)
        torch.cuda.synchronize()
        plan.profile(False)
        prof = plan.profile_read()
        ncomp2 = 2 if (case.bc_x or case.bc_y) else 1
        moved = 0.0
        for name, (kms, cnt) in prof.items():
            b = ALGO_BYTES_PER_CELL.get(name, 0.0)
            if name in ("yz_forward", "yz_backward"):
                b = 16.0 + 4.0 * ncomp2
            moved += b * cnt / steps
        out[f"configs[{cfg - 1}]"] = {
            "grid": f"{case.nx}x{case.ny}x{case.nz}", "bc": "PN"[case.bc_x] + "PN"[case.bc_y], "ms": round(ms, 4),
            "Mcell_per_s": round(case.cells / ms / 1e3, 1), "kernel_family": fam.get(plan.kernel_family, str(plan.kernel_family)),
            "launches_per_step": plan.last_launch_count, "moved_bytes_per_cell": round(moved, 1),
            "moved_GBps": round(moved * case.cells / (ms * 1e-3) / 1e9, 1), "frac_of_copy": round(moved * case.cells / (ms * 1e-3) / 1e9 / peak, 3),
            "kernels_ms": {k: round(v[0] / v[1], 4) for k, v in prof.items()}, "steps": steps}
        plan.destroy()
        del u, v, w, p, phi
        torch.cuda.empty_cache()
    return out


def _fluid_leg(plan, case, fields, stream, barrier, dev, peak, world, steps=3):
    """One whole fluid substep (fsei_fluid_substep) on the same workload: ms, per-kernel breakdown and a roofline entry for
    the implicit viscous step.  Extra device fields: 3 H + 3 rhs."""
    import torch
    u, v, w, p, phi = fields
    free, _ = torch.cuda.mem_get_info()
    if free < 6.5 * case.cells * 8:
        return {"skipped": "not enough device memory for 6 more fields"}, 0
    h = [torch.zeros_like(u) for _ in range(3)]
    r = [torch.empty_like(u) for _ in range(3)]
    dt, Re = case.alpha_dt, 3000.0
    gdt, rdt, adt, beta = 1.5 * dt, -0.5 * dt, dt, dt / (2 * Re)
    u.mul_(1e-2); v.mul_(1e-2); w.mul_(1e-2)          # keep the re-stepped synthetic field bounded (cost is data-independent)
    # synthetic immersed body: a sphere of markers about one grid cell apart
    from paper_2103_15187_b200 import inputs
    nmark = int(min(2_000_000, max(1000, 4 * 3.14159 * 0.3 ** 2 * case.nx * case.ny / (case.Lx * case.Ly))))
    xm, ym, zm, area, V = inputs.sphere_markers(nmark, (0.5 * case.Lx, 0.5 * case.Ly, 0.5), 0.3, seed=7, omega=(0.0, 0.0, 0.0),
                                                vel=(0.0, 0.0, 0.0))
    mk = [torch.from_numpy(a).to(u.device) for a in (xm, ym, zm, area, *V)]
    Fb = [torch.empty(nmark, dtype=torch.float64, device=u.device) for _ in range(3)]
    fib = [torch.zeros_like(u) for _ in range(3)] if free > 9.6 * case.cells * 8 else None     # zero-filled ONCE

    def substep():
        if fib is None:
            plan.fluid_substep(u, v, w, p, *h, *r, phi, gdt, rdt, adt, beta, stream=stream)
            return plan.last_launch_count
        n = 0
        for call, a in ((plan.ibm_forcing, (nmark, *mk[:4], *mk[4:], u, v, w, 1.0 / dt, *Fb, *fib)),
                        (plan.explicit_terms, (u, v, w, p, *h, *r, gdt, rdt, adt, beta)),
                        (plan.ibm_apply_forcing, (nmark, *mk[:3], *fib, *r, adt)),       # rhs += alpha dt f on the supports; clears f
                        (plan.viscous_step, (u, v, w, *r, beta)),
                        (plan.pressure_projection, (u, v, w, p, phi, adt, beta))):
            call(*a, stream=stream)
            n += plan.last_launch_count
        return n

    nl = 0
    for _ in range(2):
        nl += substep()
    barrier()
    plan.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        nl += substep()
    e1.record(stream)
    barrier()
    plan.profile(False)
    ms = max_over_ranks(e0.elapsed_time(e1), dev) / steps
    prof = plan.profile_read()
    kernels, moved = {}, 0.0
    for name, (kms, cnt) in prof.items():
        per = kms / cnt
        ab = ALGO_BYTES_PER_CELL.get(name, 0.0)
        moved += ab * cnt / steps
        kernels[name] = {"ms_per_launch": round(per, 4), "launches_per_step": cnt / steps,
                         "algo_GBps": round(ab * case.cells / (per * 1e-3) / 1e9, 1) if per > 0 else None}
    visc = [k for k in prof if k.startswith("visc_") and k != "visc_factor"]
    vms = sum(prof[k][0] for k in visc) / steps
    vbytes = sum(ALGO_BYTES_PER_CELL[k] * prof[k][1] for k in visc) / steps * case.cells
    finite = bool(torch.isfinite(u).all().item())
    has_ib = fib is not None
    del h, r, fib
    torch.cuda.empty_cache()
    out = {"ms_per_substep": round(ms, 4), "ib_markers": nmark, "Mcell_per_s": round(replica_throughput(case.cells, world, ms), 1), "steps": steps,
           "params": {"gamma_dt": gdt, "rho_dt": rdt, "alpha_dt": adt, "beta": beta, "Re": Re},
           "chain": "fsei_ibm_forcing -> fsei_explicit_terms -> fsei_ibm_apply_forcing (the forcing enters the rhs on the markers' "
                    "supports only) -> fsei_viscous_step -> fsei_pressure_projection" if has_ib else "fsei_fluid_substep",
           "ib_forcing_fields": has_ib,
           "moved_bytes_per_cell": round(moved, 1), "achieved_GBps": round(moved * case.cells / (ms * 1e-3) / 1e9, 1),
           "viscous_step": {"ms": round(vms, 4), "bytes_per_cell": round(vbytes / case.cells, 1), "bound": "hbm",
                            "achieved": round(vbytes / (vms * 1e-3) / 1e9, 1), "peak": peak, "unit": "GB/s",
                            "frac": round(vbytes / (vms * 1e-3) / 1e9 / peak, 4)},
           "kernels": kernels, "finite": finite}
    return out, nl



def run_ours(args) -> dict:
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2103_15187_b200 import inputs
    from paper_2103_15187_b200.binding import Plan

    rank = int(os.environ.get("RANK", 0))
    local = int(os.environ.get("LOCAL_RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libfsei has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: generated once on the host (seeded), one field at a time ---------------
    case = inputs.make_case(args.config, fields=False)
    shp = (case.nz, case.ny, case.nx)
    fbytes = case.cells * 8
    want_e2e = args.e2e_steps > 0 and _mem_available_gb() > 4.6 * fbytes / 1e9 + 8
    host = [torch.empty(shp, dtype=torch.float64, pin_memory=want_e2e) for _ in range(3)]
    # replicas: rank r perturbs nothing but the seed substream (independent problems, no exchange)
    t_gen = time.time()
    inputs.make_case(args.config, out=[h.numpy() for h in host], substep=0)
    t_gen = time.time() - t_gen
    u, v, w = (h.to(dev, non_blocking=False) for h in host)
    p = torch.zeros_like(u)
    phi = torch.empty_like(u)
    plan = Plan.from_grid(case.grid)
    stream = torch.cuda.current_stream()

    def step():
        plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, 0.0, stream)
        return plan.last_launch_count

    # ---- device-resident timing ------------------------------------------------------------------------
    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    sampler = ClockSampler(local)
    time.sleep(0.3)
    plan.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    barrier()
    t0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        launches += step()
    e1.record(stream)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms_total = e0.elapsed_time(e1)
    plan.profile(False)
    prof = plan.profile_read()
    ms_total = max_over_ranks(ms_total, dev)
    ms_step = ms_total / args.steps
    value = replica_throughput(case.cells, world, ms_step)

    # ---- roofline of the dominant kernel (live CUDA-event durations from the timed region) ---------------
    peak, peak_src = _peaks()
    kernels = {}
    for name, (ms, cnt) in prof.items():
        per = ms / cnt
        ab = ALGO_BYTES_PER_CELL.get(name, 0.0) * case.cells
        kernels[name] = {"ms_per_launch": round(per, 4), "launches_per_step": cnt / args.steps,
                         "algo_GBps": round(ab / (per * 1e-3) / 1e9, 1) if per > 0 else None,
                         "share": round(ms / ms_total, 4)}
    # whole step on the bytes the launches actually move (sum over the kernels of one step)
    moved = sum(ALGO_BYTES_PER_CELL.get(name, 0.0) * cnt / args.steps for name, (ms, cnt) in prof.items())
    moved_gbps = moved * case.cells / (ms_step * 1e-3) / 1e9
    top = max(prof, key=lambda k: prof[k][0])
    top_ms = prof[top][0] / prof[top][1]
    achieved = ALGO_BYTES_PER_CELL.get(top, 0.0) * case.cells / (top_ms * 1e-3) / 1e9
    traffic = _ncu_traffic(case.cfg, top)
    roofline = {"bound": "hbm", "kernel": top, "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4), "traffic": traffic, "peak_source": peak_src,
                "algo_bytes_per_launch": ALGO_BYTES_PER_CELL.get(top, 0.0) * case.cells,
                "ms_per_launch": round(top_ms, 4), "frac_of_8TBps": round(achieved / 8000.0, 4),
                "peak_note": "peak is the measured COPY bandwidth of this pool (one read + one write stream), not the HBM3e limit "
                             "(8 TB/s nominal): a kernel with 5 read and 4 write streams can exceed it, frac > 1 is not an error",
                "whole_step": {"moved_bytes_per_cell": round(moved, 2), "achieved": round(moved_gbps, 1),
                               "frac": round(moved_gbps / peak, 4), "frac_of_8TBps": round(moved_gbps / 8000.0, 4),
                               "unfused_bytes_per_cell": A_REF,
                               "unfused_equivalent_GBps": round(A_REF * case.cells / (ms_step * 1e-3) / 1e9, 1)},
                "kernels": kernels}

    # ---- the projection with beta != 0 (the branch a viscous time step takes: p += phi - beta L phi) ---------
    beta_nz = case.alpha_dt / (2.0 * 3000.0)
    plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, beta_nz, stream)
    b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    b0.record(stream)
    for _ in range(3):
        plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, beta_nz, stream)
    b1.record(stream)
    barrier()
    ms_beta = max_over_ranks(b0.elapsed_time(b1), dev) / 3
    launches += 4 * plan.last_launch_count

    # ---- whole fluid substep (explicit terms -> implicit viscous step -> projection) ------
    fluid = None
    if not args.no_fluid:
        fluid, nl = _fluid_leg(plan, case, (u, v, w, p, phi), stream, barrier, dev, peak, world)
        launches += nl

    # ---- the other BASELINE.json configs, compact ------------------------------------------------------------
    all_cfg = None
    if rank == 0 and world == 1 and not args.no_all_configs:
        del u, v, w, p, phi
        torch.cuda.empty_cache()
        all_cfg = _config_table(args.config, dev, peak)
        u = v = w = p = phi = None

    # ---- end to end: HOST buffers through the C ABI, H2D + D2H inside the timed region -------------------
    e2e = None
    if want_e2e:
        u = v = w = p = phi = None
        torch.cuda.empty_cache()
        hp = torch.zeros(shp, dtype=torch.float64, pin_memory=True)
        hu, hv, hw = host
        for _ in range(1):
            plan.pressure_projection_host(hu, hv, hw, hp, case.alpha_dt, 0.0, stream)
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for _ in range(args.e2e_steps):
            plan.pressure_projection_host(hu, hv, hw, hp, case.alpha_dt, 0.0, stream)
        a1.record(stream)
        barrier()
        ems = max_over_ranks(a0.elapsed_time(a1), dev) / args.e2e_steps
        e2e = {"value": replica_throughput(case.cells, world, ems), "unit": UNIT, "h2d_bytes_per_step": 4 * fbytes,
               "d2h_bytes_per_step": 4 * fbytes, "ms_per_step": ems, "steps": args.e2e_steps,
               "api": "fsei_pressure_projection_host (pinned u,v,w,p in; u,v,w,p out)"}
    else:
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
               "skipped": "--e2e-steps 0 or not enough host memory for 4 pinned fields"}
    plan.destroy()

    # ---- CPU baseline: the oracle as it stands, rank 0 at N = 1 only --------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = _cpu_baseline(args.config, 1, 0, fields=[h.numpy() for h in host])

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": _workload_name(case), "cells": case.cells, "projections_timed": args.steps,
                   "buffers": "same u,v,w,p re-projected back to back (direct method: cost is data-independent)",
                   "l2": f"inputs larger than L2 ({fbytes / 1e6:.0f} MB per field vs 126 MB)" if fbytes > 126e6 * 2
                         else "fields fit in L2 (small config; no flush)",
                   "parallelism": "replicas only" if world > 1 else "single GPU", "input_gen_s": round(t_gen, 1)},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
        "beta_nonzero": {"beta": beta_nz, "ms_per_step": round(ms_beta, 4), "Mcell_per_s": round(replica_throughput(case.cells, world, ms_beta), 1),
                         "note": "headline value is timed with beta = 0 (BASELINE configs state no Re); this is the same step with "
                                 "beta = alpha dt/(2 Re), Re = 3000"},
        "fluid_substep": fluid, "all_configs": all_cfg,
        "hbm_GBps_vs_8TBps": round(moved_gbps / 8000.0, 4),
    }
    if world > 1:
        dist.destroy_process_group()
    return out if rank == 0 else None


def run_slab(args) -> dict:
    """--parallel slab: ONE projection of the workload decomposed over the ranks: z-slabs for a1-a3 and
    a5-a7, x-slot pencils for a4, two exchanges over torch.distributed (NCCL).  Strong scaling: total work fixed."""
    import torch
    import torch.distributed as dist
    from paper_2103_15187_b200 import inputs, slab
    rank = int(os.environ.get("RANK", 0)); local = int(os.environ.get("LOCAL_RANK", 0)); world = int(os.environ.get("WORLD_SIZE", 1))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libfsei has no CPU fallback")
    local = local % torch.cuda.device_count()        # (more ranks than GPUs only with --dist-backend gloo: a functional check)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if not dist.is_initialized():
        if world > 1 and args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        elif world > 1:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("gloo", init_method="tcp://127.0.0.1:29533", rank=0, world_size=1)
    case = inputs.make_case(args.config, fields=False)
    sp = (slab.SlabFluid if args.slab_substep else slab.SlabProjection)(case.grid, rank, world, device=dev)
    g = torch.Generator(device=dev).manual_seed(100 + rank)
    for t in (sp.u, sp.v, sp.w):
        t.copy_(torch.randn(t.shape, dtype=torch.float64, device=dev, generator=g))
    if rank == 0:
        sp.w[0] = 0
    comm = slab.DistComm()
    if args.slab_peers:                                  # the exchanges happen in the kernels' epilogues (peer stores)
        if world > 1:                                    # one node: CUDA IPC handles of every rank's buffers
            pencils, specs = comm.ipc_buffers(sp.x)
        else:
            pencils, specs = [sp.x.pencil.data_ptr()], [sp.x.spec.data_ptr()]
        sp.set_peers(pencils, specs)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.slab_substep:                                # the whole fluid substep on slabs (explicit terms, viscous step, projection)
        for t in (sp.u, sp.v, sp.w):
            t.mul_(0.05)
        beta = case.alpha_dt / (2 * 3000.0)
        step = lambda: sp.substep(comm, 1.5 * case.alpha_dt, -0.5 * case.alpha_dt, case.alpha_dt, beta)
    else:
        step = lambda: sp.project(comm, case.alpha_dt, 0.0)
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sp.launches = 0
    barrier()
    t0 = time.time()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = max_over_ranks(e0.elapsed_time(e1), dev) / args.steps
    x = sp.x
    out = {"metric": METRIC, "value": case.cells / (ms * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": _workload_name(case), "cells": case.cells, "parallelism": f"z-slabs x{world} / x-slot pencils x{world}" + (", peer-store exchange" if args.slab_peers else ", grouped send/recv"),
                      "step": "fluid substep (explicit terms, viscous step, projection)" if args.slab_substep else "projection",
                      "exchange_bytes_per_rank_per_step": (8 if args.slab_substep else 2) * 16 * x.nzl * x.ny * (x.N - x.nsl),
                      "note": "unfused fast-family kernels per rank + 2 all-to-all exchanges (NCCL grouped send/recv); inputs N(0,1) "
                              "generated on the device; fields larger than L2"},
           "clocks": clocks, "gpu_launches": sp.launches,
           "e2e": {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "skipped": "slab mode times device-resident fields"}}
    if args.slab_peers and world > 1:
        comm.fence()
        return out if rank == 0 else None
    sp.destroy()
    if dist.is_initialized():
        dist.destroy_process_group()
    return out if rank == 0 else None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number 1..5 (default 4 = configs[3])")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fluid", action="store_true", help="skip the whole-fluid-substep leg")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the compact table of the other configs")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="--parallel slab: process-group backend (gloo stages through the host and lets several ranks share one GPU)")
    ap.add_argument("--slab-substep", action="store_true", help="--parallel slab: time the whole fluid substep instead of the projection")
    ap.add_argument("--slab-peers", action="store_true", help="--parallel slab: exchanges by peer stores from the kernels' epilogues")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default; the headline path is single-GPU) or ONE projection decomposed into "
                         "z-slabs / x-slot pencils over the N ranks (paper_2103_15187_b200/slab.py; strong scaling)")
    args = ap.parse_args()
    if args.parallel == "slab" and args.impl != "reference":
        out = run_slab(args)
        if out is not None:
            print(json.dumps(out), flush=True)
        if args.slab_peers and int(os.environ.get("WORLD_SIZE", 1)) > 1:
            sys.stdout.flush()
            os._exit(0)              # CUDA-IPC-shared tensors: torch's teardown order at interpreter exit is undefined
        return
    if args.impl == "reference":
        if int(os.environ.get("RANK", 0)) != 0:
            return
        args.steps = min(args.steps, 3)          # ~12 s per full-size projection on the box's cores
        args.warmup = min(args.warmup, 1)
        out = run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3
        out = run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
