#!/usr/bin/env python
"""bench.py - psdns_step throughput on B200 (grid-point-steps/s, ms/step, FP64) with roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 5c-channel|5c|5b|5a|cfg1|cfg2|cfg3|cfg4|fig3] [--impl reference]

One "step" = one pass of the whole hot path (rows a1-a11 of DESIGN.md) over the state.
Default workload = BASELINE.json config 5 on the 1024x512x513 grid (the grid the >= 60 % HBM
roofline target is quoted on): seeded random Hermitian-consistent spectra, k^-2 envelope.
N > 1: the path does not shard without an exchange step and north_star excludes a second GPU,
so ranks run independent replicas; value = sum over ranks.

`--impl reference` times the CPU oracle (oracle/psdns_oracle.py, as it stands) on the host cores
on a bounded sample of the same workload and prints the same JSON line with "impl": "reference".
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import psdns_inputs as I  # noqa: E402

METRIC = "grid-point-steps/s"
TRAFFIC_CSV = "r2e_traffic_5c.csv"   # ncu dram bytes per launch and kernel class, written from the --set full capture


# ------------------------------------------------------------------------------------------------
# workload table
# ------------------------------------------------------------------------------------------------
def workload(tag: str):
    if tag in I.SCALING_GRIDS:
        c = I.scaling_config(tag)
        kind = "random-spectra"
    elif tag.endswith("-channel") and tag[:-8] in I.SCALING_GRIDS:
        # config-3 recipe (channel state: Poiseuille + solenoidal k^-5/3 perturbation + 64 drops, Ch = 0.025, We = 3,
        # dt = 2e-5) on a config-5 grid.  SURVEY 8(d): "if the timed steps go non-finite, time the step on the config-3
        # recipe at these grids instead and say so" - the random-spectra state blows up at 1024x512x513 with dt = 2e-5
        # (an explicit-coupling time-step limit of the method at that resolution), so this is the
        # default workload
        nx, ny, nz = I.SCALING_GRIDS[tag[:-8]]
        k3 = I.CONFIGS[3]
        c = I.Config("cfg" + tag, nx, ny, nz, re=k3.re, ch=k3.ch, pe=k3.pe, we=k3.we, dt=k3.dt, steps=k3.steps,
                     ndrops=k3.ndrops, radius=k3.radius, seed=k3.seed)
        kind = "channel-state, config-3 recipe"
    elif tag == "cfg3":
        c = I.CONFIGS[3]
        kind = "channel-state"
    elif tag in ("cfg1", "cfg2", "cfg4"):
        c = I.CONFIGS[int(tag[3])]
        kind = "channel-state"
    elif tag == "fig3":   # the paper's Fig. 3 shape: single-phase 256x256x257
        c = I.Config("fig3", 256, 256, 257, re=3000.0, ch=1.0, pe=1.0, we=1.0, dt=2e-5, steps=10, seed=1006,
                     phase_field=0)
        kind = "channel-state"
    elif tag.count("x") == 2 and all(t.isdigit() for t in tag.split("x")):
        # config-5 recipe (random spectra, SURVEY 8(d) step parameters) on any supported grid, e.g. 512x256x65
        nx, ny, nz = (int(t) for t in tag.split("x"))
        k5 = I.scaling_config("5a")
        c = I.Config("cfg5-" + tag, nx, ny, nz, re=k5.re, ch=k5.ch, pe=k5.pe, we=k5.we, dt=k5.dt, steps=k5.steps, seed=k5.seed)
        kind = "random-spectra"
    else:
        raise SystemExit(f"unknown workload {tag}")
    return c, kind


def workload_string(c, kind) -> str:
    """One string for both arms (ours and --impl reference), so the driver sees the same config."""
    return (f"{c.name} psdns_step {c.nx}x{c.ny}x{c.nz} ({kind}), phase_field={c.phase_field}, "
            f"visc_ratio={c.visc_ratio}")


def algorithmic_bytes(c):
    """SURVEY.md 8(d) / DESIGN.md: bytes the method itself must move per step, per kernel class, with the
    structurally-zero dealiased modes never moved.  Unpadded retained sizes."""
    nx, ny, nz = c.nx, c.ny, c.nz
    N = nz - 1
    nkx, nky, nkz = nx // 3 + 1, 2 * (ny // 3) + 1, (2 * N) // 3 + 1
    S_ppp = 16 * nkx * nky * nkz
    S_ppz = 16 * nkx * nky * nz
    S_pyz = 16 * nkx * ny * nz
    R = 8 * nx * ny * nz
    phase = bool(c.phase_field)
    visc = phase and c.visc_ratio != 1.0
    nin = (12 if visc else 7) if phase else 3
    nout = 8 if phase else 6
    # field counts of the pipeline AS BUILT: matched viscosity sends 5 spectra through the
    # backward z pass (u v w phi Dphi; i ky phi is a second output of the phi columns), 6 through the backward y
    # pass (i kx phi is formed inside the fused x kernel) and 7 deviatoric products through the forward passes
    # (T_zz is subtracted pointwise).  Variable viscosity: 10 / 11 / 11 backward (5 strain spectra more), fused 16-slot x kernel.
    if phase:
        nzr, nzw, nyb, nfw = (10, 11, 11, 7) if visc else (5, 6, 6, 7)
    else:
        nzr, nzw, nyb, nfw = 3, 3, 3, 5
    per_kernel = {
        "zbwd": nzr * S_ppp + nzw * S_ppz,
        "ybwd": nyb * (S_ppz + S_pyz),
        "xbwd": nyb * (S_pyz + R),
        "pointwise": (nyb + nfw) * R,
        "xfwd": nfw * (R + S_pyz),
        "yfwd": nfw * (S_pyz + S_ppz),
        "zfwd": nfw * (S_ppz + S_ppp),
        "xfused": (nyb + nfw) * S_pyz,
        # solver stage, column-resident bound (every array crosses HBM once): k_rhs_elim reads the nfw product spectra,
        # the three AB2 history spectra and omega_z^, theta^, phi^ (all nz modes), writes the history; the sweeps that
        # follow write u^ v^ w^ phi^ theta^ omega_z^ (all nz modes) and D phi^.  The g' arrays between the down and up
        # sweeps of a solve are NOT algorithmic: whatever they add shows up as frac < 1.
        "rhs": (nfw + 3) * S_ppp + 3 * S_ppz + 3 * S_ppp,
        "solve": 6 * S_ppz + S_ppp,
    }
    per_kernel["solver"] = per_kernel["rhs"] + per_kernel["solve"]
    # fused-pipeline figure of SURVEY 8(d) (7 in / 8 out fields; the contract figure, about 310 B per grid point):
    # physical-space arrays never leave the SM
    step_fused = (4 * S_ppp + nin * S_ppz) + nin * (S_ppz + S_pyz) + (nin + nout) * S_pyz \
        + nout * (S_pyz + S_ppz) + (nout * S_ppz + 7 * S_ppp + 7 * S_ppp)
    return per_kernel, step_fused, dict(nkx=nkx, nky=nky, nkz=nkz, nin=nin, nout=nout)


# ------------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[6]))
            except ValueError:
                continue
            for nm, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(pw)}


# ------------------------------------------------------------------------------------------------
# CPU oracle, bounded sample (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sampled_step_seconds(c, budget_s: float = 20.0):
    """Times every stage of ONE oracle step (oracle/psdns_oracle.py, unmodified) on a thin slab of the
    workload's lines / columns and scales each stage by (full count / sampled count).
    Returns (estimated seconds per full step, description, threads)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import psdns_oracle as O
    nx, ny, nz = c.nx, c.ny, c.nz
    N = nz - 1
    nkxh = nx // 2 + 1
    g = O.Grid(nx, ny, nz, c.lx, c.ly)
    _, _, cnt = algorithmic_bytes(c)
    nin, nout = cnt["nin"], cnt["nout"]
    rng = np.random.default_rng(0)
    total = 0.0
    parts = {}

    def timed(fn, reps=1):
        t0 = time.perf_counter()
        for _ in range(reps):
            fn()
        return (time.perf_counter() - t0) / reps

    # slab widths chosen so that each stage takes about budget/8 seconds at most
    si = max(1, min(nkxh, 48))         # kx columns kept for the z / y matrix transforms
    sk = max(1, min(nz, 8))            # z planes kept for the x transform
    a_zy = rng.standard_normal((nz, ny, si)) + 1j * rng.standard_normal((nz, ny, si))
    Cb, Cf = O.cheb_bwd_matrix(N), O.cheb_fwd_matrix(N)
    By, Fy = O.dft_matrix(ny, +1), O.dft_matrix(ny, -1) / ny
    D = O.cheb_deriv_matrix(N)
    t = timed(lambda: O.apply_along(Cb, a_zy, 0)); parts["z_bwd"] = t * nin * nkxh / si
    t = timed(lambda: O.apply_along(By, a_zy, 1)); parts["y_bwd"] = t * nin * nkxh / si
    t = timed(lambda: O.apply_along(Fy, a_zy, 1)); parts["y_fwd"] = t * nout * nkxh / si
    t = timed(lambda: O.apply_along(Cf, a_zy, 0)); parts["z_fwd"] = t * nout * nkxh / si
    t = timed(lambda: O.apply_along(D, a_zy, 0)); parts["cheb_deriv"] = t * 14 * nkxh / si   # _Dz/_D2z/_lap calls per step
    # x direction on a z-slab (the oracle's own transform functions on a thin grid)
    gs = O.Grid(nx, ny, sk + 1 if sk + 1 >= 5 else 5, c.lx, c.ly)
    f_x = rng.standard_normal((gs.nz, ny, nx))
    Fx = O.dft_matrix(nx, -1)[:nkxh, :] / nx
    t = timed(lambda: O.apply_along(Fx, f_x, 2)); parts["x_fwd"] = t * nout * nz / gs.nz
    b_x = rng.standard_normal((gs.nz, ny, nkxh)) + 1j * rng.standard_normal((gs.nz, ny, nkxh))
    ang = 2.0 * np.pi * np.outer(np.arange(nkxh), np.arange(nx)) / nx
    cosm, sinm = np.cos(ang), np.sin(ang)
    t = timed(lambda: b_x.real @ cosm - b_x.imag @ sinm); parts["x_bwd"] = t * nin * nz / gs.nz
    # pointwise
    fs = [rng.standard_normal((gs.nz, ny, nx)) for _ in range(7)]
    p = O.Params(re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, phase_field=c.phase_field)
    if c.phase_field:
        t = timed(lambda: O.pointwise_terms(p, *fs))
    else:
        t = timed(lambda: O.pointwise_terms(p, *fs[:3]))
    parts["pointwise"] = t * nz / gs.nz
    # solves on a few columns
    ncol_full = cnt["nkx"] * cnt["nky"]
    m = min(64, ncol_full)
    rhs = rng.standard_normal((nz, m)) + 1j * rng.standard_normal((nz, m))
    sig = np.linspace(1.0e6, 2.0e6, m)
    nh = 2 + (2 if c.phase_field else 0)
    t = timed(lambda: O.helmholtz_solve(rhs, sig, O.DIRICHLET)); parts["helmholtz"] = t * nh * ncol_full / m
    t = timed(lambda: O.coupled_w_solve(rhs, sig, np.linspace(10.0, 20.0, m), 1e-8)); parts["coupled_w"] = t * ncol_full / m
    total = sum(parts.values())
    try:
        import threadpoolctl
        threads = max([d.get("num_threads", 1) for d in threadpoolctl.threadpool_info()] or [1])
    except Exception:
        threads = os.cpu_count() or 1
    desc = (f"each oracle stage of one {nx}x{ny}x{nz} step timed on a slab ({si} of {nkxh} kx columns for the z/y "
            f"matrix transforms, {gs.nz} of {nz} z planes for the x transform and pointwise terms, {m} of {ncol_full} "
            f"(kx,ky) columns for the dense tau solves) and scaled by full/sampled counts")
    return total, desc, threads, parts


def run_reference(args):
    c, kind = workload(args.workload)
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    M = c.nx * c.ny * c.nz
    for _ in range(max(0, min(args.warmup, 1))):
        oracle_sampled_step_seconds(c)
    ts = []
    for _ in range(max(1, min(args.steps, 3))):
        sec, desc, threads, parts = oracle_sampled_step_seconds(c)
        ts.append(sec)
    sec = float(np.mean(ts))
    val = M / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": METRIC, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(c, kind)},
        "cpu_baseline": {"value": val, "unit": METRIC, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# ours
# ------------------------------------------------------------------------------------------------
def reduce_max_ms(ms: float, world: int, device: str) -> float:
    """Replicas only: the job time is the MAX over ranks (device-timed milliseconds)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(points_per_replica: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job grid-point-steps/s over `world` independent replicas."""
    return world * points_per_replica * steps / (ms_max * 1e-3)


def make_state(c, kind):
    """Boundary-layout host arrays: SPECTRAL complex for random spectra, PHYSICAL real for channel states."""
    if kind == "random-spectra":
        return "spectral", list(I.random_spectral_state(c.nx, c.ny, c.nz, c.seed, cut=True))
    st = I.channel_state(c)
    return "physical", [s for s in st if s is not None]


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2406_01322_b200 as P

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libpsdns has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    c, kind = workload(args.workload)
    M = c.nx * c.ny * c.nz
    space_name, host = make_state(c, kind)
    space = P.SPECTRAL if space_name == "spectral" else P.PHYSICAL
    solver = P.Solver(c.nx, c.ny, c.nz, c.lx, c.ly, re=c.re, dt=c.dt, pe=c.pe, ch=c.ch, we=c.we, gradp_x=c.gradp_x,
                      visc_ratio=c.visc_ratio, phase_field=c.phase_field, device=f"cuda:{local}",
                      unfused_workspace=any(kv.startswith("xfuse=0") for kv in args.option))
    options = {}
    for kv in args.option:
        name, val = kv.split("=")
        solver.set_option(name, float(val))
        options[name] = float(val)
    pinned_in = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in host]
    del host
    dev = [t.cuda(non_blocking=True) for t in pinned_in]
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -------------------------------------------------------------------
    # step i) of the algorithm on the device: set_state (forward transform of the four fields when the
    # workload is a physical-space state), timed on its own (warm call first)
    solver.set_state(space, *dev)
    torch.cuda.synchronize()
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record()
    solver.set_state(space, *dev)
    s1.record()
    torch.cuda.synchronize()
    set_state_ms = s0.elapsed_time(s1)
    solver.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = solver.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    solver.step(args.steps)
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = solver.launch_count() - l0
    out = solver.get_state(P.SPECTRAL)
    finite = all(bool(torch.isfinite(torch.view_as_real(t)).all()) for t in out)
    maxabs = [float(torch.view_as_real(t).abs().max()) for t in out]
    del out
    # device-side diagnostics (psdns_diagnostics: mean phi, max |div u|, kinetic energy, wall shear, bulk velocity)
    solver.diagnostics()
    torch.cuda.synchronize()
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    d0.record()
    diag = solver.diagnostics()
    d1.record()
    torch.cuda.synchronize()
    diag_ms = d0.elapsed_time(d1)
    diag = dict(zip(P.Solver.DIAG_NAMES, [float(x) for x in diag.cpu().numpy()]))
    if not finite:
        # a timing of kernels processing NaN / Inf is not a measurement of this workload: no metric line, non-zero exit
        sys.stderr.write(f"bench.py: state of workload {args.workload} is non-finite after {args.warmup} + {args.steps} steps "
                         f"(max-abs {maxabs}); refusing to report a value\n")
        if world > 1:
            dist.destroy_process_group()
        raise SystemExit(3)
    ms_max = reduce_max_ms(ms, world, "cuda")
    value = aggregate_value(M, args.steps, ms_max, world)

    # ---- per-kernel-class CUDA-event timing (same steps, direct launches) -------------------------------
    per_kernel, step_fused_bytes, cnt = algorithmic_bytes(c)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    kernels = {}
    if rank == 0:
        ksteps = max(1, min(args.steps, 3))
        for name in ["zbwd", "ybwd", "xbwd", "pointwise", "xfused", "xfwd", "yfwd", "zfwd", "rhs", "solve"]:
            solver.kernel_timing(name, True)
            solver.step(ksteps)
            torch.cuda.synchronize()
            tot, n = solver.kernel_time_ms()
            solver.kernel_timing(name, False)
            if n == 0:
                continue
            ent = {"ms_per_step": tot / ksteps, "launches_per_step": n / ksteps}
            if name in per_kernel:
                ent["alg_bytes_per_step"] = per_kernel[name]
                ent["gbs"] = per_kernel[name] / (tot / ksteps * 1e-3) / 1e9 if tot > 0 else None
                ent["frac"] = ent["gbs"] / peak if tot > 0 else None
            kernels[name] = ent
    if "rhs" in kernels and "solve" in kernels:
        tms = kernels["rhs"]["ms_per_step"] + kernels["solve"]["ms_per_step"]
        kernels["solver"] = {"ms_per_step": tms, "launches_per_step": kernels["rhs"]["launches_per_step"] + kernels["solve"]["launches_per_step"],
                             "alg_bytes_per_step": per_kernel["solver"], "gbs": per_kernel["solver"] / (tms * 1e-3) / 1e9,
                             "frac": per_kernel["solver"] / (tms * 1e-3) / 1e9 / peak,
                             "note": "rhs + solve classes together (k_rhs_elim ... k_finish), column-resident bound"}
    dominant = max((k for k in kernels if k in per_kernel and k != "solver"), key=lambda k: kernels[k]["ms_per_step"], default=None)
    # measured DRAM traffic per launch from the committed ncu --set full capture of this workload (text summary
    # under profiles/; null for workloads that were not captured)
    traffic = {}
    try:
        if args.workload in ("5c", "5c-channel") and not options:   # same grid, same kernels: traffic does not depend on the data
            with open(os.path.join(ROOT, "profiles", TRAFFIC_CSV)) as fh:
                for ln in fh.read().strip().splitlines()[1:]:
                    kname, val = ln.split(",")
                    traffic[kname] = float(val)
    except Exception:
        pass

    # ---- end to end through the C ABI with host buffers -----------------------------------------------
    pinned_out = [torch.empty_like(t).pin_memory() for t in pinned_in]
    nbytes = sum(t.numel() * t.element_size() for t in pinned_in)
    solver.run_host(space, 1, pinned_in, pinned_out)   # warm-up
    solver.run_host_wait()
    barrier()
    # consecutive calls on one handle: the device -> host copy of call k (side stream) overlaps the upload and the compute
    # of call k + 1; the timed region ends when the LAST copy-back has landed (run_host_wait), so every step's H2D and D2H
    # are inside it.  g1 is recorded after the host has seen that completion.
    esteps = max(1, min(args.steps, 10))
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record()
    for _ in range(esteps):
        solver.run_host(space, 1, pinned_in, pinned_out)
    solver.run_host_wait()
    g1.record()
    barrier()
    e2e_ms = g0.elapsed_time(g1)
    e2e_max = reduce_max_ms(e2e_ms, world, "cuda")
    e2e_val = aggregate_value(M, esteps, e2e_max, world)
    e2e_finite = all(bool(torch.isfinite(torch.view_as_real(t) if t.is_complex() else t).all()) for t in pinned_out)
    if not e2e_finite:
        sys.stderr.write("bench.py: end-to-end output is non-finite; refusing to report a value\n")
        raise SystemExit(3)
    del pinned_out

    # ---- forward + backward transform round trip of one field, dealiasing off (BASELINE.json config 5) ----------
    roundtrip = None
    if rank == 0:
        R = 8 * M
        S_full = 16 * (c.nx // 2 + 1) * c.ny * c.nz
        xin = torch.from_numpy(I.random_physical_field(c.nx, c.ny, c.nz, seed=5)).cuda()
        rt = solver.transform_roundtrip(P.PHYSICAL, xin)           # warm-up, and the identity check
        rt_err = float(torch.linalg.vector_norm(rt - xin) / torch.linalg.vector_norm(xin))
        del rt
        rsteps = max(1, min(args.steps, 5))
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        r0.record()
        for _ in range(rsteps):
            rt = solver.transform_roundtrip(P.PHYSICAL, xin)
        r1.record()
        torch.cuda.synchronize()
        rt_ms = r0.elapsed_time(r1) / rsteps
        del rt, xin
        # each of the 3 + 3 one-dimensional passes reads and writes its array once (x: R <-> S_full, y and z: S_full <->
        # S_full); the spectrum stays in the private layout between the two transforms (no d_mid requested)
        passes = 2 * R + 10 * S_full
        roundtrip = {"ms": rt_ms, "rel_l2_identity_error": rt_err, "fields": 1, "dealias": 0,
                     "alg_bytes_min": 2 * (R + S_full), "gbs_min": 2 * (R + S_full) / (rt_ms * 1e-3) / 1e9,
                     "alg_bytes_passes": passes, "gbs_passes": passes / (rt_ms * 1e-3) / 1e9,
                     "frac_passes": passes / (rt_ms * 1e-3) / 1e9 / peak,
                     "note": "psdns_transform_roundtrip PHYSICAL -> SPECTRAL -> PHYSICAL, full (unpruned) sizes; "
                             "alg_bytes_min = read R, write S, read S, write R; alg_bytes_passes = six 1-D passes each "
                             "reading and writing its array once"}
        if rt_err > 1e-11:
            sys.stderr.write(f"bench.py: transform round trip error {rt_err:.2e} > 1e-11\n")
            raise SystemExit(3)

    if rank == 0:
        roof = None
        if dominant is not None:
            k = kernels[dominant]
            roof = {"bound": "hbm", "kernel": dominant, "achieved": k["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": k["frac"], "traffic": traffic.get(dominant), "traffic_unit": "bytes per launch (ncu dram read + write)",
                    "alg_bytes_per_launch": k["alg_bytes_per_step"] / max(k["launches_per_step"], 1), "peak_source": peak_src,
                    "launch_ms": k["ms_per_step"] / max(k["launches_per_step"], 1)}
        # second view of the dominant kernel when it is the fused x kernel: it is FP64-issue bound as much as HBM bound
        # (ncu: FP64 pipe 56 %, DRAM 28 %).  Algorithmic flops: 2.5 N_x log2 N_x per real line and transform,
        # 45 per grid point for the products; peak = 148 SMs x 64 FP64 FMA/clk x 2 x max SM clock.
        roof_alu = None
        if dominant == "xfused":
            lines = c.ny * c.nz
            flops = lines * ((cnt["nin"] + (7 if c.phase_field else 5)) * 2.5 * c.nx * math.log2(c.nx) + 45.0 * c.nx)
            sm_clock = float((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6
            nominal_tf = 148 * 64 * 2 * sm_clock / 1e12
            peak_tf = solver.measure_fp64_peak()        # FMA-chain microbenchmark on this GPU
            tf = flops / (kernels["xfused"]["ms_per_step"] * 1e-3) / 1e12
            roof_alu = {"bound": "alu", "kernel": "xfused", "achieved": tf, "peak": peak_tf, "unit": "TFLOP/s (FP64)",
                        "frac": tf / peak_tf, "alg_flops_per_launch": flops,
                        "peak_source": "measured: FP64 FMA-chain microbenchmark (psdns_measure_fp64_peak)",
                        "peak_nominal": nominal_tf,
                        "peak_nominal_source": "148 SMs x 64 FP64 FMA/clk x 2 x max SM clock (B200 guide unit counts)"}
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            sec, desc, threads, parts = oracle_sampled_step_seconds(c)
            cpu = {"value": M / sec, "unit": METRIC, "cores": threads, "kind": "oracle", "sample": desc,
                   "ms_per_step": sec * 1e3}
        line = {
            "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(c, kind), "grid": [c.nx, c.ny, c.nz],
                       "l2": "inputs larger than L2 (state and intermediates >> 126 MB)" if M > 4e6 else "small grid: L2-resident, no roofline claim",
                       "parallelism": "replicas only" if world > 1 else "single GPU", "finite": finite, "max_abs": maxabs,
                       "options": options},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": METRIC, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                    "ms_per_step": e2e_max / esteps, "steps": esteps, "finite": e2e_finite,
                    "call": "psdns_run_host x steps, then psdns_run_host_wait (copy-back of one call overlaps the next call)"},
            "gpu_launches": launches,
            "roofline": roof,
            "roofline_alu": roof_alu,
            "step_roofline": {"alg_bytes_per_step_fused_design": step_fused_bytes,
                              "alg_bytes_per_grid_point": step_fused_bytes / M,
                              "achieved_gbs": step_fused_bytes / (ms_max / args.steps * 1e-3) / 1e9,
                              "frac": step_fused_bytes / (ms_max / args.steps * 1e-3) / 1e9 / peak},
            "kernels": kernels,
            "roundtrip": roundtrip,
            "step_i": {"call": f"psdns_set_state({space_name.upper()})", "ms": set_state_ms, "fields": len(dev),
                       "note": "PAPER.md L138 step i): one full forward transform per field (x, y, z) when the input is "
                               "physical, a re-layout when it is spectral; plus the hidden state theta^, omega_z^, D phi^"},
            "diagnostics": {"ms": diag_ms, **diag},
            "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="5c-channel")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="psdns_set_option before the run (A/B measurements: ztma=0, zgemm=1, xfuse=0, graph=0, ...)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
