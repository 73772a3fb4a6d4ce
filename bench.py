#!/usr/bin/env python
"""bench.py -- throughput of the echellogram-rendering hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A step = one pass of the whole hot path (a1-a6: zero-fill, sample setup, render, detector stage) over one frame
of the synthetic workload (default: ESPRESSO-like, BASELINE.json configs[1]).  Prints ONE JSON line.
N > 1 (torchrun): every rank renders its own replica of the frame ("replicas only"); no collective
on the data path.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "fp64 lambda-sample x pixel contributions/s"
UNIT = "contributions/s"

# flop-equivalents of the special-function edge evaluations, SURVEY.md 8(d) (used only for the secondary
# "survey_formula" figure; the headline roofline counts the irreducible FMAs only)
C_ERFC, C_PSI = 60.0, 90.0

# dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed `ncu --set full` captures: profiles/traffic.json
# holds, per (workload, kernel), the bytes, the profile file they come from and the sha256 of the kernel's source file at
# capture time.  A value is reported only while that hash still matches the source in the tree (else null + a note).
# kernel -> the source files its device code comes from (a capture in profiles/traffic.json is stale once any of them changed)
KERNEL_SOURCES = {"render_moment_kernel": ("render_moment.cuh",), "render_tabcell_kernel": ("render_tabcell.cuh",),
                  "render_poly_kernel": ("render_poly.cuh",), "render_analytic_kernel": ("render_analytic.cuh",),
                  "render_tabulated_kernel": ("render_tabulated.cuh",), "detector_kernel": ("detector.cu",),
                  "cell_flush_kernel": ("render_cells.cuh", "render_moment.cuh"), "cell_flush_wide_kernel": ("render_cells.cuh", "render_moment.cuh"),
                  "cell_moment_kernel": ("render_cells.cuh", "render_moment.cuh", "setup.cuh"),
                  "setup_samples_kernel": ("setup.cuh",)}


def source_hash(kernel: str):
    import hashlib
    files = KERNEL_SOURCES.get(kernel.split("<")[0])
    if not files:
        return None
    h = hashlib.sha256()
    for name in files:
        f = ROOT / "paper_2008_05858_b200" / "csrc" / name
        if not f.is_file():
            return None
        h.update(f.read_bytes())
    return h.hexdigest()


def ncu_traffic(workload: str, kernel: str):
    """(bytes per launch or None, note)"""
    try:
        table = json.loads((ROOT / "profiles" / "traffic.json").read_text())
    except Exception:
        return None, "profiles/traffic.json missing"
    e = table.get(f"{workload}:{kernel}")
    if not e:
        return None, "no ncu capture committed for this (workload, kernel)"
    if e.get("source_sha256") != source_hash(kernel):
        return None, f"stale: {' / '.join(KERNEL_SOURCES.get(kernel.split('<')[0], ()))} changed since {e.get('profile')}"
    return float(e["bytes_per_launch"]), f"{e.get('profile')} ({e.get('launches_per_step')} launches per step)"


def measured_peaks():
    """driver-written MEASURED_PEAKS.json (HBM GB/s, bf16 TF/s); fallback = B200_PROFILING.md's figure, flagged"""
    try:
        d = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback): MEASURED_PEAKS.json absent"


def make_scene(name: str):
    from paper_2008_05858_b200 import workloads as W
    if name == "espresso_like":
        return W.espresso_like(), "espresso_like (BASELINE.json configs[1]: 2 fibers x 85 orders, 9216x9216, 32 samples/px)"
    if name == "tiny":
        return W.tiny(), "tiny (BASELINE.json configs[0])"
    if name == "hires_like":
        return W.hires_like(), "hires_like (BASELINE.json configs[2]: 10 fibers x 60 orders, 9216x9216, 32 samples/px)"
    if name == "field_psf":
        return W.field_psf(), "field_psf (BASELINE.json configs[3]: ESPRESSO-like geometry, 5x5 grid of 11x11-px 8x kernels)"
    if name == "rv_sweep":
        return W.rv_sweep(10.0), "rv_sweep (BASELINE.json configs[4], one of the 5 frames, v = 10 m/s)"
    raise SystemExit(f"unknown workload {name}")


def support_half_widths(psf):
    """hb = footprint half-width + 1/2 per axis (G9) -- used only to COUNT contributions"""
    if psf.kind == 1:
        h = 0.5 * psf.tab_npix + 0.5
        return h, h
    t = psf.support_nsigma if psf.support_nsigma > 0 else 7.5
    return 0.5 * psf.fiber_dx_px + t * psf.sigma_x + 0.5, 0.5 * psf.fiber_dy_px + t * psf.sigma_y + 0.5


def algorithmic_flops_per_sample(psf, Q: int, ncols: float, nrows: float):
    """(irreducible FMA flops, SURVEY 8(d) formula) per sample for the analytic path."""
    if psf.kind != 0:
        return None, None
    T = (Q + 1) // 2 if Q > 1 else 1                       # paired chord terms
    fma_only = 2.0 * T * ncols * nrows
    n = 0.5 * (ncols + nrows)
    survey = 200.0 + Q * (n + 1) * C_ERFC + (Q / 2.0) * 2 * (n + 1) * C_PSI + 2.0 * Q * ncols * nrows
    return fma_only, survey


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.2] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline at N=1, and --impl reference)
# ----------------------------------------------------------------------------------------------------------------
def oracle_sample_scene(scene, target_samples: int):
    """A bounded sample of the workload: the middle order, all fibers, a wavelength sub-range holding about
    target_samples / n_fibers samples per fiber; returns (sub-scene, window) with the window enclosing the footprints."""
    import oracle
    o = scene.n_orders // 2
    sub = scene.subset(orders=[o])
    n_full = oracle.order_nsamples(sub, 0)
    per_fiber = max(64, target_samples // scene.n_fibers)
    frac = min(1.0, per_fiber / max(n_full, 1))
    lmin, lmax = float(sub.lam_min[0]), float(sub.lam_max[0])
    mid = 0.5 * (lmin + lmax)
    half = 0.5 * (lmax - lmin) * frac
    # keep the sampling density of the full order: N = ceil(spp * |dx|) over the sub-range
    sub.lam_min = np.array([mid - half]); sub.lam_max = np.array([mid + half])
    hbx, hby = support_half_widths(scene.psf)
    xs, ys = [], []
    for f in range(sub.n_fibers):
        n = oracle.order_nsamples(sub, 0)
        for k in (0, n // 2, n - 1):
            lam, x, y, w = oracle.samples(sub, f, 0, k, k + 1)
            xs.append(x[0]); ys.append(y[0])
    # the trace is smooth: pad the bounding box of its ends and middle generously
    i0 = max(0, int(np.floor(min(xs) - hbx)) - 8); i1 = min(scene.nx, int(np.ceil(max(xs) + hbx)) + 8)
    j0 = max(0, int(np.floor(min(ys) - hby)) - 64); j1 = min(scene.ny, int(np.ceil(max(ys) + hby)) + 64)
    return sub, (i0, j0, i1 - i0, j1 - j0)


def time_oracle(scene, target_samples: int, steps: int = 1, warmup: int = 0):
    import oracle
    sub, win = oracle_sample_scene(scene, target_samples)
    hbx, hby = support_half_widths(scene.psf)
    ncols, nrows = np.floor(2 * hbx), np.floor(2 * hby)
    times, touched = [], 0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.render(sub, window=win)
        dt = time.perf_counter() - t0
        touched = oracle.render.last_touched
        if it >= warmup:
            times.append(dt)
    n_samples = sum(oracle.order_nsamples(sub, 0) for _ in range(sub.n_fibers))
    contrib = float(n_samples) * float(ncols * nrows)
    t = float(np.mean(times))
    return {"value": contrib / t, "unit": UNIT, "cores": oracle.cpu_threads(), "kind": "oracle",
            "sample": f"{n_samples} samples ({sub.n_fibers} fibers x 1 order, {touched} touched the window) of the "
                      f"{scene.name} workload, oracle Q=32 long double, {t:.2f} s per pass",
            "seconds": t, "contributions": contrib}


def run_reference(args, rank: int):
    if rank != 0:
        return
    scene, wname = make_scene(args.workload)
    r = time_oracle(scene, args.oracle_samples, steps=max(1, args.steps), warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": min(args.warmup, 1), "ms_per_step": r["seconds"] * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wname, "note": "CPU oracle (oracle/e2e_oracle.c) as it stands, each step a bounded sample"},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------------------
def count_contributions(B, r, hbx, hby):
    """exact number of (sample, pixel) pairs inside the footprint boxes (G9) clipped to the detector; a COUNT for
    the metric's unit, computed with torch ops on the setup kernel's own x, y"""
    import torch
    nmax = int(r.per_order.max())
    x = torch.empty(max(nmax, 1), dtype=torch.float64, device=r.device)
    y = torch.empty_like(x)
    total, cells = 0, 0
    for f in range(r.scene.n_fibers):
        for o in range(r.scene.n_orders):
            n = int(r.per_order[o])
            if n == 0:
                continue
            B.e2e_setup_samples(r.fmt, r.spectra[f], f, o, None, x, y, None, capacity=nmax)
            xs, ys = x[:n], y[:n]
            ilo = torch.clamp(torch.ceil(xs - hbx), min=0); ihi = torch.clamp(torch.floor(xs + hbx), max=r.scene.nx - 1)
            jlo = torch.clamp(torch.ceil(ys - hby), min=0); jhi = torch.clamp(torch.floor(ys + hby), max=r.scene.ny - 1)
            total += int((torch.clamp(ihi - ilo + 1, min=0) * torch.clamp(jhi - jlo + 1, min=0)).sum().item())
            # footprint cells: maximal runs of consecutive samples with one (unclipped) footprint box
            b = torch.stack([torch.ceil(xs - hbx), torch.floor(xs + hbx), torch.ceil(ys - hby), torch.floor(ys + hby)])
            cells += 1 + int((b[:, 1:] != b[:, :-1]).any(dim=0).sum().item())
    return total, cells


def max_over_ranks(x: float, world: int, device=None) -> float:
    """max over ranks of a per-rank time (the only cross-rank exchange of the bench: "replicas only")"""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world: int, units_per_rank: float, seconds_per_step: float) -> float:
    """whole-job throughput: every rank processes its own replica of the workload (weak scaling)"""
    return world * units_per_rank / seconds_per_step


def measure_device(B, W, torch, name: str, steps: int, warmup: int, rank: int, world: int, dev, batch_frames: int = 1,
                   sampler=None):
    """K timed steps of the whole hot path (a1-a6) on one workload with inputs resident in HBM.  Returns the raw numbers
    (times in ms per step, counts per step) plus the live objects the e2e leg reuses."""
    scene, wname = make_scene(name)
    det = scene.detector or W.Detector(gain=1.0, dark_e=0.0, ron_e=3.0, bias=0.0, seed=2008_05858 + rank)
    r = B.Renderer(scene, device=str(dev))
    info = r.psf.info()
    hbx, hby = support_half_widths(scene.psf)
    contrib, n_cells = count_contributions(B, r, hbx, hby)
    kinfo = B.e2e_render_kernel_info(r.fmt, r.psf)
    alg = B.e2e_render_algorithmic_fma(r.fmt, r.psf)
    n_samples = r.n_samples
    frame = torch.empty((scene.ny, scene.nx), dtype=torch.float64, device=dev)
    noisy = torch.empty_like(frame)
    stream = torch.cuda.current_stream()
    nbatch = max(1, batch_frames)
    host_dopplers = [1.0]
    if nbatch > 1:
        # --batch-frames N: N Doppler-shifted copies of the workload's spectra (the RV-sweep velocities, cycled) rendered by
        # ONE e2e_render_frames call per step; a unit of work is still one (sample, pixel) contribution
        import copy
        vs = [0.0, 0.01, 0.1, 1.0, 10.0]
        host_dopplers = [1.0 + vs[b % 5] / W.C_LIGHT for b in range(nbatch)]
        batch_descs = []
        for dop in host_dopplers:
            sp = [copy.copy(x) for x in scene.spectra]
            for x in sp:
                x.doppler = x.doppler * dop
            batch_descs.append(B.spectra_array(sp, [t.data_ptr() for t in r.flux]))
        batch_frames_t = [torch.empty_like(frame) for _ in range(nbatch)]
        batch_ws = torch.empty(B.e2e_render_frames_workspace_bytes(r.fmt, r.psf, nbatch), dtype=torch.uint8, device=dev)
        contrib, n_cells, n_samples = contrib * nbatch, n_cells * nbatch, n_samples * nbatch
        wname += f", batch of {nbatch} Doppler-shifted frames per step (e2e_render_frames)"

    def step():
        if nbatch > 1:
            B.e2e_render_frames(r.fmt, r.psf, batch_descs, batch_frames_t, False, batch_ws, stream)
            for fr in batch_frames_t:
                B.e2e_apply_detector(fr, noisy, scene.nx, scene.ny, det, stream)
            return
        B.e2e_render_frame(r.fmt, r.psf, r.spectra, frame, False, r.workspace, stream)
        B.e2e_apply_detector(frame, noisy, scene.nx, scene.ny, det, stream)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(warmup, 3)):
        step()
    barrier()
    # ---- device-timed region: K steps, inputs resident in HBM
    B.e2e_profile_enable(True)
    B.e2e_profile_read(reset=True)
    if sampler is not None:
        sampler.start()
        time.sleep(0.25)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = B.e2e_launch_count()
    t_wall0 = time.time()
    torch.cuda.profiler.start()                          # ncu --profile-from-start off: launch list of the timed region only
    ev0.record(stream)
    for _ in range(steps):
        step()
    ev1.record(stream)
    barrier()
    torch.cuda.profiler.stop()
    t_wall1 = time.time()
    launches = B.e2e_launch_count() - n0
    ms_total = ev0.elapsed_time(ev1)
    prof = B.e2e_profile_read(reset=True)
    B.e2e_profile_enable(False)
    clocks = sampler.stop(t_wall0, t_wall1) if sampler is not None else None
    ms_step = max_over_ranks(ms_total, world, dev) / steps
    ncalls = max(prof["n_calls"], 1)
    return {"scene": scene, "wname": wname, "det": det, "r": r, "info": info, "hbx": hbx, "hby": hby, "contrib": contrib,
            "n_cells": n_cells, "n_samples": n_samples, "kinfo": kinfo, "alg": alg, "ms_step": ms_step, "steps": steps,
            "stage_ms": {k: prof[k] / ncalls for k in ("ms_zero", "ms_setup", "ms_render", "ms_detector")},
            "render_launches": prof["n_render"] / ncalls, "launches": int(launches), "clocks": clocks, "nbatch": nbatch,
            "host_dopplers": host_dopplers, "barrier": barrier, "stream": stream}


def stage_rooflines(m, name: str, peak_tf: float, burst_tf: float):
    """SURVEY 8(d) 'report the respective bound too': one entry per stage.  setup / zero-fill / detector against the HBM roof
    (algorithmic bytes: what the stage must move once), render against the FP64 pipe (DESIGN.md 5.3 / 5.5 work counts)."""
    scene, kinfo, alg = m["scene"], m["kinfo"], m["alg"]
    hbm_gbs, hbm_src = measured_peaks()
    npx = scene.nx * scene.ny * m["nbatch"]
    n_samples, n_cells = m["n_samples"], m["n_cells"]
    table_bytes = sum(int(np.asarray(sp.flux).shape[0]) * 8 for sp in {id(sp.flux): sp for sp in scene.spectra}.values())
    out = {}

    def hbm(stage, ms, nbytes, what, kernel):
        if ms <= 0:
            return
        ach = nbytes / (ms * 1e-3) / 1e9
        traffic, tnote = ncu_traffic(name, kernel) if kernel else (None, "cudaMemsetAsync (no kernel of the library)")
        out[stage] = {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs, "traffic": traffic,
                      "traffic_note": tnote, "kernel": kernel, "ms_per_step": ms, "algorithmic_bytes": nbytes, "definition": what,
                      "peak_source": hbm_src}

    hbm("zero", m["stage_ms"]["ms_zero"], 8.0 * npx, "8 B per pixel written", None)
    split = kinfo["name"].startswith("cell_flush_")
    if split:
        # two-kernel analytic path: the setup stage is cell_moment_kernel (a1-a3 fused + step 1); it writes one record per cell
        npt = int(kinfo["name"].split("<")[1].rstrip(">"))
        rec = 32.0 + 512.0 * npt
        # large frames are zero-filled inside this kernel (no separate pass: ms_zero = 0), 8 B per pixel more
        fused_zero = m["stage_ms"]["ms_zero"] <= 0
        hbm("setup", m["stage_ms"]["ms_setup"], rec * n_cells + table_bytes * m["nbatch"] + (8.0 * npx if fused_zero else 0.0),
            "cell_moment_kernel: %d B per footprint cell written (header + moment tiles) + the spectrum tables read once%s; its step 1 is "
            "%.3g fp64 flop per frame (2 x 8 (P+1) per sample)" % (rec, " + the frame's zero-fill (8 B per pixel written)" if fused_zero else "",
                                                                  2.0 * n_samples * alg["fma_per_sample"]), "cell_moment_kernel<%d>" % npt)
    else:
        hbm("setup", m["stage_ms"]["ms_setup"], 24.0 * n_samples + table_bytes * m["nbatch"],
            "24 B per sample written (x, y, w) + the spectrum tables read once", "setup_samples_kernel")
    hbm("detector", m["stage_ms"]["ms_detector"], 16.0 * npx, "16 B per pixel (fp64 frame read + fp64 frame written)", "detector_kernel<double, false>")
    ms_render = m["stage_ms"]["ms_render"]
    if ms_render > 0:
        sec = ms_render * 1e-3
        alg_flops = 2.0 * (n_cells * alg["fma_per_cell"] + (0 if split else n_samples * alg["fma_per_sample"]))
        executed = 2.0 * (n_cells * kinfo["executed_fma_per_cell"] + n_samples * kinfo["executed_fma_per_sample"])
        ncols, nrows = np.floor(2 * m["hbx"]), np.floor(2 * m["hby"])
        fma_flops, survey_flops = algorithmic_flops_per_sample(scene.psf, m["info"]["n_nodes"], ncols, nrows)
        definition = ("algorithmic = un-padded fp64 flops of the cell-moment method (DESIGN.md 5.3 'Roofline'): per cell "
                      "2 T (8 (P+1) w + 8 w h), per sample 2 * 8 (P+1); x measured cell / sample counts of the workload")
        if split:
            definition = ("algorithmic = un-padded fp64 flops of the contraction this kernel performs (steps 2 + 3 of the cell-moment method, "
                          "DESIGN.md 5.3): per cell 2 T (8 (P+1) w + 8 w h) x the measured cell count; the moment update (2 * 8 (P+1) per "
                          "sample) runs in cell_moment_kernel and is counted there (stage_roofline.setup)")
        if kinfo["name"].startswith("render_tabcell"):
            definition = ("algorithmic = fp64 flops of the cell-deposit method (DESIGN.md 5.5): per cell 2 x nodes x 2 y-offset rows x "
                          "(os+1) x-offsets x (npix+1)^2 window pixels, per sample 2 x 4 x nodes deposit products; x measured counts")
        if alg_flops <= 0 and fma_flops is not None:         # kernels that do not work cell by cell: the direct method's accumulate
            alg_flops = n_samples * fma_flops
            definition = "algorithmic = bare rank-T accumulate of the per-sample method, 2 T w h flop per sample"
        traffic, tnote = ncu_traffic(name, kinfo["name"])
        ach = alg_flops / sec / 1e12
        rl = {"bound": "alu", "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf, "traffic": traffic,
              "traffic_note": tnote, "kernel": kinfo["name"], "kernel_ms_per_step": ms_render,
              "kernel_launches_per_step": m["render_launches"],
              "peak_source": "measured in this run: e2e_measure_fp64_peak, sustained FP64-pipe rate (max of DFMA and DMMA chains) x 2 "
                             "(MEASURED_PEAKS.json has no fp64 entry)",
              "peak_burst": burst_tf, "flops_per_sample": alg_flops / max(n_samples, 1), "definition": definition,
              "footprint_cells": n_cells}
        if executed > 0:
            rl.update({"executed_tflops": executed / sec / 1e12, "executed_frac": executed / sec / 1e12 / peak_tf,
                       "executed_definition": "fp64 FMAs the kernel issues (DMMA = 256, padded tiles) x 2, from e2e_render_kernel_info x cell / sample counts"})
        if fma_flops is not None:
            rl.update({"direct_method_flops_per_sample": fma_flops,
                       "direct_method_tflops_equivalent": n_samples * fma_flops / sec / 1e12,
                       "direct_method_definition": "bare rank-T accumulate of the per-sample method, 2*T*w*h flop per sample: what this kernel would "
                                                   "have to sustain if it evaluated every (sample, pixel) product (it does not: context only)",
                       "survey_flops_per_sample": survey_flops,
                       "survey_formula_tflops_equivalent": n_samples * survey_flops / sec / 1e12})
        out["render"] = rl
    return out


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    from paper_2008_05858_b200 import build as _build
    if rank == 0:
        _build.build()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        dist.barrier()
    from paper_2008_05858_b200 import binding as B, workloads as W
    B.load()                                             # raises if libe2e.so is missing: no CPU fallback
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    m = measure_device(B, W, torch, args.workload, args.steps, args.warmup, rank, world, dev, args.batch_frames,
                       sampler=ClockSampler(local_rank) if rank == 0 else None)
    scene, r, det, stream, barrier = m["scene"], m["r"], m["det"], m["stream"], m["barrier"]
    contrib, n_samples, nbatch = m["contrib"], m["n_samples"], m["nbatch"]
    value = aggregate_value(world, contrib, m["ms_step"] * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of the spectra, D2H of the frame, every step
    e2e = None
    if not args.no_e2e:
        pinned = {}                                          # fibers that share one table share one pinned copy (and one H2D)
        for sp in scene.spectra:
            if id(sp.flux) not in pinned:
                pinned[id(sp.flux)] = torch.from_numpy(np.ascontiguousarray(sp.flux, dtype=np.float64)).pin_memory()
        host_tabs = [pinned[id(sp.flux)] for sp in scene.spectra]
        desc = B.spectra_array(scene.spectra, [t.data_ptr() for t in host_tabs])
        nbytes = B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc)
        ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        h_frame = torch.empty((scene.ny, scene.nx), dtype=torch.float64).pin_memory()
        h_adu = torch.empty((scene.ny, scene.nx), dtype=torch.uint16).pin_memory()
        h2d = nbatch * sum(int(np.asarray(sp.flux).shape[0]) * 8 for sp in {id(sp.flux): sp for sp in scene.spectra}.values())
        # raw-frame variant: the same stage through the ADC (1 e-/ADU, bias 1000 ADU), delivered as uint16
        adu_desc, _keep = B.detector_ex_desc(W.Detector(gain=det.gain, dark_e=det.dark_e, ron_e=det.ron_e, bias=1000.0, seed=det.seed),
                                             e_per_adu=1.0, adu_max=65535.0)

        def host_step(adu16: bool):
            for dop in m["host_dopplers"]:                    # one host call per frame of the batch (1 frame by default)
                for f in range(len(desc)):
                    desc[f].doppler = float(scene.spectra[f].doppler) * dop
                if adu16:
                    B.e2e_render_frame_host_ex(r.fmt, r.psf, desc, h_adu.data_ptr(), ws, adu_desc, stream=stream, adu16=True)
                else:
                    B.e2e_render_frame_host(r.fmt, r.psf, desc, h_frame.data_ptr(), ws, det=det, stream=stream)   # synchronises

        k_e2e = max(2, min(args.steps, 5))
        res = {}
        for adu16 in (False, True):
            host_step(adu16)                                  # warm-up
            barrier()
            t0 = time.perf_counter()
            for _ in range(k_e2e):
                host_step(adu16)
            barrier()
            res[adu16] = max_over_ranks((time.perf_counter() - t0) / k_e2e, world, dev)
        e2e = {"value": aggregate_value(world, contrib, res[False]), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": nbatch * scene.nx * scene.ny * 8, "ms_per_step": res[False] * 1e3, "steps": k_e2e,
               "call": "e2e_render_frame_host (fp64 electrons out)",
               "adu16": {"value": aggregate_value(world, contrib, res[True]), "unit": UNIT, "h2d_bytes_per_step": h2d,
                         "d2h_bytes_per_step": nbatch * scene.nx * scene.ny * 2, "ms_per_step": res[True] * 1e3, "steps": k_e2e,
                         "call": "e2e_render_frame_host_adu16 (uint16 ADC counts out: the raw frame, P:89 / P:119)"}}
        del ws, h_frame, h_adu

    # ---- the other BASELINE.json configs, device-resident only (parity-test sizes and the other full-size frames)
    others = {}
    if args.others and rank == 0 and world == 1 and nbatch == 1:
        r.close()
        del m["r"]
        torch.cuda.empty_cache()
    if rank != 0:
        return
    # ---- roofline of every stage; the dominant kernel (render) against the FP64 pipe
    burst, sustained = B.e2e_measure_fp64_peak(80)
    peak_tf, burst_tf = 2.0 * sustained / 1e12, 2.0 * burst / 1e12
    stages = stage_rooflines(m, args.workload, peak_tf, burst_tf)
    if "render" in stages:
        stages["render"]["fp64_pipe_probe"] = B.e2e_probe_fp64_pipe()        # why the mix stops short of the peak
    if args.others and world == 1 and nbatch == 1:
        for name in ("tiny", "espresso_like", "hires_like", "field_psf", "rv_sweep"):
            if name == args.workload:
                continue
            o = measure_device(B, W, torch, name, max(3, min(args.steps, 5)), 3, 0, 1, dev)
            st = stage_rooflines(o, name, peak_tf, burst_tf)
            others[name] = {"workload": o["wname"], "n_samples": o["n_samples"], "contributions": o["contrib"],
                            "frame_ms": o["ms_step"], "value": o["contrib"] / (o["ms_step"] * 1e-3), "unit": UNIT,
                            "stage_ms_per_step": o["stage_ms"], "gpu_launches_per_step": o["launches"] / o["steps"],
                            "render_kernel": o["kinfo"]["name"],
                            "stage_roofline_frac": {k: (v["frac"], v["bound"]) for k, v in st.items()},
                            "render_executed_frac": st.get("render", {}).get("executed_frac")}
            o["r"].close()
            del o
            torch.cuda.empty_cache()
        # BASELINE.json configs[4] as a whole: the 5 Doppler-shifted RV-sweep frames in ONE e2e_render_frames call per step
        o = measure_device(B, W, torch, "rv_sweep", max(3, min(args.steps, 5)), 3, 0, 1, dev, 5)
        others["rv_sweep_batch5"] = {"workload": o["wname"] + ", all 5 frames by one e2e_render_frames call + 5 detector calls",
                                     "n_samples": o["n_samples"], "contributions": o["contrib"], "frame_ms": o["ms_step"] / 5.0,
                                     "step_ms": o["ms_step"], "value": o["contrib"] / (o["ms_step"] * 1e-3), "unit": UNIT,
                                     "stage_ms_per_step": o["stage_ms"], "gpu_launches_per_step": o["launches"] / o["steps"],
                                     "render_kernel": o["kinfo"]["name"]}
        o["r"].close()
        del o
        torch.cuda.empty_cache()
    cpu = None
    if not args.no_cpu:
        c = time_oracle(scene, args.oracle_samples)
        cpu = {k: c[k] for k in ("value", "unit", "cores", "kind", "sample")}
    info = m["info"]
    nominal = float(np.floor(2 * m["hbx"]) * np.floor(2 * m["hby"]))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": m["ms_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": m["wname"], "n_samples": n_samples, "contributions": contrib, "footprint_nominal_px": nominal,
                       "chord_nodes_Q": info["n_nodes"], "frame": [scene.ny, scene.nx], "stages": "a1-a6 (zero-fill, setup, render, detector)",
                       "l2": ("inputs larger than L2: cell records %.0f MB + frame %.0f MB vs 126 MB L2" % (m["n_cells"] * (32 + 512 * int(m["kinfo"]["name"].split("<")[1].rstrip(">"))) / 1e6, scene.nx * scene.ny * 8 / 1e6))
                             if m["kinfo"]["name"].startswith("cell_flush_") else
                             ("inputs larger than L2: sample arrays %.0f MB + frame %.0f MB vs 126 MB L2" % (n_samples * 24 / 1e6, scene.nx * scene.ny * 8 / 1e6)),
                       "multi_gpu": "replicas only", "others": others or None},
            "frame_ms": m["ms_step"], "samples_per_s": world * n_samples / (m["ms_step"] * 1e-3),
            "stage_ms_per_step": m["stage_ms"], "stage_roofline": {k: v for k, v in stages.items() if k != "render"},
            "clocks": m["clocks"], "e2e": e2e, "gpu_launches": m["launches"], "roofline": stages.get("render"), "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="espresso_like")
    ap.add_argument("--oracle-samples", type=int, default=1_500_000, help="size of the CPU oracle's bounded sample")
    ap.add_argument("--batch-frames", type=int, default=1, help="render N Doppler-shifted frames per step with e2e_render_frames")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-others", dest="others", action="store_false",
                    help="skip the device-resident numbers of the other BASELINE.json configs (config.others)")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
