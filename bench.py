#!/usr/bin/env python
"""bench.py — EPR projections/s on B200 (BASELINE.json metric), with roofline, e2e and the oracle baseline.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--batch B] [--impl ours|reference]

A step = one pass of the whole hot path (epr_retrieve: Paganin init + `iterations` correction iterations) over
one batch of B synthetic projections of the named config (default C2: 2048x2048, monochromatic, local O(L^2)
solver, 20 iterations — the configuration the metric is quoted on).  B distinct noisy projections (B x plane
>> L2) are resident in HBM when the timed region starts.  N > 1 (torchrun): every rank runs its own batch on
its own GPU (projections are independent units: weak scaling, no data-path collective); the time is the max
over ranks.  `--impl reference` times the fp64 numpy oracle on the host cores instead.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "EPR projections/s (2048^2, 20 iters) on 1 B200; % HBM roofline per kernel"
UNIT = "projections/s"


# ---- algorithmic bytes per pixel per LAUNCH of each kernel family (fp32) ----
def kernel_bytes_per_px(name, nb, solver):
    return {
        "k_forward_local": 12 if nb == 1 else 4 + 4 * nb,   # 1 line: fused march R tau, R d, W e; else R tau, W (P_s - f_s) x nb
        # splat with the residual (a2) fused: R tau, R d, W e_s x nb.  Not counted: the second read of tau by the
        # block-maximum prepass and the N prediction planes that stay in L2 between flush and split (design overheads)
        "k_splat": 8 + 4 * nb,
        "k_residual": 4 + 8 * nb,               # R d, R pred x nb, W e_s x nb
        "k_gather": 4 + 8 * nb,                 # R tau, R e_s x nb, W r_s x nb
        "k_rows_r2c": 8,                        # per plane: R 4, W half spectrum 4
        "k_cols": 4 * nb + 4,                   # R nb spectra, W summed spectrum
        "k_rows_c2r": 12,                       # R spectrum 4, R tau 4, W tau 4
        "k_output": 8,
        "k_resample": 8,                        # replaced per call by 4 + 4/m² (see main)
        "k_pred_out": 4 * nb + 4,
        "k_update": 16,                         # general path: R two block-filtered planes (non-zero weights), R tau, W tau
        "k_diagnostics": 4 * nb + 4,
        "k_wkb1_sub": 4 + 8 * nb,
    }[name]


def max_over_ranks(value, device):
    """Max over ranks of a per-rank scalar (the timing reduction of the N > 1 path; works on gloo and nccl)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


TRAFFIC_FILE = os.path.join("profiles", "r3_dram_traffic.json")


def measured_traffic(epr, kernel, nb, solver, config, algorithmic_bytes_per_launch):
    """DRAM bytes per launch of `kernel` from the committed `ncu --set full` capture (TRAFFIC_FILE: per kernel and
    configuration, dram__bytes_read.sum + dram__bytes_write.sum of one launch divided by that launch's algorithmic
    bytes), scaled to this run's launch size.  The capture names the library version it was taken from; when the
    library loaded now reports another version the number is stale and null is returned instead.
    Returns (bytes per launch or None, provenance string)."""
    path = os.path.join(ROOT, TRAFFIC_FILE)
    try:
        tab = json.load(open(path))
    except Exception:
        return None, f"{TRAFFIC_FILE} absent"
    lib_now = epr.load_library().epr_version().decode()
    if tab.get("lib_version") != lib_now:
        return None, f"{TRAFFIC_FILE} was captured from '{tab.get('lib_version')}', library is '{lib_now}': stale, dropped"
    ratio = tab.get("dram_over_algorithmic", {}).get(f"{config}:{kernel}")
    if ratio is None:
        return None, f"{TRAFFIC_FILE} has no capture of {kernel} at {config}"
    return ratio * algorithmic_bytes_per_launch, f"{TRAFFIC_FILE} ({tab.get('command', 'ncu --set full')}; {tab.get('lib_version')})"


def issue_ceiling(epr, kernel, config, sm_mhz, px_lines_per_launch, avg_ms):
    """The secondary ceiling SURVEY.md §8(d) names, for kernels that instruction issue bounds rather than HBM: executed warp
    instructions per pixel and line and the IPC of the committed `ncu --set full` capture (TRAFFIC_FILE, version-checked like
    `traffic`), and the fraction of the SM's issue peak THIS run reached — instructions of one launch (inst_per_px_line x pixel-lines
    / 32) over what 148 SMs issuing 4 warp instructions per clock at the sampled SM clock could issue in the measured launch time."""
    try:
        tab = json.load(open(os.path.join(ROOT, TRAFFIC_FILE)))
    except Exception:
        return None
    if tab.get("lib_version") != epr.load_library().epr_version().decode():
        return None
    ent = tab.get("issue", {}).get(f"{config}:{kernel}")
    if ent is None or not sm_mhz:
        return None
    warp_inst = ent["inst_per_px_line"] * px_lines_per_launch / 32.0
    peak = 4.0 * 148 * sm_mhz * 1e6 * (avg_ms * 1e-3)
    return {"inst_per_px_line": ent["inst_per_px_line"], "ipc_ncu": ent["ipc"], "frac_of_issue_peak": warp_inst / peak,
            "derivation": "inst_per_px_line x pixel-lines per launch / 32 warp instructions over 4 per clock x 148 SMs x the sampled SM "
                          f"clock ({sm_mhz:.0f} MHz) x the launch time measured in this run; counts from {TRAFFIC_FILE}"}


def expected_launches_per_step(kernel, w, m, blocks=0):
    """Launches of a kernel family in one epr_retrieve over a batch that fits the plan's work batch."""
    it = w.iterations
    if blocks > 0:                                  # general path: block filters, splat = scatter + conversion
        return {"k_rows_r2c": it + 1, "k_cols": (it + 1) * blocks, "k_rows_c2r": (it + 1) * blocks, "k_update": it + 1,
                "k_splat": it if (w.nx % 16 == 0 and w.ny % 16 == 0) else 2 * it, "k_resample": 2}.get(kernel, it)
    return {"k_rows_r2c": it + 1, "k_cols": it + 1, "k_rows_c2r": it + 1, "k_resample": 2}.get(kernel, it)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms during the timed region."""

    def __init__(self, index):
        self.index, self.rows, self.proc, self.start = index, [], None, 0

    def __enter__(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
            t0 = time.time()
            while not self.rows and time.time() - t0 < 3.0:      # nvidia-smi needs a moment before its first sample
                time.sleep(0.01)
        except Exception:
            self.proc = None
        self.start = len(self.rows)                              # samples before the timed region are dropped
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.05)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows[self.start:]:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for n, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def override_lines(w, n):
    """Retrieval with n spectral lines on the config's detector data (only the spectral discretisation the retrieval
    assumes changes): E = linspace(60, 140) keV, Gaussian weights (sigma 20 keV), delta/beta proportional to E."""
    db100 = float(w.delta_over_beta[np.argmin(np.abs(w.energy_keV - 100.0))])
    e = np.linspace(60.0, 140.0, n) if n > 1 else np.array([100.0])
    wt = np.exp(-0.5 * ((e - 100.0) / 20.0) ** 2)
    w.energy_keV, w.weight, w.delta_over_beta = e, wt / wt.sum(), db100 * e / 100.0


def fine_shift_clamp(w, m):
    """S in pixels of the grid refined m times (the library accepts at most 30)."""
    return float(min(30.0, m * w.max_shift_px))


def workload_string(name, w, m=1, blocks=0):
    """`config.workload` of both arms (the driver compares the two strings)."""
    return (f"{name}: {w.ny}x{w.nx}, {w.n_bins} line(s), {w.solver} solver, {w.iterations} iterations, step {w.step}"
            + (f", oversampling {m} (computational grid {m * w.ny}x{m * w.nx})" if m > 1 else "")
            + (f", x-dependent spectrum on {blocks} blocks (general path)" if blocks > 0 else ""))


def oracle_time_one(w, j=0, m=1):
    """The oracle as it stands, one projection of the workload, on the host cores (numpy: 1 thread).  Returns (seconds,
    the oracle's result): the result is compared with the GPU's output for the same projection (`parity`)."""
    from oracle import epr_oracle as O
    lines = O.derive_lines(w.pixel_m / m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    t0 = time.perf_counter()
    if m == 1:
        tau = O.retrieve(w.d[j].astype(np.float64), lines, w.solver, w.iterations, w.step, S=w.max_shift_px)
    else:
        tau = O.retrieve_oversampled(w.d[j].astype(np.float64), lines, m, w.solver, w.iterations, w.step, S=fine_shift_clamp(w, m))
    return time.perf_counter() - t0, tau


def parity_of(gpu_tau, oracle_tau):
    """The oracle acting as checker, outside every timed region: the GPU's result for one projection of the timed
    batch against the oracle's for the same input (north_star: retrieved thickness / phase within 1e-4 relative L2)."""
    g = np.asarray(gpu_tau, dtype=np.float64)
    r = np.asarray(oracle_tau, dtype=np.float64)
    return {"rel_l2": float(np.linalg.norm(g - r) / np.linalg.norm(r)),
            "max_rel": float(np.max(np.abs(g - r)) / np.max(np.abs(r))), "tolerance_rel_l2": 1e-4,
            "what": "tau of projection 0 of the timed batch, all iterations: GPU (epr_retrieve) vs the fp64 oracle"}


def _oracle_sample_worker(a):
    """One host process of the bounded oracle sample: the initial Paganin solve alone (iterations = 0) and the initial
    solve plus ONE correction iteration on one projection; returns the two wall times."""
    (d, pixel_m, L_m, energy, weight, db, solver, step, S) = a
    from oracle import epr_oracle as O
    lines = O.derive_lines(pixel_m, L_m, energy, weight, db)
    d64 = d.astype(np.float64)
    t0 = time.perf_counter()
    O.retrieve(d64, lines, solver, 0, step, S=S)
    t1 = time.perf_counter()
    O.retrieve(d64, lines, solver, 1, step, S=S)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1


def host_procs(w):
    """All host cores, unless the host's free memory cannot hold that many oracle processes (one fp64 retrieval keeps
    about 5 planes per line alive: ~45 planes of 8 bytes per pixel for 8 lines)."""
    cores = os.cpu_count() or 1
    try:
        import psutil
        need = 8.0 * w.nx * w.ny * (6 * w.n_bins + 8) * 1.5
        cores = max(1, min(cores, int(psutil.virtual_memory().available * 0.6 / need)))
    except Exception:
        pass
    return cores


def oracle_sample(w, procs):
    """Bounded sample of the oracle for the expensive configurations (a full 8-line retrieval takes minutes per
    projection): `procs` host processes (multiprocessing, one projection each, all running at once, so that memory
    bandwidth contention is in the number) time the initial solve and the initial solve + 1 iteration; the cost of the
    workload's `iterations` is extrapolated linearly, t = t_init + iterations · (t_1 − t_init) — every iteration of the
    oracle does the same work.  Returns the cpu_baseline object."""
    import multiprocessing as mp
    B = w.d.shape[0]
    idx = [0, B // 2, B - 1] if B >= 3 else list(range(B))           # projections 0 / 31 / 63 of C5
    jobs = [(w.d[idx[k % len(idx)]], w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver, w.step,
             w.max_shift_px) for k in range(procs)]
    t0 = time.perf_counter()
    if procs == 1:
        res = [_oracle_sample_worker(jobs[0])]
    else:
        with mp.get_context("spawn").Pool(procs) as pool:
            res = pool.map(_oracle_sample_worker, jobs)
    wall = time.perf_counter() - t0
    t_init = max(r[0] for r in res)
    t_one = max(r[1] for r in res)
    t_full = t_init + w.iterations * max(t_one - t_init, 0.0)
    return {"value": procs / t_full, "unit": UNIT, "cores": procs, "kind": "oracle",
            "sample": f"{procs} process(es) x 1 projection ({w.ny}x{w.nx}, {w.n_bins} line(s)) at once: initial solve "
                      f"{t_init:.2f} s, initial solve + 1 iteration {t_one:.2f} s (slowest process); extrapolated to "
                      f"{w.iterations} iterations = {t_full:.1f} s per projection per process; sample wall {wall:.1f} s; "
                      f"numpy fp64, host has {os.cpu_count()} cores"}


def cufft_compare(epr, plan, B, reps=5):
    """Comparison point only (north_star: "a cuFFT-based variant is kept only as a reported comparison point"): the
    a4 preconditioner q_s = IFFT2(H_s FFT2(r_s)), H_s = 1/(1 + a_s λ) with the discrete 5-point symbol (PAPER.md:51,
    reading R5), once through epr_precondition (the library's own row/column FFT kernels) and once through cuFFT
    (torch.fft.rfft2 · H · irfft2) on the same device planes.  Nothing on the product path calls this."""
    import torch
    nb, ny, nx = plan.n_bins, plan.ny, plan.nx
    Bc = max(1, min(B, 256 // max(nb, 1), 16))     # planes of both variants plus the cuFFT spectra stay within a few GB
    g = torch.Generator(device="cuda").manual_seed(7)
    r = torch.randn((Bc, nb, ny, nx), device="cuda", dtype=torch.float32, generator=g)
    q = torch.empty_like(r)
    a = torch.tensor(plan.lines()["a"], device="cuda", dtype=torch.float64)
    th_y = 2 * math.pi * torch.fft.fftfreq(ny, device="cuda", dtype=torch.float64)
    th_x = 2 * math.pi * torch.fft.rfftfreq(nx, device="cuda", dtype=torch.float64)
    lam = (2 - 2 * torch.cos(th_y))[:, None] + (2 - 2 * torch.cos(th_x))[None, :]
    H = (1.0 / (1.0 + a[:, None, None] * lam[None])).to(torch.float32)          # [nb][ny][nx/2+1]

    def ours():
        epr.epr_precondition(plan, r, q)

    def cufft():
        return torch.fft.irfft2(torch.fft.rfft2(r) * H, s=(ny, nx))

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps
    t_ours, t_cufft = timed(ours), timed(cufft)
    ref = cufft()
    diff = float(torch.linalg.vector_norm((q - ref).double()) / torch.linalg.vector_norm(ref.double()))
    del r, q, ref, H
    torch.cuda.empty_cache()
    return {"op": "epr_precondition (a4) on %d x %d line(s) x %dx%d" % (Bc, nb, ny, nx),
            "ours_us_per_plane": 1e3 * t_ours / (Bc * nb), "cufft_us_per_plane": 1e3 * t_cufft / (Bc * nb),
            "cufft_over_ours": t_cufft / t_ours, "rel_l2_between": diff,
            "note": "cuFFT leg = torch.fft.rfft2 * H -> irfft2 (library kernels, comparison point only)"}


def oracle_time_iters(w, n_it, m=1, j=0):
    """The oracle as it stands on one projection of the workload with n_it correction iterations (initial solve included)."""
    from oracle import epr_oracle as O
    lines = O.derive_lines(w.pixel_m / m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta)
    d64 = w.d[j].astype(np.float64)
    t0 = time.perf_counter()
    if m == 1:
        O.retrieve(d64, lines, w.solver, n_it, w.step, S=w.max_shift_px)
    else:
        O.retrieve_oversampled(d64, lines, m, w.solver, n_it, w.step, S=fine_shift_clamp(w, m))
    return time.perf_counter() - t0


def run_reference(args, rank):
    """`--impl reference`: the fp64 numpy oracle on one host core.  A step is one projection of the workload; so that the
    whole `--steps K --warmup W` run stays within `--ref-budget` seconds (default 150), a step runs the initial solve and
    the first n of the workload's iterations, n chosen from an untimed calibration (initial solve alone, t_0; initial solve
    + 1 iteration), and its time is extrapolated to all iterations, t = t_0 + iterations (t_step − t_0) / n — every
    iteration of the oracle does the same work.  n = all iterations (no extrapolation) whenever the budget allows."""
    if rank != 0:
        return
    from epr_inputs import make_workload
    w = make_workload(args.config, batch=1, distinct=1)
    if args.lines > 0:
        override_lines(w, args.lines)
    m = args.oversample
    c0 = float(np.median([oracle_time_iters(w, 0, m) for _ in range(3)]))     # initial solve alone: median of three
    c1 = oracle_time_iters(w, 1, m)
    t_iter = max(c1 - c0, 1e-3)
    per_step = (args.ref_budget - 4 * c0 - t_iter) / max(1, args.steps + args.warmup)
    n_it = int(max(1, min(w.iterations, (per_step - c0) // t_iter)))
    for _ in range(args.warmup):
        oracle_time_iters(w, n_it, m)
    t = np.array([oracle_time_iters(w, n_it, m) for _ in range(args.steps)])
    full = t if n_it == w.iterations else c0 + w.iterations * np.maximum(t - c0, 0.0) / n_it
    tot = float(np.sum(full))
    val = args.steps / tot
    if n_it == w.iterations:
        sample = f"1 projection {w.ny}x{w.nx} per step, all {w.iterations} iterations, numpy fp64 oracle"
    else:
        sample = (f"1 projection {w.ny}x{w.nx} per step: initial solve + the first {n_it} of {w.iterations} iterations "
                  f"({float(np.mean(t)):.2f} s per step measured), extrapolated linearly to all iterations with the initial "
                  f"solve of the calibration ({c0:.2f} s, median of 3); numpy fp64 oracle; run bounded to {args.ref_budget:.0f} s")
    # ONE time base in the line: value, ms_per_step, cpu_baseline and e2e all describe the full workload (extrapolated where
    # the budget cut the iterations); what was actually timed per step sits in config.ms_per_step_measured
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(args.config, w, m),
                   "iterations_run_per_step": n_it, "ms_per_step_measured": 1e3 * float(np.mean(t)),
                   "extrapolated": bool(n_it != w.iterations)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def block_profiles(w, n_blocks):
    """Synthetic x-dependent effective spectrum for `--blocks` (beam hardening stronger at the centre of a
    cylindrical container): the weights tilt towards the high-energy lines and delta/beta rises by up to 10 % at the centre."""
    t = 1.0 - np.abs(np.linspace(-1.0, 1.0, n_blocks))[:, None]            # 0 at the edges, 1 at the centre
    e = (np.asarray(w.energy_keV, dtype=np.float64) - 100.0) / 40.0
    wt = np.asarray(w.weight, dtype=np.float64)[None, :] * (1.0 + 0.4 * t * e[None, :])
    db = np.asarray(w.delta_over_beta, dtype=np.float64)[None, :] * (1.0 + 0.1 * t)
    return wt, db


def measure_config(epr, name, B, steps, warmup, distinct, rank, world, local, lines=0, m=1, cufft=False, blocks=0, n=None,
                   S_fine=None):
    """Time one configuration: K steps of epr_retrieve over B resident projections (CUDA events on the launch stream),
    the same through epr_retrieve_host with pinned host buffers, and a profiling pass with the in-library per-kernel
    events.  Returns the pieces of the JSON line for this configuration (everything already reduced over ranks)."""
    import torch
    import torch.distributed as dist
    from epr_inputs import make_workload

    # N > 1: ONE seeded batch of N x B projections, rank k retrieves its contiguous share [lo, hi) (shard_range; no
    # data-path collective: projections are independent) — generated by the rank that needs it
    from epr_inputs import shard_range
    lo, hi = shard_range(world * B, rank, world)
    w = make_workload(name, n=n, batch=hi - lo, distinct=min(distinct, B), first=lo)
    if lines > 0:
        override_lines(w, lines)
    plane = w.nx * w.ny
    nb = w.n_bins
    plan = epr.epr_plan(m * w.nx, m * w.ny, w.pixel_m / m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver,
                        max_batch=B, max_shift_px=w.max_shift_px if m == 1 else (S_fine or fine_shift_clamp(w, m)))
    if blocks > 0:                                  # x-dependent effective spectrum (reading R17): the general path
        epr.epr_plan_profiles(plan, *block_profiles(w, blocks))
    d_host = torch.from_numpy(w.d).pin_memory()
    out_host = torch.empty_like(d_host).pin_memory()
    d = d_host.cuda()
    out = torch.empty_like(d)

    def step():
        if m == 1:
            epr.epr_retrieve(plan, d, out, w.iterations, w.step)
        else:
            epr.epr_retrieve_oversampled(plan, m, d, out, w.iterations, w.step)

    def step_host():
        epr.epr_retrieve_host(plan, d_host, out_host, w.iterations, w.step, factor=m)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # L2 policy: a step streams B input planes plus the plan's workspaces (several times B planes) through HBM, so
    # consecutive steps cannot reuse L2 contents when B x plane > L2; for smaller batches L2 is flushed (a 256 MB
    # device buffer is overwritten) between timed steps, outside the timed region.
    in_bytes = B * plane * 4
    flush = None
    if in_bytes <= 2 * 126e6:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(warmup):
        step()
    barrier()
    l0 = plan.launches
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    with ClockSampler(local) as clk:
        for e0, e1 in evs:
            if flush is not None:
                flush.fill_(1)
            e0.record()
            step()
            e1.record()
        barrier()
    ms = sum(e0.elapsed_time(e1) for e0, e1 in evs)
    launches = plan.launches - l0
    ms = max_over_ranks(ms, torch.device("cuda", local))
    value = world * B * steps / (ms * 1e-3)

    # ---- end to end through the public host API: pinned host buffers, H2D + loop + D2H inside the timed region.
    # (i) per call: every epr_retrieve_host waits for its own last copy; (ii) the streaming session of PAPER.md:245
    # (epr_retrieve_host_async x K, one epr_host_wait): the K batches follow each other as the chunks of a scan do, every
    # copy in and every copy out still inside the timed region — the headline e2e where the API offers it (factor 1)
    step_host()
    barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        step_host()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, torch.device("cuda", local))
    e2e_call = world * B * steps / e2e_s
    e2e, e2e_api = e2e_call, "epr_retrieve_host (pinned host buffers, chunks double-buffered on three streams), one call per step"
    if m == 1:
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            epr.epr_retrieve_host(plan, d_host, out_host, w.iterations, w.step, wait=False)
        epr.epr_host_wait(plan)
        e2e_s = time.perf_counter() - t0
        e2e_s = max_over_ranks(e2e_s, torch.device("cuda", local))
        e2e = world * B * steps / e2e_s
        e2e_api = (f"epr_retrieve_host_async x {steps} + epr_host_wait (streaming session: pinned host buffers, chunks "
                   "double-buffered on three streams across consecutive batches); per_call = epr_retrieve_host, one call per step")

    # ---- per-kernel device times (CUDA events around every launch, on the launch stream), same K steps
    plan.profile(True)
    for _ in range(steps):
        step()
    prof = plan.profile_read()
    plan.profile(False)
    flags = plan.read_flags()

    cmp_cufft = None
    if rank == 0 and m == 1 and cufft:
        try:
            cmp_cufft = cufft_compare(epr, plan, B)
        except Exception as exc:                    # a comparison point must never cost the bench line
            cmp_cufft = {"error": f"{type(exc).__name__}: {exc}"[:200]}

    peak, peak_src = peaks()
    per_kernel = []
    for kname, (tot_ms, cnt) in prof.items():
        bpp = kernel_bytes_per_px(kname, nb, w.solver)
        # px per launch: every launch covers the whole batch; r2c covers nb planes per projection in the loop
        launches_per_step = cnt / steps
        px = B * plane * m * m                  # pixels of the computational grid
        if kname == "k_rows_r2c":
            # (iterations launches of nb planes + 1 init launch of 1 plane) per step
            px = px * (w.iterations * nb + 1) / (w.iterations + 1)
        if kname == "k_resample":                # replication: R 4/m² + W 4; block mean: R 4 + W 4/m²; one launch each
            bpp = 4.0 + 4.0 / (m * m)
        # a batch larger than the plan's work batch goes through the loop in passes: launches cover B / passes projections
        passes = max(1, round(launches_per_step / expected_launches_per_step(kname, w, m, blocks)))
        if blocks > 0 and kname == "k_rows_c2r":
            bpp = 8                                 # general path: plain inverse transform (R spectrum, W q)
        px = px / passes
        avg_ms = tot_ms / cnt
        gbs = bpp * px / (avg_ms * 1e-3) / 1e9
        per_kernel.append({"kernel": kname, "launches_per_step": launches_per_step, "avg_ms": avg_ms, "passes": passes,
                           "share": None, "algorithmic_bytes_per_launch": bpp * px, "achieved_gbs": gbs,
                           "frac": gbs / peak})
    tot = sum(k["avg_ms"] * k["launches_per_step"] for k in per_kernel)
    for k in per_kernel:
        k["share"] = k["avg_ms"] * k["launches_per_step"] / tot
    per_kernel.sort(key=lambda k: -k["share"])
    dom = per_kernel[0]
    traffic, traffic_src = measured_traffic(epr, dom["kernel"], nb, w.solver, name, dom["algorithmic_bytes_per_launch"])
    # whole-iteration view: algorithmic bytes of one iteration (sum over the loop's kernels) over the time per iteration
    roofline = {"bound": "hbm", "kernel": dom["kernel"], "achieved": dom["achieved_gbs"], "peak": peak,
                "unit": "GB/s", "frac": dom["frac"], "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src, "per_kernel": per_kernel}
    issue = issue_ceiling(epr, dom["kernel"], name, clk.summary().get("sm_mhz"), B * plane * m * m * nb / dom.get("passes", 1),
                          dom["avg_ms"])
    if issue is not None:
        roofline["issue"] = issue
    res = {
        "value": value, "unit": UNIT, "ms_per_step": ms / steps, "steps": steps, "warmup": warmup,
        "config": {"workload": workload_string(name, w, m, blocks),
                   "batch_per_gpu": B, "global_batch": world * B, "sharding": "contiguous ranges of one seeded batch, no collective",
                   "distinct_projections": min(distinct, B),
                   "l2": (f"inputs {in_bytes / 1e6:.0f} MB per step > 2 x 126 MB L2: no flush needed" if flush is None else
                          f"inputs {in_bytes / 1e6:.0f} MB per step: L2 flushed (256 MB overwrite) between timed steps"),
                   "ms_per_iteration_per_projection": ms / steps / B / (w.iterations + 1)},
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": B * plane * 4, "d2h_bytes_per_step": B * plane * 4,
                "per_call": e2e_call, "api": e2e_api},
        "gpu_launches": int(launches) * world,
        "clocks": clk.summary(),
        "roofline": roofline,
        "flags": flags,
    }
    if cmp_cufft is not None:
        res["cufft_compare"] = cmp_cufft
    if m > 1:
        res["config"]["max_shift_fine_px"] = float(S_fine or fine_shift_clamp(w, m))
    step()
    torch.cuda.synchronize()
    res["_tau0"] = out[0].cpu().numpy()             # for `parity` (popped before the line is printed)
    plan.destroy()
    del d, out, d_host, out_host, flush
    torch.cuda.empty_cache()
    return res, w


def measure_c1(epr, local, calls=200):
    """BASELINE.json configs[0] (C1: ONE 256 x 256 projection, local solver, 10 iterations — launch-bound): microseconds per
    epr_retrieve on a non-default stream, launched kernel by kernel (EPR_GRAPH = 0 at plan time) and as the CUDA graph the
    library captures on the second identical call and replays afterwards (include/epr.h, epr_retrieve)."""
    import torch
    from epr_inputs import make_workload
    w = make_workload("C1")
    d = torch.from_numpy(w.d).cuda()
    out = torch.empty_like(d)
    st = torch.cuda.Stream()
    res = {}
    for mode, env in (("eager", "0"), ("graph", "1")):
        os.environ["EPR_GRAPH"] = env
        plan = epr.epr_plan(w.nx, w.ny, w.pixel_m, w.L_m, w.energy_keV, w.weight, w.delta_over_beta, w.solver, max_batch=1)
        os.environ.pop("EPR_GRAPH")
        with torch.cuda.stream(st):
            for _ in range(5):
                epr.epr_retrieve(plan, d, out, w.iterations, w.step)
            st.synchronize()
            l0 = plan.launches
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record(st)
            for _ in range(calls):
                epr.epr_retrieve(plan, d, out, w.iterations, w.step)
            e1.record(st)
            st.synchronize()
            wall = time.perf_counter() - t0
        res[mode] = {"us_per_retrieval_device": 1e3 * e0.elapsed_time(e1) / calls, "us_per_retrieval_wall": 1e6 * wall / calls,
                     "kernel_launches_per_retrieval": (plan.launches - l0) / calls}
        plan.destroy()
    res["config"] = {"workload": workload_string("C1", w), "batch": 1, "calls": calls,
                     "l2": "one 256 KB plane: deliberately L2-resident (the configuration is launch-bound, not HBM-bound)"}
    res["value"] = 1e6 / res["graph"]["us_per_retrieval_device"]
    res["unit"] = UNIT
    res["summary"] = [round(res["value"], 1), None, f"graph {res['graph']['us_per_retrieval_device']:.0f} us / eager "
                      f"{res['eager']['us_per_retrieval_device']:.0f} us per retrieval", None, None]
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2")
    ap.add_argument("--batch", type=int, default=0, help="projections per GPU and step (default: 64 for C2 / C3 / C5, 8 for C4)")
    ap.add_argument("--distinct", type=int, default=2, help="distinct simulated projections (rest: new noise only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-budget", type=float, default=150.0, help="--impl reference: seconds the whole run may take")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft-compare", action="store_true",
                    help="skip the preconditioner-through-cuFFT comparison point (rank 0, outside every timed region)")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="headline configuration only: skip the C3 / C4 / C5 sub-results of the default run")
    ap.add_argument("--lines", type=int, default=0,
                    help="retrieve with this many spectral lines (60-140 keV, Gaussian weights) instead of the config's own "
                         "discretisation, e.g. --config C2 --lines 5: the paper's 'local L2 poly' rows (PAPER.md:116-119)")
    ap.add_argument("--blocks", type=int, default=0,
                    help="x-dependent effective spectrum on this many blocks (PAPER.md:431-441; epr_plan_profiles, general path)")
    ap.add_argument("--oversample", type=int, default=1,
                    help="run the loop on the grid refined this many times (PAPER.md:79; epr_retrieve_oversampled)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2601_22793_b200 as epr

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    args.warmup = max(args.warmup, 3)
    default_batch = {"C1": 64, "C2": 64, "C3": 64, "C4": 8, "C5": 64}
    B = args.batch if args.batch > 0 else default_batch[args.config]

    head, w = measure_config(epr, args.config, B, args.steps, args.warmup, args.distinct, rank, world, local,
                             lines=args.lines, m=args.oversample, cufft=not args.no_cufft_compare, blocks=args.blocks)
    result = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
              "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
              "vs_baseline": None, "dtype": "f32", "data": "synthetic"}
    for k in ("config", "e2e", "gpu_launches", "clocks", "roofline", "flags", "cufft_compare"):
        if k in head:
            result[k] = head[k]
    tau_gpu = head.pop("_tau0")
    if rank == 0 and not args.no_cpu_baseline:
        t1, tau_ref = oracle_time_one(w, m=args.oversample)
        result["cpu_baseline"] = {"value": 1.0 / t1, "unit": UNIT, "cores": 1, "kind": "oracle",
                                  "sample": f"1 of the {B} projections ({w.ny}x{w.nx}, all {w.iterations} "
                                            f"iterations) in {t1:.1f} s, numpy fp64, host has {os.cpu_count()} cores"}
        result["parity"] = parity_of(tau_gpu, tau_ref)
        del tau_ref
    del w, tau_gpu

    def compact(r):
        """[projections/s device-resident, through host buffers, dominant kernel, its HBM fraction, median SM MHz]"""
        if "error" in r:
            return r["error"][:80]
        return [round(r["value"], 1), round(r["e2e"]["value"], 1), r["roofline"]["kernel"], round(r["roofline"]["frac"], 3),
                r["clocks"].get("sm_mhz")]

    summary = {args.config: compact(head)}
    # ---- the other BASELINE.json configurations, each measured the same way (same protocol, fewer steps), in the same
    # line: C3 (non-local, one line), C4 (non-local, 8 lines), C5 (2560 x 2160, 8 lines, batch 64 — more than the
    # plan's work batch holds, so the device call passes through HBM in sub-batches and the host call streams chunks);
    # then the SURVEY.md §8(f) shapes: the oversampled loop and the x-dependent spectrum,
    # and BASELINE.json configs[0] (C1: one 256 x 256 retrieval, launch-bound, eager and as a replayed CUDA graph)
    default_run = (args.config == "C2" and args.lines == 0 and args.oversample == 1 and args.batch == 0 and args.blocks == 0)
    if default_run and not args.no_other_configs:
        other = {}
        # the splat's ring width and candidate list depend on the data: these batches hold more distinct projections
        # (C5: 8 different rotation angles of the phantom) than the headline's local solver needs
        for name, ob, osteps, odist in (("C3", 64, 3, 4), ("C4", 8, 3, 4), ("C5", 64, 2, 8)):
            try:
                r, ow = measure_config(epr, name, ob, osteps, 3, max(args.distinct, odist), rank, world, local)
                tau_gpu = r.pop("_tau0")
                if rank == 0 and not args.no_cpu_baseline:
                    if name == "C3":               # one line: the full 20 iterations of one projection fit the budget
                        t1, tau_ref = oracle_time_one(ow)
                        r["cpu_baseline"] = {"value": 1.0 / t1, "unit": UNIT, "cores": 1, "kind": "oracle",
                                             "sample": f"1 of the {ob} projections ({ow.ny}x{ow.nx}, all {ow.iterations} "
                                                       f"iterations) in {t1:.1f} s, numpy fp64"}
                        r["parity"] = parity_of(tau_gpu, tau_ref)
                        del tau_ref
                    else:
                        r["cpu_baseline"] = oracle_sample(ow, host_procs(ow) if name == "C5" else 1)
                del ow, tau_gpu
                other[name] = r
            except Exception as exc:                # a sub-result must never cost the headline
                other[name] = {"error": f"{type(exc).__name__}: {exc}"[:300]}
            summary[name] = compact(other[name])
        extra = (("C2_x2", dict(name="C2", B=8, m=2)),                                     # local, x2: 4096 x 4096
                 ("C3_1024_x4", dict(name="C3", B=8, m=4, n=1024, S_fine=30.0)),            # non-local, x4: 4096 x 4096
                 ("C2_blocks4", dict(name="C2", B=16, blocks=4)), ("C4_blocks4", dict(name="C4", B=4, blocks=4)))
        for key, kw in extra:
            try:
                r, ow = measure_config(epr, kw["name"], kw["B"], 2, 3, 2, rank, world, local, m=kw.get("m", 1),
                                       blocks=kw.get("blocks", 0), n=kw.get("n"), S_fine=kw.get("S_fine"))
                r.pop("_tau0")
                r["roofline"].pop("per_kernel", None)            # keep the line short: the headline configs carry the tables
                del ow
                other[key] = r
            except Exception as exc:
                other[key] = {"error": f"{type(exc).__name__}: {exc}"[:300]}
            summary[key] = compact(other[key])
        try:
            other["C1"] = measure_c1(epr, local)
            summary["C1"] = other["C1"]["summary"]
        except Exception as exc:
            other["C1"] = {"error": f"{type(exc).__name__}: {exc}"[:300]}
            summary["C1"] = other["C1"]["error"][:80]
        result["other_configs"] = other
    # LAST in the line, so that a reader who keeps only its tail still sees every configuration
    result["summary"] = {"columns": ["projections/s device-resident", "projections/s through host buffers", "dominant kernel",
                                     "its fraction of the HBM peak", "median SM MHz"], **summary}
    if rank == 0:
        print(json.dumps(result))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
