#!/usr/bin/env python
"""bench.py — one JSON line for the TACAW hot path on B200 (contract: task prompt / DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] ...

A "step" is one pass of the whole hot path over one batch of synthetic input:
    ps_build_slices -> ps_make_incident -> ps_multislice -> ps_tacaw -> ps_sdp / ps_spectrum_image /
    ps_dispersion / ps_qbin.
Default workload = the largest single-GPU configuration of BASELINE.json, config 3 (Si 8x8x20, 10 240 atoms, 512^2,
80 slices, 30 mrad probe, 1024 frames) in the unit its full run is made of: ONE 16-probe scan row x all 1024 frames
(V of all frames 86 GB + exit waves 34 GB + I(k,w) 17 GB resident: the chunk `--full-config c3` loops 16 times).
`value` = nx*ny*n_slices*frames*probes / step time in Gpx*slice/s, inputs resident in HBM; `e2e` = the same through
the public API with pinned host positions in and the reductions a caller keeps out, copies inside the timed region.
`roofline` is for the dominant kernel of the step (per-launch CUDA events recorded by the library on its own stream
in a second pass of the same K steps); `cpu_baseline` is the float64 oracle timed on all host cores on a bounded
sample of the same workload.  With N > 1 (torchrun): `--scaling weak` (default) gives every rank an independent
trajectory and averages the reductions with one all-reduce; `--scaling strong` shards ONE problem
(paper_2602_10064_b200/sharding.py: probe shards, or frame shards + reduce-scatter of the per-bin accumulators).
`--impl reference` times the oracle (the only reference there is: the paper ships no code).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import form_factor_coefficients, make_workload  # noqa: E402

METRIC = "multislice Gpx*slice/s over frames x probes (whole TACAW hot path per step)"
UNIT = "Gpx*slice/s"
N_SM, LANES_PER_SM = 148, 128          # B200: 148 SMs x 4 schedulers x 32 lanes issue one instruction per clock each


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 1590.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1590.0, "fallback (B200_PROFILING.md: 6.65 TB/s, 1.59 PFLOP/s)"


STATS_SOURCES = ("multislice.cu", "resident.cu", "tacaw.cu", "fft_core.cuh", "tma.cuh")


def library_source_sha16():
    """sha256[:16] over the CUDA sources the slice-step, resident and time-transform kernels are built from."""
    import hashlib
    h = hashlib.sha256()
    for f in STATS_SOURCES:
        with open(os.path.join(ROOT, "paper_2602_10064_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def kernel_stats():
    """ncu-derived per-kernel constants (DRAM bytes and thread instructions per pixel of one wave, keyed by kernel<N>),
    taken from --set full captures named in the profile notes.  They describe the kernels of ONE source state: the file
    carries `_source_sha16` (library_source_sha16() when it was captured) and is ignored — `traffic` and `fp32_issue`
    print as null — when the sources have changed since, instead of silently quoting figures of older kernels."""
    for name in ("r3_kernel_stats.json", "r2_kernel_stats.json"):
        path = os.path.join(ROOT, "profiles", name)
        if os.path.exists(path):
            with open(path) as fh:
                d = json.load(fh)
            if d.get("_source_sha16") == library_source_sha16():
                d["_file"] = name
                return d
    return {}


def band_columns(cell, nx, ny):
    """Number of k-columns that hold at least one point inside the band limit (2 m_cut + 1): the columns any
    implementation of the slice step must move (workload geometry, no method arithmetic)."""
    kc = (2.0 / 3.0) * min(nx / (2.0 * cell[0]), ny / (2.0 * cell[1]))
    return 2 * int(np.floor(kc * cell[0] + 1e-9)) + 1


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        super().__init__(daemon=True)
        self.index, self.period, self.stop_flag = index, period_s, threading.Event()
        self.sm, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake": 0x80, "sync_boost": 0x10, "applications_clocks": 0x2}
        while not self.stop_flag.is_set():
            try:
                self.sm.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag.set()
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.sm)}


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# --------------------------------------------------------------------------------------------- oracle arm
def _oracle_frames(job):
    """Worker (one process = one host core): positions -> exit waves of its frames through the first `n_sl` slices.
    The oracle as it stands (oracle/tacaw_oracle.py), nothing tuned."""
    from oracle import tacaw_oracle as O
    pos, elem, coef, nl, ng, cell, nx, ny, n_slices, n_sl, kV, psi0 = job
    out = np.empty((pos.shape[0], ny, nx), dtype=np.complex128)
    sub_cell = np.array([cell[0], cell[1], cell[2] * n_sl / n_slices])       # same dz for the propagator
    for i in range(pos.shape[0]):
        V, _ = O.projected_potential(pos[i], elem, coef, nl, ng, cell, nx, ny, n_slices, slices=range(n_sl))
        out[i] = O.multislice(psi0, V[:n_sl], sub_cell, kV)
    return out


def oracle_sample(w, budget_s: float = 20.0, cores: int | None = None):
    """Times the float64 oracle on all host cores: every worker process takes one frame (two when that stays inside
    the budget) of the workload, builds its potentials and propagates one probe through the first n_sl slices (n_sl
    calibrated so that the sample costs about `budget_s` seconds), and the parent runs the oracle's time transform on
    the gathered exit waves.  Rate = nx*ny*n_sl*frames / wall time."""
    import multiprocessing as mp
    from oracle import tacaw_oracle as O
    cores = cores or os.cpu_count() or 1
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    elem = np.searchsorted(w.elements, w.Z)
    if w.beam == "plane":
        psi0 = O.plane_wave(w.nx, w.ny)
    elif w.beam == "tilt":
        psi0 = O.tilted_plane_wave(w.nx, w.ny, int(w.tilts[-1][0]), int(w.tilts[-1][1]))
    else:
        psi0 = O.probe_wave(w.cell, w.nx, w.ny, w.kV, w.semi_angle_mrad, w.probe_xy[0][0], w.probe_xy[0][1])
    n_frames = min(w.n_frames, 2 * cores)
    pos = w.positions(0, n_frames)
    # calibration: one frame, one slice, in this process
    t0 = time.perf_counter()
    _oracle_frames((pos[:1], elem, coef, nl, ng, w.cell, w.nx, w.ny, w.n_slices, 1, w.kV, psi0))
    t1 = max(time.perf_counter() - t0, 1e-3)
    per_worker = max(1, n_frames // cores)
    n_sl = int(max(1, min(w.n_slices, budget_s / (t1 * per_worker))))
    jobs = [(pos[i::cores], elem, coef, nl, ng, w.cell, w.nx, w.ny, w.n_slices, n_sl, w.kV, psi0) for i in range(cores)
            if pos[i::cores].shape[0] > 0]
    ctx = mp.get_context("spawn")                                # children never touch CUDA
    with ctx.Pool(len(jobs)) as pool:
        pool.map(_oracle_frames, [(pos[:1], elem, coef, nl, ng, w.cell, 32, 32, w.n_slices, 1, w.kV,
                                   O.plane_wave(32, 32))] * len(jobs))    # start-up (imports) outside the timed region
        t0 = time.perf_counter()
        parts = pool.map(_oracle_frames, jobs)
        ex = np.concatenate(parts)
        O.tacaw_intensity(ex, None)
        t = time.perf_counter() - t0
    units = float(w.nx) * w.ny * n_sl * n_frames
    return {"value": units / t / 1e9, "unit": UNIT, "cores": len(jobs), "kind": "oracle",
            "sample": f"{n_frames} of {w.n_frames} frames x 1 of {w.n_probes} probe(s) x first {n_sl} of {w.n_slices} "
                      f"slices, positions -> potentials -> exit waves -> |Psi(k,w)|^2; float64 NumPy oracle, "
                      f"{len(jobs)} worker processes (os.cpu_count() = {os.cpu_count()}), {t:.1f} s wall"}, t, units


def run_reference(args, w, rank):
    if rank != 0:
        return
    t_all, u_all, cb = 0.0, 0.0, None
    for _ in range(1 if args.warmup > 0 else 0):
        oracle_sample(w, budget_s=2.0)
    per = max(3.0, min(20.0, 120.0 / max(1, args.steps)))
    for _ in range(max(1, args.steps)):
        cb, t, u = oracle_sample(w, budget_s=per)
        t_all += t; u_all += u
    val = u_all / t_all / 1e9
    cb["value"] = val
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_all / max(1, args.steps), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, note="float64 NumPy oracle on the host cores; each step is a bounded sample"),
        "cpu_baseline": cb,
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def workload_config(w, **extra):
    d = {"workload": w.label, "grid": [w.nx, w.ny], "n_slices": w.n_slices, "frames": w.n_frames, "probes": w.n_probes,
         "atoms": int(w.n_atoms), "kV": w.kV}
    d.update(extra)
    return d


def build_workload(args):
    w = make_workload(args.workload, n_frames=args.frames, grid=args.grid, n_probes_side=args.probes_side)
    w.label = w.name
    if w.beam == "probe" and args.probe_chunk and args.probe_chunk < w.n_probes:
        w.probe_xy = w.probe_xy[:args.probe_chunk]                # one scan row (x fixed, 16 y positions)
        w.label = f"{w.name}: one {args.probe_chunk}-probe scan row x {w.n_frames} frames"
    if args.frames or args.grid or args.probes_side:
        w.label += " (size overridden)"
    return w


# --------------------------------------------------------------------------------------------- micro benches
def _event_time(torch, fn, flush, reps=5, warm=3):
    for _ in range(warm):
        fn()
    ts = []
    for _ in range(reps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return float(np.median(ts))


def tacaw_micro(shapes_a=None, shapes_b=None):
    """ps_tacaw (path A) and ps_tacaw_add (path B) alone on random complex64 stacks (every pixel non-zero; only
    in-band pixels are read): median of 5 runs after 3 warm-ups, L2 flushed between runs; one JSON line per shape.
    `shapes_a` = [(P, frames, grid, bins)], `shapes_b` = [(grid, chunk frames, bins)] override the default lists
    (--micro-a / --micro-b: one shape per ncu capture)."""
    import torch
    import paper_2602_10064_b200 as ps
    from paper_2602_10064_b200.binding import TacawStream
    peak, _, _ = measured_peaks()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    w0 = make_workload("c1_si_128", mini=True)
    nl, ng, coef = form_factor_coefficients(w0.elements, w0.ff_kind)

    def ctx_for(n):
        ctx = ps.Context(0)
        ctx.set_form_factors(w0.elements, nl, ng, coef)
        ctx.set_geometry(np.array([n * 0.1, n * 0.1, 8.0]), n, n, 2.0)
        return ctx

    if shapes_a is None and shapes_b is None:
        shapes_a = [(1, 512, 256, 50), (1, 512, 256, 512), (16, 1024, 512, 1024), (4, 1024, 512, 128),
                    (1, 2048, 512, 2048), (1, 4096, 256, 256), (8, 256, 512, 256), (16, 128, 512, 128),
                    (1, 256, 1024, 256), (1, 64, 128, 64)]
        shapes_b = [(1024, 64, 256), (512, 64, 256), (1024, 64, 64)]
    for shp in shapes_a or []:
        P, F, n, nb = shp[:4]
        tiled = len(shp) > 4 and shp[4] == 1
        ctx = ctx_for(n)
        eshape = ps.exit_shape(ctx, P, F, ps.PS_LAYOUT_TILED_APERTURE if tiled else ps.PS_LAYOUT_DENSE)
        ex = torch.view_as_complex(torch.randn(tuple(eshape) + (2,), device="cuda"))
        bins = None if nb == F else np.arange(nb, dtype=np.int32)
        I = torch.empty((P, nb, n, n), dtype=torch.float32, device="cuda")
        ms = _event_time(torch, lambda: ps.ps_tacaw(ctx, ex, 2.0, bins, d_I=I), flush)
        nk = ctx.n_k_aperture
        byts = (8.0 * F + 4.0 * nb) * nk * P                        # in-aperture reads + in-aperture writes
        zero = 4.0 * nb * (n * n - nk) * P                          # zero fill of the dense I cube: traffic, not algorithm
        print(json.dumps({"micro": "ps_tacaw", "layout": "tiled" if tiled else "dense", "P": P, "frames": F, "grid": n, "bins": nb, "ms": ms,
                          "algorithmic_GB": byts / 1e9, "GBps": byts / ms / 1e6, "frac_of_hbm_peak": byts / ms / 1e6 / peak,
                          "zero_fill_GB": zero / 1e9, "frac_with_zero_fill": (byts + zero) / ms / 1e6 / peak}))
        del ex, I, ctx
    # path B: one 64-frame chunk of a 4096-frame stream, 256 bins (config 4's shape) and a 1024^2 grid
    for n, Fc, nb in shapes_b or []:
        ctx = ctx_for(n)
        ex = torch.view_as_complex(torch.randn((1, Fc, n, n, 2), device="cuda"))
        ts = TacawStream(ctx, 1, 4096, 2.0, np.arange(nb, dtype=np.int32))
        ts.add(ex, 0)
        state = {"f": Fc}

        def add():
            ts.add(ex, state["f"]); state["f"] += Fc

        ms = _event_time(torch, add, flush, reps=5, warm=3)
        nk = ctx.n_k_aperture
        byts = 8.0 * Fc * nk + 2.0 * 8.0 * nb * nk                  # exit values once + accumulators read and written
        fma = 4.0 * Fc * nb * nk
        sm_clock = 1.965e9
        print(json.dumps({"micro": "ps_tacaw_add", "grid": n, "chunk_frames": Fc, "bins": nb, "ms": ms,
                          "algorithmic_GB": byts / 1e9, "frac_of_hbm_peak": byts / ms / 1e6 / peak,
                          "fma_per_s": fma / ms * 1e3, "frac_of_fp32_fma_peak": fma / ms * 1e3 / (N_SM * LANES_PER_SM * sm_clock)}))
        del ex, ts, ctx


# --------------------------------------------------------------------------------------------- cuFFT reference point
def cufft_reference(w, n_waves, n_slices=8):
    """The slice step written with library calls (north_star: "cuFFT timed only as a reference point"): torch.exp for
    the transmission function, torch.fft.fft2 / ifft2 (cuFFT) and elementwise products, on `n_waves` random waves of the
    workload's grid.  Not part of the library and never linked into it: a yardstick for the fused passes."""
    import torch
    nx, ny = w.nx, w.ny
    dev = torch.device("cuda")
    psi = torch.view_as_complex(torch.randn((n_waves, ny, nx, 2), device=dev))
    V = torch.randn((n_slices, ny, nx), device=dev)
    kx = torch.fft.fftfreq(nx, d=w.cell[0] / nx, device=dev)[None, :]
    ky = torch.fft.fftfreq(ny, d=w.cell[1] / ny, device=dev)[:, None]
    k2 = kx * kx + ky * ky
    kc = (2.0 / 3.0) * min(nx / (2 * w.cell[0]), ny / (2 * w.cell[1]))
    prop = (torch.polar(torch.ones_like(k2), -3.14159265 * 0.037 * 1.36 * k2) * (k2 <= kc * kc)).to(torch.complex64)

    def one_slice(s):
        nonlocal psi
        t = torch.polar(torch.ones_like(V[s]), 9.24e-4 * V[s])
        psi = torch.fft.ifft2(torch.fft.fft2(psi * t) * prop)

    for s in range(3):
        one_slice(s % n_slices)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for s in range(n_slices):
        one_slice(s)
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / n_slices
    out = {"reference": "cuFFT slice step (torch.fft.fft2/ifft2 + elementwise kernels; no band-limit pruning, no fusion)",
           "grid": [nx, ny], "waves": n_waves, "ms_per_slice": ms, "gpx_slice_s": nx * ny * n_waves / ms / 1e6}
    print(json.dumps(out))
    # the time transform with cuFFT: fft along the frame axis of a dense [P][F][ny][nx] stack, then |.|^2
    P, F = 4, min(w.n_frames, 1024)
    while P > 1 and P * F * ny * nx * 8 > (10 << 30):
        P //= 2
    ex = torch.view_as_complex(torch.randn((P, F, ny, nx, 2), device=dev))
    for _ in range(2):
        I = torch.fft.fft(ex - ex.mean(dim=1, keepdim=True), dim=1).abs().square()
    torch.cuda.synchronize()
    a.record()
    I = torch.fft.fft(ex - ex.mean(dim=1, keepdim=True), dim=1).abs().square()
    b.record()
    torch.cuda.synchronize()
    ms_t = a.elapsed_time(b)
    byts = (8.0 * F + 4.0 * F) * P * nx * ny
    peak, _, _ = measured_peaks()
    out_t = {"reference": "cuFFT time transform (mean removal, torch.fft.fft over the frame axis of the dense stack, |.|^2; all pixels)",
             "P": P, "frames": F, "grid": [nx, ny], "ms": ms_t, "frac_of_hbm_peak_on_its_own_bytes": byts / ms_t / 1e6 / peak}
    print(json.dumps(out_t))
    return out


# --------------------------------------------------------------------------------------------- configs 3 / 4 at full size
def slice_step_roofline(prof, px, f_col, P):
    """HBM roofline of the two slice-step passes from the library's per-launch events: `px` pixel-slices of one wave
    batch, algorithmic bytes per pixel 16 f_col + 4/P (row pass: wave in + out on the in-band columns, V once per frame)
    and 16 f_col (column pass), against the measured copy rate."""
    peak, _, src = measured_peaks()
    alg = {"k_row_transmit": 16.0 * f_col + 4.0 / P, "k_col_propagate": 16.0 * f_col}
    out = {"bound": "hbm", "unit": "GB/s", "peak": peak, "peak_source": src}
    ms_pair = 0.0
    for k, b in alg.items():
        if k not in prof or prof[k][1] == 0:
            return None
        ms = prof[k][0]
        ms_pair += ms
        out[k] = {"ms": ms, "algorithmic_bytes_per_px": b, "achieved": b * px / (ms * 1e-3) / 1e9,
                  "frac": b * px / (ms * 1e-3) / 1e9 / peak}
    tot = sum(alg.values())
    out["slice_step_pair"] = {"achieved": tot * px / (ms_pair * 1e-3) / 1e9, "frac": tot * px / (ms_pair * 1e-3) / 1e9 / peak,
                              "gpx_slice_s": px / (ms_pair * 1e-3) / 1e9}
    return out


def full_config(which, quiet=False, fused_v=False):
    """Config 4: 4096 frames x 1024^2 x 120 slices, V built and propagated 64 frames at a time, exit waves folded into the
    streaming per-bin DFT (path B, 256 bins) chunk by chunk (SURVEY.md 8(d) capacity plan).  Config 3: 1024 frames x
    256 probes x 512^2 x 80 slices: V of all frames resident (86 GB), probes 16 at a time (34 GB of exit waves),
    path A per probe chunk, spectrum image and probe-summed diffraction pattern accumulated on the fly."""
    import torch
    import paper_2602_10064_b200 as ps
    from paper_2602_10064_b200.binding import TacawStream
    t_host = time.perf_counter()
    w = make_workload("c4_interface_1024" if which == "c4" else "c3_si_probe_512")
    F, P, S, nx, ny = w.n_frames, w.n_probes, w.n_slices, w.nx, w.ny
    ctx = ps.Context(0)
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    ctx.set_form_factors(w.elements, nl, ng, coef)
    ctx.set_geometry(w.cell, nx, ny, w.slice_dz)
    step = 256
    pos_d = torch.cat([torch.from_numpy(w.positions(f0, min(F, f0 + step))).cuda() for f0 in range(0, F, step)])
    Z_d = torch.from_numpy(w.Z.copy()).cuda()
    t_host = time.perf_counter() - t_host
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.reset_peak_memory_stats()
    l0 = ctx.launches
    if which == "c4":
        chunk = 64
        bins = w.bins
        V = torch.empty((chunk, S, ny, nx), dtype=torch.float32, device="cuda")
        ex = torch.empty((1, chunk, ny, nx), dtype=torch.complex64, device="cuda")
        psi0 = ps.ps_make_incident(ctx, w.kV)
        ts0 = TacawStream(ctx, 1, F, w.dt_fs, bins)                      # warm-up of every kernel on one chunk
        ps.ps_build_slices(ctx, pos_d[:chunk], Z_d, d_V=V); ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=ex); ts0.add(ex, 0)
        del ts0
        torch.cuda.synchronize()
        a.record()
        ts = TacawStream(ctx, 1, F, w.dt_fs, bins)
        for f0 in range(0, F, chunk):
            if fused_v:
                ps.ps_multislice_fused(ctx, w.kV, psi0, pos_d[f0:f0 + chunk], Z_d, d_exit=ex)
            else:
                ps.ps_build_slices(ctx, pos_d[f0:f0 + chunk], Z_d, d_V=V)
                ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=ex)
            ts.add(ex, f0)
        I = ts.finish()
        simg = ps.ps_spectrum_image(ctx, I)
        b.record()
        torch.cuda.synchronize()
        check = float(simg.sum())
        # untimed: one more chunk with the library's per-launch events -> kernel split and slice-step roofline of config 4
        ctx.profile_read(reset=True)
        ctx.profile_enable(True)
        ts1 = TacawStream(ctx, 1, F, w.dt_fs, bins)
        ps.ps_build_slices(ctx, pos_d[:chunk], Z_d, d_V=V); ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=ex); ts1.add(ex, 0)
        prof = ctx.profile_read(reset=True)
        ctx.profile_enable(False)
        del ts1
        extra = {"kernel_ms_per_chunk": {k: v[0] for k, v in prof.items() if v[1] > 0},
                 "roofline": slice_step_roofline(prof, float(nx) * ny * S * chunk, band_columns(w.cell, nx, ny) / nx, 1)}
        plan = (f"{F // chunk} chunks of {chunk} frames: " + ("ps_multislice_fused (no V array)" if fused_v else "build V (30 GB) -> multislice") +
                f" -> ps_tacaw_add (path B, {len(bins)} bins)")
    else:
        pc = 16
        V = ps.ps_build_slices(ctx, pos_d[:8], Z_d)                      # warm-up
        del V
        torch.cuda.synchronize()
        ex = torch.empty(ps.exit_shape(ctx, pc, F, ps.PS_LAYOUT_TILED_APERTURE), dtype=torch.complex64, device="cuda")
        I = torch.empty((pc, F, ny, nx), dtype=torch.float32, device="cuda")
        simg = torch.empty((P, F), dtype=torch.float32, device="cuda")
        sdp = torch.zeros((ny, nx), dtype=torch.float32, device="cuda")
        sdp_c = torch.empty((ny, nx), dtype=torch.float32, device="cuda")
        a.record()
        V = torch.empty((F, S, ny, nx), dtype=torch.float32, device="cuda")
        ps.ps_build_slices(ctx, pos_d, Z_d, d_V=V)
        for p0 in range(0, P, pc):
            psi0 = ps.ps_make_incident(ctx, w.kV, w.semi_angle_mrad, w.probe_xy[p0:p0 + pc])
            ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=ex)
            ps.ps_tacaw(ctx, ex, w.dt_fs, d_I=I)
            ps.ps_spectrum_image(ctx, I, d_out=simg[p0:p0 + pc])
            ps.ps_sdp(ctx, I, 1, 32, d_out=sdp_c)
            ps.ps_accumulate_intensity(ctx, sdp, sdp_c, 1.0, 1.0)
        b.record()
        torch.cuda.synchronize()
        check = float(simg.sum())
        # untimed: Parseval on the last probe chunk (pin P11; tests/test_gpu_full_size.py::test_c3_bench_shape checks the same
        # identity against the oracle-verified exit waves): sum_{k,n} I = F sum_{k,t} |Psi - <Psi>_t|^2, left side from simg
        worst = 0.0
        for p in range(pc):
            tot = 0.0
            for y0 in range(0, ny, 64):
                blk = ex[p, y0:y0 + 64].to(torch.complex128)              # tiled layout [rows][tiles][F][8]
                blk = blk - blk.mean(dim=2, keepdim=True)
                tot += float((blk.real ** 2 + blk.imag ** 2).sum())
            worst = max(worst, abs(float(simg[P - pc + p].double().sum()) - F * tot) / (F * tot))
        extra = {"parseval_rel_err_last_probe_chunk": worst}
        plan = (f"V of all {F} frames resident (86 GB); {P // pc} chunks of {pc} probes: incident -> multislice (tiled exit "
                f"layout, {ex.numel() * 8 / 1e9:.0f} GB) -> ps_tacaw -> reductions")
    sec = a.elapsed_time(b) * 1e-3
    units = float(nx) * ny * S * F * P
    out = {"full_config": w.name, "grid": [nx, ny], "n_slices": S, "frames": F, "probes": P, "atoms": int(w.n_atoms),
           "tacaw_end_to_end_s": sec, "value": units / sec / 1e9, "unit": UNIT, "plan": plan,
           "gpu_launches": int(ctx.launches - l0), "host_setup_s": t_host, "checksum_spectrum_image": check,
           "hbm_peak_allocated_GB": torch.cuda.max_memory_allocated() / 1e9}
    out.update(extra)
    del V, ex, I, ctx, pos_d
    torch.cuda.empty_cache()
    if not quiet:
        print(json.dumps(out))
    return out


# --------------------------------------------------------------------------------------------- our arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3_si_probe_512")
    ap.add_argument("--probe-chunk", type=int, default=16,
                    help="probe workloads: probes per step (default: one 16-probe scan row, the chunk the full run loops over)")
    ap.add_argument("--frames", type=int, default=None, help="override the number of frames (parity/debug only)")
    ap.add_argument("--grid", type=int, default=None, help="override the grid size (config 5 sweeps 256..2048)")
    ap.add_argument("--probes-side", type=int, default=None, help="override probes per scan side / number of tilts")
    ap.add_argument("--wave-chunk", type=int, default=0)
    ap.add_argument("--exit-layout", default="auto", choices=["auto", "dense", "tiled"],
                    help="exit-wave layout between ps_multislice and ps_tacaw: tiled = PS_LAYOUT_TILED_APERTURE (auto: tiled "
                         "unless the batch takes the chip-resident small-grid path, which writes the dense layout)")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="ps_set_tuning knob (resident=-1|0|1); repeatable")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = an independent trajectory per rank (reductions averaged); strong = ONE problem "
                         "sharded by sharding.plan() (probe shards, or frame shards + reduce-scatter of the accumulators)")
    ap.add_argument("--vk-mode", type=int, default=0, choices=[0, 1, 2],
                    help="ps_set_vk_mode: 0 library default, 1 FP32 SIMT structure-factor sums, 2 tcgen05 3xTF32")
    ap.add_argument("--fused-v", action="store_true",
                    help="positions -> exit waves through ps_multislice_fused (the row pass builds V row by row from the "
                         "y-transformed slice pairs; no V array; dense exit layout) instead of ps_build_slices + ps_multislice")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--with-full-configs", action="store_true",
                    help="also run configs 3 and 4 at their FULL size after the timed steps and carry their end-to-end "
                         "seconds in the same JSON line (adds about two minutes); on by default for the default workload "
                         "on one GPU")
    ap.add_argument("--no-full-configs", action="store_true", help="skip the full-size runs of configs 3 and 4")
    ap.add_argument("--full-config", choices=["c3", "c4"], default=None,
                    help="run config 3 or 4 at its FULL size (all frames, all probes) in chunks that fit 180 GB, one step, "
                         "and print one JSON line")
    ap.add_argument("--cufft-reference", action="store_true",
                    help="time the slice step written with torch.fft (cuFFT) + elementwise kernels on 1024 waves (or as many "
                         "as fit 2 GB) of the workload's grid and exit: a reference point, not part of the library")
    ap.add_argument("--tacaw-micro", action="store_true",
                    help="time ps_tacaw / ps_tacaw_add alone on synthetic stacks of several shapes and exit")
    ap.add_argument("--micro-a", action="append", default=None, metavar="P,FRAMES,GRID,BINS[,TILED]",
                    help="--tacaw-micro: this path-A shape instead of the default list (repeatable)")
    ap.add_argument("--micro-b", action="append", default=None, metavar="GRID,CHUNK_FRAMES,BINS",
                    help="--tacaw-micro: this path-B shape instead of the default list (repeatable)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    w = build_workload(args)

    if args.impl == "reference":
        run_reference(args, w, rank)
        return
    if args.cufft_reference:
        cufft_reference(w, max(1, min(1024, (2 << 30) // (w.nx * w.ny * 8))))
        return
    if args.tacaw_micro:
        parse = lambda xs: None if xs is None else [tuple(int(v) for v in x.split(",")) for x in xs]
        if args.micro_a is None and args.micro_b is None:
            tacaw_micro()
        else:
            tacaw_micro(parse(args.micro_a) or [], parse(args.micro_b) or [])
        return
    if args.full_config:
        full_config(args.full_config, fused_v=args.fused_v)
        return

    import torch
    import torch.distributed as dist
    import paper_2602_10064_b200 as ps
    from paper_2602_10064_b200 import sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    if args.scaling == "strong":                                  # world = 1 too: the same loop on one rank
        sharding.run_strong_bench(args, w, rank, world, dev, ps, METRIC, UNIT)
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- inputs: an independent seeded trajectory per rank (rank 0 = the workload's own seed)
    if rank > 0:
        w.seed += 7919 * rank
        w.mode_phi = np.random.default_rng(w.seed).uniform(0, 2 * np.pi, w.mode_phi.shape[0])
    pos_h = torch.from_numpy(w.positions()).pin_memory()
    Z_h = torch.from_numpy(w.Z.copy())
    F, P, S, nx, ny = w.n_frames, w.n_probes, w.n_slices, w.nx, w.ny
    bins = w.bins if w.bins is not None else None
    nb = F if bins is None else len(bins)

    ctx = ps.Context(local_rank)
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    ctx.set_form_factors(w.elements, nl, ng, coef)
    ctx.set_geometry(w.cell, nx, ny, w.slice_dz)
    small_resident = nx == ny and nx <= 128 and P * F <= 2 * N_SM          # ps_multislice's chip-resident path (dense only)
    tiled = (args.exit_layout == "tiled" or (args.exit_layout == "auto" and not small_resident)) and not args.fused_v
    exit_shape = ps.exit_shape(ctx, P, F, ps.PS_LAYOUT_TILED_APERTURE if tiled else ps.PS_LAYOUT_DENSE)
    exit_bytes = 8.0 * float(np.prod(exit_shape))
    need = 4.0 * F * S * ny * nx + exit_bytes + 4.0 * P * nb * ny * nx
    free_b, _ = torch.cuda.mem_get_info()
    if need > 0.97 * free_b:
        raise SystemExit(f"workload needs {need / 1e9:.0f} GB of HBM (V + exit waves + I), {free_b / 1e9:.0f} GB free")
    if args.wave_chunk:
        ctx.set_wave_chunk(args.wave_chunk)
    if args.vk_mode:
        ctx.set_vk_mode(args.vk_mode)
    for kv in args.tune:
        k, v = kv.split("=")
        ctx.set_tuning(k, int(v))

    pos_d = pos_h.to(dev)
    Z_d = Z_h.to(dev)
    V = torch.empty((F, S, ny, nx), dtype=torch.float32, device=dev)
    psi0 = torch.empty((P, ny, nx), dtype=torch.complex64, device=dev)
    exitw = torch.empty(exit_shape, dtype=torch.complex64, device=dev)
    I = torch.empty((P, nb, ny, nx), dtype=torch.float32, device=dev)
    sdp = torch.empty((ny, nx), dtype=torch.float32, device=dev)
    simg = torch.empty((P, nb), dtype=torch.float32, device=dev)
    n_path, n_q = 100, 64
    kc = (2.0 / 3.0) * min(nx / (2 * w.cell[0]), ny / (2 * w.cell[1]))
    kx_path = np.linspace(0.0, 0.9 * kc, n_path); ky_path = np.zeros(n_path)
    disp = torch.empty((nb, n_path), dtype=torch.float32, device=dev)
    qb = torch.empty((nb, n_q), dtype=torch.float32, device=dev)
    red_d = (sdp, simg, disp, qb)
    red_h = [torch.empty(t.shape, dtype=torch.float32).pin_memory() for t in red_d]
    # what a caller keeps: the whole I(k,w) cube when it is small (plane-wave / tilt runs look at it directly), only the
    # reductions for probe scans (config 3's cube is 17 GB per 16-probe row, 275 GB per scan: it is never kept)
    keep_cube = I.numel() * 4 <= (1 << 30)
    I_h = torch.empty(I.shape, dtype=torch.float32).pin_memory() if keep_cube else None
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)      # > 126 MB L2

    if w.beam == "probe":
        inc = dict(semi_angle_mrad=w.semi_angle_mrad, xy_or_tilt=w.probe_xy)
    elif w.beam == "tilt":
        inc = dict(semi_angle_mrad=0.0, xy_or_tilt=w.tilts.astype(np.float64), is_tilt=True)
    else:
        inc = dict(n=1)

    def step(pos_dev):
        ps.ps_make_incident(ctx, w.kV, d_psi0=psi0, **inc)
        if args.fused_v:
            ps.ps_multislice_fused(ctx, w.kV, psi0, pos_dev, Z_d, d_exit=exitw)
        else:
            ps.ps_build_slices(ctx, pos_dev, Z_d, d_V=V)
            ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=exitw)
        ps.ps_tacaw(ctx, exitw, w.dt_fs, bins, d_I=I)
        ps.ps_sdp(ctx, I, 1, min(8, nb - 1), d_out=sdp)
        ps.ps_spectrum_image(ctx, I, 0.0, 0.0, d_out=simg)
        ps.ps_dispersion(ctx, I, kx_path, ky_path, d_out=disp)
        ps.ps_qbin(ctx, I, kc / n_q, n_q, d_out=qb)
        if world > 1:                                            # trajectory averaging: the reductions are
            for t in red_d:                                      # linear in I, so their sum over ranks is the reduction of
                sharding.all_reduce_sum_(t)                      # the summed I(k,w)

    def step_e2e():
        pos_dev = pos_h.to(dev, non_blocking=True)
        step(pos_dev)
        if keep_cube:
            I_h.copy_(I, non_blocking=True)
        for h, d in zip(red_h, red_d):
            h.copy_(d, non_blocking=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, K):
        """K steps, each bracketed by its own event pair, L2 flushed (outside the pairs) between steps."""
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        barrier()
        for a, b in evs:
            flush.zero_()
            a.record()
            fn()
            b.record()
        barrier()
        ms = sum(a.elapsed_time(b) for a, b in evs)
        return sharding.max_over_ranks(ms, device=dev) if world > 1 else ms

    W = max(3, args.warmup)
    for _ in range(W):
        step(pos_d)
    barrier()

    K = max(1, args.steps)
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    l0 = ctx.launches
    ms_total = timed(lambda: step(pos_d), K)
    launches = ctx.launches - l0
    clocks = sampler.result()

    units_rank = float(nx) * ny * S * F * P
    value = units_rank * world * K / (ms_total * 1e-3) / 1e9

    # ---- end to end through the public API with host buffers
    step_e2e(); barrier()
    ms_e2e = timed(step_e2e, K)
    e2e_value = units_rank * world * K / (ms_e2e * 1e-3) / 1e9
    h2d = pos_h.numel() * 4
    d2h = (I_h.numel() * 4 if keep_cube else 0) + sum(h.numel() * 4 for h in red_h)

    # ---- per-kernel device time (library-side CUDA events on its stream), a second pass of the same K steps
    ctx.profile_read(reset=True)
    ctx.profile_enable(True)
    ms_prof_total = timed(lambda: step(pos_d), K)
    prof = ctx.profile_read(reset=True)
    ctx.profile_enable(False)

    peak, bf16_peak, peak_src = measured_peaks()
    stats = kernel_stats()
    kern = {k: v for k, v in prof.items() if v[1] > 0}
    # algorithmic bytes per pixel of one wave and slice: the wave is read and written once per pass on the
    # k-columns that hold in-band points (f_col of them); V is read once per FRAME (its rows are shared by the P probes
    # of the frame inside a launch), i.e. 4/P bytes per pixel of one wave
    f_col = band_columns(w.cell, nx, ny) / nx
    sm_clock = (clocks.get("sm_mhz") or 1965.0) * 1e6
    issue_peak = N_SM * LANES_PER_SM * sm_clock

    def issue_of(key, px_per_s):
        """FP32-issue co-limit from the ncu-derived instruction count of this kernel at this grid size."""
        st = stats.get(key)
        if not st:
            return None, None
        return st, {"thread_inst_per_px": st["thread_inst_per_px"], "peak_thread_inst_per_s": issue_peak,
                    "frac": st["thread_inst_per_px"] * px_per_s / issue_peak,
                    "note": "thread instructions per pixel (ncu, profiles/" + stats.get("_file", "?") + ") x pixels/s / (148 SMs x 128 "
                            "lanes x SM clock sampled in this run): the FP32-issue co-limit of the FFT passes"}

    if "k_slice_resident" in kern:
        # chip-resident slice loop (small square grids, small batches): the wave never leaves shared memory, so HBM sees
        # V once per frame and slice plus the incident wave in and the exit wave out: the kernel is bound by
        # instruction issue, and that is the roofline reported
        ms_res, n_res = kern["k_slice_resident"]
        px_s = units_rank * K / (ms_res * 1e-3)
        alg_px = 4.0 / P + 16.0 / S
        st, issue = issue_of(f"k_slice_resident<{nx}>", px_s)
        roofline = {"bound": "alu", "kernel": f"k_slice_resident<{nx}>", "unit": "thread-instructions/s",
                    "achieved": (st["thread_inst_per_px"] * px_s) if st else None, "peak": issue_peak,
                    "frac": issue["frac"] if issue else None,
                    "traffic": (st["dram_bytes_per_px"].get("any") * units_rank * K / n_res) if st else None,
                    "avg_launch_ms": ms_res / n_res, "gpx_slice_s": px_s / 1e9,
                    "hbm": {"algorithmic_bytes_per_px_slice": alg_px, "achieved_GBps": alg_px * px_s / 1e9,
                            "frac_of_hbm_peak": alg_px * px_s / 1e9 / peak},
                    "peak_source": "148 SMs x 128 lanes x sampled SM clock (DESIGN.md §6)",
                    "kernel_ms_per_step": {k: v[0] / K for k, v in kern.items()},
                    "kernel_times_from": "a second pass of the same K steps with per-launch CUDA events recorded by the "
                                         "library on its stream (ps_profile_*), not the pass `value` was timed on",
                    "profiled_ms_per_step": ms_prof_total / K}
    else:
        alg = {"k_row_transmit": 16.0 * f_col + 4.0 / P, "k_col_propagate": 16.0 * f_col}
        dom = max(alg, key=lambda k: kern.get(k, (0.0, 0))[0])
        other = "k_col_propagate" if dom == "k_row_transmit" else "k_row_transmit"
        per = {}
        for kname in (dom, other):
            k_ms, k_n = kern[kname]
            px_launch = units_rank * K / k_n
            n_grid = nx if kname == "k_row_transmit" else ny
            st, issue = issue_of(f"{kname}<{n_grid}>", px_launch / (k_ms / k_n * 1e-3))
            tr = None
            if st:
                tr = st["dram_bytes_per_px"].get(str(P), st["dram_bytes_per_px"].get("any"))
                tr = tr * px_launch if tr is not None else None
            ach = alg[kname] * px_launch / (k_ms / k_n * 1e-3) / 1e9
            per[kname] = {"kernel": (st or {}).get("sass_kernel", f"{kname}<{n_grid}>"), "achieved": ach, "frac": ach / peak,
                          "traffic": tr,
                          "bytes_per_launch": alg[kname] * px_launch, "avg_launch_ms": k_ms / k_n,
                          "algorithmic_bytes_per_px": alg[kname], "fp32_issue": issue}
        ms_pair = kern["k_row_transmit"][0] + kern["k_col_propagate"][0]
        pair_gbs = (alg["k_row_transmit"] + alg["k_col_propagate"]) * units_rank * K / (ms_pair * 1e-3) / 1e9
        roofline = {"bound": "hbm", "unit": "GB/s", "peak": peak, "peak_source": peak_src, "band_column_fraction": f_col}
        roofline.update(per[dom])
        roofline.update({
            "algorithmic_bytes_note": "wave read + written once per pass on the k-columns holding in-band points; V read "
                                      "once per FRAME and slice (its rows are shared by the probes of a launch): 4/P B per "
                                      "pixel of one wave (DESIGN.md §6)",
            "other_pass": per[other],
            "slice_step_pair": {"achieved": pair_gbs, "frac": pair_gbs / peak,
                                "gpx_slice_s": units_rank * K / (ms_pair * 1e-3) / 1e9,
                                "algorithmic_bytes_per_px_slice": alg["k_row_transmit"] + alg["k_col_propagate"]},
            "kernel_ms_per_step": {k: v[0] / K for k, v in kern.items()},
            "kernel_times_from": "a second pass of the same K steps with per-launch CUDA events recorded by the library "
                                 "on its stream (ps_profile_*), not the pass `value` was timed on",
            "profiled_ms_per_step": ms_prof_total / K})
    if "k_tacaw_fft" in kern:
        # the method's own bytes are the in-aperture exit values read once (8 B k F P) and the in-aperture
        # intensities written once (4 B k n_w P).  The dense I[P][n_w][ny][nx] cube also makes the stage write zeros to the
        # out-of-band pixels: that is traffic, not algorithm, and is reported as such.
        tb_in = (8.0 * F + 4.0 * nb) * ctx.n_k_aperture * P
        tb_zero = 4.0 * nb * (nx * ny - ctx.n_k_aperture) * P
        tms = kern["k_tacaw_fft"][0] / K
        tst = stats.get(f"k_tacaw<{F}>")
        roofline["tacaw"] = {"achieved": tb_in / (tms * 1e-3) / 1e9, "frac": tb_in / (tms * 1e-3) / 1e9 / peak,
                             "bytes_per_step": tb_in, "ms_per_step": tms,
                             "zero_fill_bytes_per_step": tb_zero,
                             "frac_with_zero_fill": (tb_in + tb_zero) / (tms * 1e-3) / 1e9 / peak,
                             "traffic": (tst["dram_bytes_per_inband_algorithmic_byte"] * tb_in + tb_zero) if tst else None,
                             "note": "frac counts the method's bytes only (in-aperture reads + in-aperture writes); the dense "
                                     "I cube adds zero_fill_bytes_per_step of writes the method does not need"}
    if "k_vk" in kern:
        # V(k) structure-factor sums over the in-aperture quarter plane: 4 real sums = 8 flops per (point, atom) in the
        # method; the tensor path issues each product three times (3xTF32 split) to stay at fp32 accuracy
        flop8 = 8.0 * (ctx.n_k_aperture / 4.0) * float(w.n_atoms) * F
        tms = kern["k_vk"][0] / K
        tf32_peak = 0.5 * bf16_peak
        fp32_alu_peak = 2.0 * N_SM * LANES_PER_SM * sm_clock / 1e12
        roofline["vk"] = {"bound": "tensor", "unit": "TFLOP/s", "achieved": flop8 / (tms * 1e-3) / 1e12,
                          "peak": tf32_peak, "frac": flop8 / (tms * 1e-3) / 1e12 / tf32_peak,
                          "issued_3xtf32": {"achieved": 3.0 * flop8 / (tms * 1e-3) / 1e12,
                                            "frac": 3.0 * flop8 / (tms * 1e-3) / 1e12 / tf32_peak},
                          "vs_fp32_alu_peak": flop8 / (tms * 1e-3) / 1e12 / fp32_alu_peak,
                          "note": "frac = the method's 8 flops per (k point, atom) against measured bf16 x 0.5 (guide's nominal "
                                  "tf32:bf16 ratio); issued_3xtf32 counts the three TF32 products per fp32-accurate product; "
                                  "vs_fp32_alu_peak = the same 8 flops against 2 x 148 x 128 lanes x sampled clock; FP32 SIMT "
                                  "path when ps_set_vk_mode(1) or few atoms per slice"}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline, _, _ = oracle_sample(w)

    cube_gb = I.numel() * 4 / 1e9
    full = None
    is_default = (args.workload == "c3_si_probe_512" and not (args.frames or args.grid or args.probes_side) and
                  args.probe_chunk == 16 and not args.fused_v and not args.tune and not args.wave_chunk)
    if rank == 0 and world == 1 and (args.with_full_configs or (is_default and not args.no_full_configs)):
        del V, exitw, I, psi0
        torch.cuda.empty_cache()
        ctx = None                                               # this process keeps only its CUDA context
        torch.cuda.empty_cache()
        full = {}
        import subprocess
        for k in ("c3", "c4"):                                   # a child process each: a failure there cannot take the main line along
            try:
                res = subprocess.run([sys.executable, os.path.abspath(__file__), "--full-config", k], capture_output=True,
                                     text=True, timeout=1500)
                last = [ln for ln in res.stdout.strip().splitlines() if ln.startswith("{")]
                full[k] = json.loads(last[-1]) if (res.returncode == 0 and last) else {
                    "error": f"exit code {res.returncode}: {res.stderr.strip()[-300:]}"}
            except Exception as exc:                             # noqa: BLE001
                full[k] = {"error": f"{type(exc).__name__}: {exc}"[:300]}

        # the other shapes the bar is held on, small samples through this same script: config 5's largest grid (2 tilts x 32
        # frames of 2048^2) and the time transform alone at config 2's (50 of 512 bins) and config 5's (2048 frames) shapes
        me = [sys.executable, os.path.abspath(__file__)]
        for k, cmd in (("c5_2048_sample", me + ["--workload", "c5_al_sweep", "--grid", "2048", "--frames", "32", "--probes-side", "2",
                                                 "--steps", "2", "--no-cpu-baseline", "--no-full-configs"]),
                       ("tacaw_micro", me + ["--tacaw-micro", "--micro-a", "1,512,256,50", "--micro-a", "8,2048,512,2048,1",
                                             "--micro-a", "16,1024,512,1024,1"])):
            try:
                res = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
                rows = [json.loads(ln) for ln in res.stdout.strip().splitlines() if ln.startswith("{")]
                if res.returncode != 0 or not rows:
                    full[k] = {"error": f"exit code {res.returncode}: {res.stderr.strip()[-300:]}"}
                elif k == "tacaw_micro":
                    full[k] = rows
                else:
                    r = rows[-1]
                    full[k] = {"config": r["config"], "value": r["value"], "unit": r["unit"], "ms_per_step": r["ms_per_step"],
                               "roofline": {kk: r["roofline"].get(kk) for kk in ("kernel", "achieved", "frac", "peak", "avg_launch_ms",
                                                                               "other_pass", "slice_step_pair", "tacaw")}}
            except Exception as exc:                             # noqa: BLE001
                full[k] = {"error": f"{type(exc).__name__}: {exc}"[:300]}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex64 (f32)", "data": "synthetic",
            "config": workload_config(w, omega_bins=nb,
                                      l2="256 MiB buffer written between timed steps (L2 flush); per-step CUDA events",
                                      hbm_resident_GB=need / 1e9,
                                      exit_layout="tiled [P][ny][tile][F][8] (PS_LAYOUT_TILED_APERTURE)" if tiled else "dense [P][F][ny][nx]",
                                      potential="ps_multislice_fused (no V array)" if args.fused_v else "ps_build_slices -> V",
                                      parallelism=f"independent trajectory per GPU x{world}, one all-reduce of the reductions"),
            "tacaw_end_to_end_s": ms_total / K * 1e-3,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / K, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h,
                    "copied_back": ("I(k,w) cube + " if keep_cube else "") +
                                   "spectral diffraction pattern, spectrum image, dispersion, q-bins" +
                                   ("" if keep_cube else f" (the {cube_gb:.0f} GB I(k,w) cube of a probe chunk "
                                                         "is reduced on the device and never kept: 275 GB per 256-probe scan)")},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu_baseline}
        if full:
            line["full_configs"] = full
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
