#!/usr/bin/env python
"""bench.py — one JSON line for the TACAW hot path on B200 (contract: task prompt / DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path over one synthetic trajectory of the workload
(BASELINE.json configs[1] by default: hBN-like monolayer, 256x256, 10 slices, 512 frames):
    ps_build_slices -> ps_make_incident -> ps_multislice -> ps_tacaw -> ps_sdp / ps_spectrum_image /
    ps_dispersion / ps_qbin.
`value` = nx*ny*n_slices*frames*probes / step time, in Gpx*slice/s, inputs resident in HBM;
`e2e` = the same with host buffers (pinned positions in, I(k,w) cube + reductions out) inside the timed
region.  `roofline` is for the dominant kernel family of the step (per-launch CUDA events recorded by the
library's ps_profile_* on its own stream, in a second pass of the same K steps); `cpu_baseline` is the
float64 oracle timed on this box's host cores on a bounded sample of the same workload.
With N > 1 (torchrun) every rank processes an independent trajectory (averaging over
independent trajectories) and the I(k,w) cubes are summed with one NCCL all-reduce: weak scaling.
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
# algorithmic bytes per pixel*slice of the slice step (pruned figure):
#   row pass 4 (V) + 16 * f_col, column pass 16 * f_col, f_col = 2/3 of the columns inside the band limit
ROW_BYTES = 4.0 + 16.0 * (2.0 / 3.0)
COL_BYTES = 16.0 * (2.0 / 3.0)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


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
def oracle_sample(w, budget_s: float = 20.0):
    """Times the float64 oracle (as it stands) on the first n frames of the workload; n is chosen from
    a one-frame calibration so that the sample costs about `budget_s` seconds of CPU work."""
    from oracle import tacaw_oracle as O
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    elem = np.searchsorted(w.elements, w.Z)
    if w.beam == "plane":
        psi0 = [O.plane_wave(w.nx, w.ny)]
    elif w.beam == "tilt":
        psi0 = [O.tilted_plane_wave(w.nx, w.ny, int(m), int(n)) for m, n in w.tilts]
    else:
        psi0 = [O.probe_wave(w.cell, w.nx, w.ny, w.kV, w.semi_angle_mrad, x, y) for x, y in w.probe_xy]
    psi0 = psi0[:1]                                             # one probe / tilt is enough for a rate
    pos = w.positions(0, min(w.n_frames, 64))

    def run(n):
        t0 = time.perf_counter()
        O.run_path(pos[:n], elem, coef, nl, ng, w.cell, w.nx, w.ny, w.n_slices, w.kV, psi0, None, frames=range(n))
        return time.perf_counter() - t0

    t1 = run(1)
    n = int(max(2, min(pos.shape[0], budget_s / max(t1, 1e-3))))
    t = run(n)
    units = float(w.nx) * w.ny * w.n_slices * n * len(psi0)
    return {"value": units / t / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{n} of {w.n_frames} frames x {len(psi0)} probe(s), positions -> |Psi(k,w)|^2 "
                      f"(float64 NumPy oracle, {t:.1f} s)"}, t, units


def run_reference(args, w, rank):
    if rank != 0:
        return
    t_all, u_all = 0.0, 0.0
    cb = None
    for _ in range(args.warmup if args.warmup < 2 else 1):
        oracle_sample(w, budget_s=2.0)
    for _ in range(max(1, args.steps)):
        cb, t, u = oracle_sample(w, budget_s=max(2.0, 60.0 / max(1, args.steps)))
        t_all += t; u_all += u
    val = u_all / t_all / 1e9
    cb["value"] = val
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_all / max(1, args.steps), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "note": "float64 NumPy oracle on host cores; each step is a bounded sample"},
        "cpu_baseline": cb,
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# --------------------------------------------------------------------------------------------- ps_tacaw alone
def tacaw_micro():
    """ps_tacaw on random complex64 stacks [P][F][n][n] (every pixel non-zero; only in-band pixels are read):
    median of 5 runs after 3 warm-ups, L2 flushed between runs; one JSON line per shape."""
    import torch
    import paper_2602_10064_b200 as ps
    peak, _ = measured_peaks()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    w0 = make_workload("c1_si_128", mini=True)
    nl, ng, coef = form_factor_coefficients(w0.elements, w0.ff_kind)
    for P, F, n, nb in [(1, 512, 256, 50), (1, 512, 256, 512), (4, 1024, 512, 1024), (4, 1024, 512, 128), (1, 2048, 512, 2048),
                        (1, 4096, 256, 256), (8, 256, 512, 256), (16, 128, 512, 128), (1, 256, 1024, 256)]:
        ctx = ps.Context(0)
        ctx.set_form_factors(w0.elements, nl, ng, coef)
        ctx.set_geometry(np.array([n * 0.1, n * 0.1, 8.0]), n, n, 2.0)
        ex = torch.view_as_complex(torch.randn((P, F, n, n, 2), device="cuda"))
        bins = None if nb == F else np.arange(nb, dtype=np.int32)
        I = torch.empty((P, nb, n, n), dtype=torch.float32, device="cuda")
        for _ in range(3):
            ps.ps_tacaw(ctx, ex, 2.0, bins, d_I=I)
        ts = []
        for _ in range(5):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); ps.ps_tacaw(ctx, ex, 2.0, bins, d_I=I); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        ms = float(np.median(ts))
        nk = ctx.n_k_aperture
        byts = (8.0 * F + 4.0 * nb) * nk * P + 4.0 * nb * (n * n - nk) * P
        print(json.dumps({"micro": "ps_tacaw", "P": P, "frames": F, "grid": n, "bins": nb, "ms": ms,
                          "algorithmic_GB": byts / 1e9, "GBps": byts / ms / 1e6, "frac_of_hbm_peak": byts / ms / 1e6 / peak}))
        del ex, I, ctx


# --------------------------------------------------------------------------------------------- configs 3 / 4 at full size
def full_config(which):
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
            ps.ps_build_slices(ctx, pos_d[f0:f0 + chunk], Z_d, d_V=V)
            ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=ex)
            ts.add(ex, f0)
        I = ts.finish()
        simg = ps.ps_spectrum_image(ctx, I)
        b.record()
        torch.cuda.synchronize()
        check = float(simg.sum())
        plan = f"{F // chunk} chunks of {chunk} frames: build V (30 GB) -> multislice -> ps_tacaw_add (path B, {len(bins)} bins)"
    else:
        pc = 16
        V = ps.ps_build_slices(ctx, pos_d[:8], Z_d)                      # warm-up
        del V
        torch.cuda.synchronize()
        ex = torch.empty((pc, F, ny, nx), dtype=torch.complex64, device="cuda")
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
        plan = f"V of all {F} frames resident (86 GB); {P // pc} chunks of {pc} probes: incident -> multislice (34 GB) -> ps_tacaw -> reductions"
    sec = a.elapsed_time(b) * 1e-3
    units = float(nx) * ny * S * F * P
    print(json.dumps({"full_config": w.name, "grid": [nx, ny], "n_slices": S, "frames": F, "probes": P, "atoms": int(w.n_atoms),
                      "tacaw_end_to_end_s": sec, "value": units / sec / 1e9, "unit": UNIT, "plan": plan,
                      "gpu_launches": int(ctx.launches - l0), "host_setup_s": t_host, "checksum_spectrum_image": check,
                      "hbm_peak_allocated_GB": torch.cuda.max_memory_allocated() / 1e9}))


# --------------------------------------------------------------------------------------------- our arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2_hbn_256")
    ap.add_argument("--frames", type=int, default=None, help="override the number of frames (parity/debug only)")
    ap.add_argument("--grid", type=int, default=None, help="override the grid size (config 5 sweeps 256..2048)")
    ap.add_argument("--probes-side", type=int, default=None, help="override probes per scan side / number of tilts")
    ap.add_argument("--wave-chunk", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--full-config", choices=["c3", "c4"], default=None,
                    help="run config 3 or 4 at its FULL size (all frames, all probes) in chunks that fit 180 GB, one step, "
                         "and print one JSON line (minutes of host-side trajectory generation before the timed region)")
    ap.add_argument("--tacaw-micro", action="store_true",
                    help="time ps_tacaw alone on synthetic stacks of several shapes (profiles/r1_tacaw_kernels.md) and exit")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    w = make_workload(args.workload, n_frames=args.frames, grid=args.grid, n_probes_side=args.probes_side)

    if args.impl == "reference":
        run_reference(args, w, rank)
        return
    if args.tacaw_micro:
        tacaw_micro()
        return
    if args.full_config:
        full_config(args.full_config)
        return

    import torch
    import torch.distributed as dist
    import paper_2602_10064_b200 as ps

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

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
    if args.wave_chunk:
        ctx.set_wave_chunk(args.wave_chunk)

    pos_d = pos_h.to(dev)
    Z_d = Z_h.to(dev)
    V = torch.empty((F, S, ny, nx), dtype=torch.float32, device=dev)
    psi0 = torch.empty((P, ny, nx), dtype=torch.complex64, device=dev)
    exitw = torch.empty((P, F, ny, nx), dtype=torch.complex64, device=dev)
    I = torch.empty((P, nb, ny, nx), dtype=torch.float32, device=dev)
    sdp = torch.empty((ny, nx), dtype=torch.float32, device=dev)
    simg = torch.empty((P, nb), dtype=torch.float32, device=dev)
    n_path, n_q = 100, 64
    kc = (2.0 / 3.0) * min(nx / (2 * w.cell[0]), ny / (2 * w.cell[1]))
    kx_path = np.linspace(0.0, 0.9 * kc, n_path); ky_path = np.zeros(n_path)
    disp = torch.empty((nb, n_path), dtype=torch.float32, device=dev)
    qb = torch.empty((nb, n_q), dtype=torch.float32, device=dev)
    I_h = torch.empty(I.shape, dtype=torch.float32).pin_memory()
    red_h = [torch.empty(t.shape, dtype=torch.float32).pin_memory() for t in (sdp, simg, disp, qb)]
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)      # > 126 MB L2

    if w.beam == "probe":
        inc = dict(semi_angle_mrad=w.semi_angle_mrad, xy_or_tilt=w.probe_xy)
    elif w.beam == "tilt":
        inc = dict(semi_angle_mrad=0.0, xy_or_tilt=w.tilts.astype(np.float64), is_tilt=True)
    else:
        inc = dict(n=1)

    def step(pos_dev):
        ps.ps_build_slices(ctx, pos_dev, Z_d, d_V=V)
        ps.ps_make_incident(ctx, w.kV, d_psi0=psi0, **inc)
        ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=exitw)
        ps.ps_tacaw(ctx, exitw, w.dt_fs, bins, d_I=I)
        if world > 1:
            dist.all_reduce(I)                                   # trajectory averaging (sum)
        ps.ps_sdp(ctx, I, 1, min(8, nb - 1), d_out=sdp)
        ps.ps_spectrum_image(ctx, I, 0.0, 0.0, d_out=simg)
        ps.ps_dispersion(ctx, I, kx_path, ky_path, d_out=disp)
        ps.ps_qbin(ctx, I, kc / n_q, n_q, d_out=qb)

    def step_e2e():
        pos_dev = pos_h.to(dev, non_blocking=True)
        step(pos_dev)
        I_h.copy_(I, non_blocking=True)
        for h, d in zip(red_h, (sdp, simg, disp, qb)):
            h.copy_(d, non_blocking=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, K, profile=False):
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
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    for _ in range(max(3, args.warmup)):
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
    d2h = I_h.numel() * 4 + sum(h.numel() * 4 for h in red_h)

    # ---- per-kernel device time (library-side CUDA events on its stream), same K steps
    ctx.profile_read(reset=True)
    ctx.profile_enable(True)
    ms_prof_total = timed(lambda: step(pos_d), K)
    prof = ctx.profile_read(reset=True)
    ctx.profile_enable(False)

    peak, peak_src = measured_peaks()
    px_slices_per_step = units_rank
    kern = {k: v for k, v in prof.items() if v[1] > 0}
    dom = max(("k_row_transmit", "k_col_propagate"), key=lambda k: kern.get(k, (0.0, 0))[0])
    dom_ms, dom_n = kern[dom]
    alg_bytes_launch = (ROW_BYTES if dom == "k_row_transmit" else COL_BYTES) * px_slices_per_step * K / dom_n
    achieved = alg_bytes_launch / (dom_ms / dom_n * 1e-3) / 1e9
    ms_pair = kern["k_row_transmit"][0] + kern["k_col_propagate"][0]
    pair_gbs = (ROW_BYTES + COL_BYTES) * px_slices_per_step * K / (ms_pair * 1e-3) / 1e9
    traffic = None                                              # DRAM bytes per launch of that kernel, from ncu
    tj = {}
    tpath = os.path.join(ROOT, "profiles", "r1_traffic.json")
    if w.name == "c2_hbn_256" and args.frames is None and args.grid is None and not args.wave_chunk and os.path.exists(tpath):
        with open(tpath) as fh:
            tj = json.load(fh)["dram_bytes_per_launch"]
        traffic = next((v for k, v in tj.items() if k.startswith(dom + "<") and k.endswith(", 0>")), None)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                "bytes_per_launch": alg_bytes_launch, "avg_launch_ms": dom_ms / dom_n,
                "slice_step_pair": {"achieved": pair_gbs, "frac": pair_gbs / peak,
                                    "gpx_slice_s": px_slices_per_step * K / (ms_pair * 1e-3) / 1e9},
                "kernel_ms_per_step": {k: v[0] / K for k, v in kern.items()},
                "profiled_ms_per_step": ms_prof_total / K}
    if "k_tacaw_fft" in kern:
        tb = (8.0 * F + 4.0 * nb) * ctx.n_k_aperture * P + 4.0 * nb * (nx * ny - ctx.n_k_aperture) * P
        tms = kern["k_tacaw_fft"][0] / kern["k_tacaw_fft"][1]
        roofline["tacaw"] = {"achieved": tb / (tms * 1e-3) / 1e9, "frac": tb / (tms * 1e-3) / 1e9 / peak,
                             "bytes_per_launch": tb, "avg_launch_ms": tms,
                             "traffic": next((v for k, v in tj.items() if k.startswith("k_tacaw_tma") or k.startswith("k_tacaw_fft")), None)}

    if "k_vk" in kern:
        # V(k) structure-factor sums: 4 real sums per quarter-plane point and atom, x3 for the 3xTF32 split (tensor path)
        bf16 = 1590.0                                           # fallback of B200_PROFILING.md
        mp = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(mp):
            with open(mp) as fh:
                bf16 = float(json.load(fh).get("bf16_tflops", bf16))
        flop = 24.0 * (ctx.n_k_aperture / 4.0) * float(w.n_atoms) * F
        tms = kern["k_vk"][0] / K
        roofline["vk"] = {"bound": "tensor", "unit": "TFLOP/s", "achieved": flop / (tms * 1e-3) / 1e12,
                          "peak": 0.5 * bf16, "frac": flop / (tms * 1e-3) / 1e12 / (0.5 * bf16),
                          "note": "algorithmic 3xTF32 flops over the in-aperture quarter plane; peak = measured bf16 x 0.5 "
                                  "(guide's nominal tf32:bf16 ratio); FP32 path when ps_set_vk_mode(1) or few atoms per slice"}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline, _, _ = oracle_sample(make_workload(args.workload, n_frames=args.frames, grid=args.grid,
                                                           n_probes_side=args.probes_side))

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(3, args.warmup),
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex64 (f32)", "data": "synthetic",
            "config": {"workload": w.name, "grid": [nx, ny], "n_slices": S, "frames": F, "probes": P,
                       "atoms": int(w.n_atoms), "kV": w.kV, "omega_bins": nb,
                       "l2": "256 MiB buffer written between timed steps (L2 flush); per-step CUDA events",
                       "parallelism": f"independent trajectory per GPU x{world}, one all-reduce of I(k,w)"},
            "tacaw_end_to_end_s": ms_total / K * 1e-3,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / K, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu_baseline}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
