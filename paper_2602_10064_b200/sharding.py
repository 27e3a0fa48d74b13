"""Host-side sharding of the TACAW path over ranks (one process per GPU, torch.distributed).

The path partitions over independent problems: (frame, probe) pairs are independent
through ps_build_slices / ps_multislice, so

  * P >= world  -> shard probes: every rank holds all frames of its probes; ps_tacaw and the
                   spectrum image are rank-local, the spectral diffraction pattern is one all-reduce
                   of a [ny][nx] image.  No exchange of waves.
  * P <  world  -> shard frames: every rank runs the streaming per-bin DFT (ps_tacaw_begin/add) on
                   its own frames with the GLOBAL frame index in the twiddle and the SAME reference
                   wave; the accumulators acc[p][b][k] are linear in the frames, so ONE reduce-scatter
                   (sum) over k followed by ps_tacaw_finish_shard on the owned k-slice gives I(k, w).
  * independent trajectories -> every rank runs a whole trajectory; I(k, w) cubes
                   are summed with one all-reduce (what bench.py --gpus N measures: weak scaling).

Only index arithmetic and the collective calls live here; every kernel call goes through binding.py.
"""
from __future__ import annotations

from dataclasses import dataclass


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous balanced shard [lo, hi) of range(n): the first n % world ranks get one extra item."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


@dataclass(frozen=True)
class ShardPlan:
    axis: str            # "probe" | "frame"
    probes: tuple[int, int]
    frames: tuple[int, int]
    exchange: str        # which collective finishes the job


def plan(n_probes: int, n_frames: int, rank: int, world: int, axis: str | None = None) -> ShardPlan:
    """Pick the sharding axis for this rank (see module docstring); `axis` ("probe" | "frame") overrides the choice
    (used to drive the frame branch at world = 1, and to shard frames although there are enough probes)."""
    if axis not in (None, "probe", "frame"):
        raise ValueError("axis must be None, 'probe' or 'frame'")
    if axis is None and world == 1:
        return ShardPlan("probe", (0, n_probes), (0, n_frames), "none")
    if axis == "probe" and n_probes < world:
        raise ValueError("fewer probes than ranks: cannot shard probes")
    if axis == "probe" or (axis is None and n_probes >= world):
        return ShardPlan("probe", shard_range(n_probes, rank, world), (0, n_frames),
                         "all_reduce(sdp image); spectrum image rank-local")
    return ShardPlan("frame", (0, n_probes), shard_range(n_frames, rank, world),
                     "reduce_scatter(sum) of the per-bin DFT accumulators over k, ps_tacaw_finish_shard, all_gather of I")


def all_reduce_sum_(t, group=None):
    """In-place sum over ranks of a torch tensor (complex tensors go through their real view, which
    every backend supports).  No-op when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return t
    v = torch.view_as_real(t) if t.is_complex() else t
    dist.all_reduce(v, op=dist.ReduceOp.SUM, group=group)
    return t


def max_over_ranks(x: float, device=None, group=None) -> float:
    """Max over ranks of a host scalar (bench.py: step time is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


# ----------------------------------------------------------------------------------------------------------------------
# ONE problem sharded over ranks (strong scaling).  `ops` supplies the per-rank device work (the C-ABI calls on a GPU,
# see LibraryOps; the CPU test injects an implementation with the same methods), so the sharding arithmetic and the
# collectives below are exactly what `bench.py --scaling strong` runs.
def reduce_scatter_sum(t, group=None):
    """t: [world][...] on every rank -> the sum over ranks of slice [rank] (complex goes through its real view).
    NCCL: one reduce_scatter_tensor.  Other backends (gloo, used by the CPU test, has no reduce-scatter) use an
    all-reduce followed by the slice: same result, more traffic.  The choice is made by backend name, never by catching
    an error, so a real NCCL failure is not turned into world x the traffic."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        assert t.shape[0] == 1
        return t[0]
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    assert t.shape[0] == world
    v = torch.view_as_real(t) if t.is_complex() else t
    v = v.contiguous()
    out = torch.empty(v.shape[1:], dtype=v.dtype, device=v.device)
    if dist.get_backend(group) == "nccl":
        dist.reduce_scatter_tensor(out, v, op=dist.ReduceOp.SUM, group=group)   # a failure here is a failure: it propagates
    else:
        dist.all_reduce(v, op=dist.ReduceOp.SUM, group=group)
        out.copy_(v[rank])
    return torch.view_as_complex(out) if t.is_complex() else out


def all_gather_cat(t, group=None):
    """[n, ...] on every rank (same shape) -> [world * n, ...] in rank order."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return t
    world = dist.get_world_size(group)
    v = (torch.view_as_real(t) if t.is_complex() else t).contiguous()
    parts = [torch.empty_like(v) for _ in range(world)]
    dist.all_gather(parts, v, group=group)
    out = torch.cat(parts, dim=0)
    return torch.view_as_complex(out) if t.is_complex() else out


def tiled_exit_fraction(cell, nx: int, ny: int) -> float:
    """Share of the nx/8 column tiles that PS_LAYOUT_TILED_APERTURE stores: tiles holding a column m with
    |m| / Lx <= kc, kc = (2/3) min(nx / 2Lx, ny / 2Ly) (reading A10) — 44 of 64 at 512^2 on a square cell."""
    kc = (2.0 / 3.0) * min(nx / (2.0 * cell[0]), ny / (2.0 * cell[1]))
    tiles = set()
    for ix in range(nx):
        m = ix if ix < (nx + 1) // 2 else ix - nx
        if abs(m) / cell[0] <= kc:
            tiles.add(ix // 8)
    return len(tiles) / (nx // 8)


def probe_branch_bytes(cell, nx: int, ny: int, n_slices: int, n_frames: int, n_bins: int, probe_chunk: int,
                       work_bytes: int = 16 << 30) -> int:
    """Device bytes the probe branch of run_sharded holds on ONE rank, whatever the number of ranks: V of all frames,
    one probe chunk of tiled exit waves, its I cube, plus the library's work array (at most `work_bytes`)."""
    npix = nx * ny
    V = 4 * n_frames * n_slices * npix
    ex = int(8 * probe_chunk * n_frames * npix * tiled_exit_fraction(cell, nx, ny))
    I = 4 * probe_chunk * n_bins * npix
    return V + ex + I + work_bytes


def run_sharded(ops, n_probes: int, n_frames: int, bins, rank: int, world: int, frame_chunk: int = 64, sdp_bins=(1, 4),
                probe_chunk: int = 16, axis: str | None = None):
    """positions -> I(k, w) reductions for ONE trajectory, sharded per plan():

    probe axis: this rank's probes x all frames.  ps_build_slices (all frames) once, then `probe_chunk` probes at a time
        through ONE reused pair of buffers: ps_multislice into the tiled in-band exit layout -> ps_tacaw -> spectrum-image
        rows of the chunk, spectral diffraction pattern added up with ps_accumulate_intensity (the loop bench.py's
        full_config("c3") runs; config 3 per rank: 86 + 24 + 17 GB whatever the number of ranks, see
        probe_branch_bytes).  Then ONE all-reduce of the [ny][nx] spectral diffraction pattern and one of the zero-padded
        [P][n_bins] spectrum image.  No wave ever leaves its GPU.
    frame axis: this rank's frames x all probes, chunk by chunk: build V -> multislice -> ps_tacaw_add with the GLOBAL
        frame index (every rank subtracts the SAME reference wave: the exit wave of global frame 0, which each rank
        computes for itself); then ONE reduce-scatter of the complex accumulators over k (rank r keeps k-slice r),
        ps_tacaw_finish_shard on the owned slice, an all-gather of the I slices and the usual reductions.

    Returns {"sdp": [ny][nx], "spectrum_image": [P][n_bins], "I_local": this rank's part of I (probe axis: the cube of
    the LAST probe chunk only — earlier chunks' cubes are reduced and overwritten), "plan": ShardPlan}."""
    import torch
    pl = plan(n_probes, n_frames, rank, world, axis)
    nb = n_frames if bins is None else len(bins)
    if pl.axis == "probe":
        p0, p1 = pl.probes
        V = ops.build_slices(0, n_frames)
        sdp = simg = I = None
        for c0 in range(p0, p1, max(1, probe_chunk)):
            c1 = min(p1, c0 + max(1, probe_chunk))
            ex = ops.multislice(ops.incident(c0, c1), V, tiled=True)
            I = ops.tacaw(ex, bins)                                       # [c1-c0][nb][ny][nx], buffer reused per chunk
            rows = ops.spectrum_image(I)
            if simg is None:
                simg = torch.zeros((n_probes, nb), dtype=torch.float32, device=rows.device)
            simg[c0:c1] = rows
            part = ops.sdp(I, *sdp_bins)
            sdp = part.clone() if sdp is None else ops.accumulate(sdp, part)
        all_reduce_sum_(sdp)
        all_reduce_sum_(simg)
        return {"sdp": sdp, "spectrum_image": simg, "I_local": I, "plan": pl}
    if bins is None:
        raise ValueError("frame sharding uses the streaming per-bin DFT: a bin list is required")
    f0, f1 = pl.frames
    psi0 = ops.incident(0, n_probes)
    ref = ops.multislice(psi0, ops.build_slices(0, 1))[:, 0].contiguous()   # exit wave of global frame 0, same on every rank
    ops.stream_begin(n_probes, n_frames, bins)
    ops.stream_set_reference(ref)
    for c0 in range(f0, f1, frame_chunk):
        c1 = min(f1, c0 + frame_chunk)
        ops.stream_add(ops.multislice(psi0, ops.build_slices(c0, c1)), c0)
    acc = ops.stream_accumulators()                                       # complex64 [P][nb][ny*nx]
    P, _, npix = acc.shape
    pad = (-npix) % world
    if pad:
        acc = torch.cat([acc, torch.zeros((P, nb, pad), dtype=acc.dtype, device=acc.device)], dim=2)
    n_k = acc.shape[2] // world
    shard = reduce_scatter_sum(acc.reshape(P * nb, world, n_k).permute(1, 0, 2).contiguous())   # [P*nb][n_k], k-slice `rank`
    I_shard = ops.stream_finish_shard(shard.reshape(P, nb, n_k))          # float32 [P][nb][n_k]
    I_full = all_gather_cat(I_shard.reshape(1, P * nb, n_k)).permute(1, 0, 2).reshape(P, nb, world * n_k)[:, :, :npix]
    I_full = ops.as_images(I_full.contiguous())                           # [P][nb][ny][nx]
    return {"sdp": ops.sdp(I_full, *sdp_bins), "spectrum_image": ops.spectrum_image(I_full), "I_local": I_shard, "plan": pl}


class LibraryOps:
    """run_sharded's device work through the C ABI (binding.py) for workload `w` on context `ctx`."""

    def __init__(self, ps, ctx, w, pos_d, Z_d):
        self.ps, self.ctx, self.w, self.pos_d, self.Z_d = ps, ctx, w, pos_d, Z_d
        self.stream = None
        self._bufs = {}

    def build_slices(self, f0, f1):
        import torch
        d_V = self._buf("V", (f1 - f0, self.ctx.n_slices, self.ctx.ny, self.ctx.nx), torch.float32)
        return self.ps.ps_build_slices(self.ctx, self.pos_d[f0:f1], self.Z_d, d_V=d_V)

    def incident(self, p0, p1):
        import numpy as np
        w = self.w
        if w.beam == "probe":
            return self.ps.ps_make_incident(self.ctx, w.kV, w.semi_angle_mrad, w.probe_xy[p0:p1])
        if w.beam == "tilt":
            return self.ps.ps_make_incident(self.ctx, w.kV, 0.0, w.tilts[p0:p1].astype(np.float64), is_tilt=True)
        return self.ps.ps_make_incident(self.ctx, w.kV)

    def _buf(self, key, shape, dtype):
        """one device buffer per role, re-used while the shape stays the same (probe chunks, timed steps)"""
        import torch
        b = self._bufs.get(key)
        if b is None or tuple(b.shape) != tuple(shape) or b.dtype != dtype:
            self._bufs.pop(key, None)
            b = self._bufs[key] = torch.empty(tuple(shape), dtype=dtype, device=self.ctx.device)
        return b

    def multislice(self, psi0, V, tiled=False):
        import torch
        ps = self.ps
        if not tiled:
            return ps.ps_multislice(self.ctx, self.w.kV, psi0, V)
        shape = ps.exit_shape(self.ctx, int(psi0.shape[0]), int(V.shape[0]), ps.PS_LAYOUT_TILED_APERTURE)
        return ps.ps_multislice(self.ctx, self.w.kV, psi0, V, d_exit=self._buf("exit_tiled", shape, torch.complex64))

    def tacaw(self, ex, bins):
        import torch
        P = int(ex.shape[0])
        F = int(ex.shape[1] if ex.dim() == 4 else ex.shape[3])
        nb = F if bins is None else len(bins)
        d_I = self._buf("I", (P, nb, self.ctx.ny, self.ctx.nx), torch.float32)
        return self.ps.ps_tacaw(self.ctx, ex, self.w.dt_fs, bins, d_I=d_I)

    def sdp(self, I, lo, hi):
        import torch
        d_out = self._buf("sdp_part", (self.ctx.ny, self.ctx.nx), torch.float32)
        return self.ps.ps_sdp(self.ctx, I, lo, min(hi, I.shape[1] - 1), d_out=d_out)

    def accumulate(self, acc, part):
        return self.ps.ps_accumulate_intensity(self.ctx, acc, part, 1.0, 1.0)

    def spectrum_image(self, I):
        return self.ps.ps_spectrum_image(self.ctx, I)

    def stream_begin(self, P, F, bins):
        from .binding import TacawStream
        self.stream = TacawStream(self.ctx, P, F, self.w.dt_fs, bins)

    def stream_set_reference(self, ref):
        self.stream.set_reference(ref)

    def stream_add(self, ex, frame0):
        self.stream.add(ex, frame0)

    def stream_accumulators(self):
        a = self.stream.d_acc
        return a.reshape(a.shape[0], a.shape[1], -1)

    def stream_finish_shard(self, acc_shard):
        return self.stream.finish_shard(acc_shard.contiguous())

    def as_images(self, I_flat):
        return I_flat.reshape(I_flat.shape[0], I_flat.shape[1], self.ctx.ny, self.ctx.nx)


def run_strong_bench(args, w, rank, world, dev, ps, metric, unit):
    """bench.py --gpus N --scaling strong: K timed steps of run_sharded on ONE trajectory (same seed on every rank),
    barrier + synchronize on both sides, max over ranks, one JSON line from rank 0."""
    import json
    import torch
    import torch.distributed as dist
    from workloads import form_factor_coefficients
    ctx = ps.Context(dev.index)
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    ctx.set_form_factors(w.elements, nl, ng, coef)
    ctx.set_geometry(w.cell, w.nx, w.ny, w.slice_dz)
    pos_d = torch.from_numpy(w.positions()).to(dev)
    Z_d = torch.from_numpy(w.Z.copy()).to(dev)
    ops = LibraryOps(ps, ctx, w, pos_d, Z_d)
    bins = w.bins
    pl = plan(w.n_probes, w.n_frames, rank, world)
    if pl.axis == "frame" and bins is None:
        import numpy as np
        bins = np.arange(min(256, w.n_frames), dtype=np.int32)

    def step():
        return run_sharded(ops, w.n_probes, w.n_frames, bins, rank, world, probe_chunk=getattr(args, "probe_chunk", 16) or 16)

    def barrier():
        if dist.is_available() and dist.is_initialized():
            dist.barrier()
        torch.cuda.synchronize()

    W, K = max(3, args.warmup), max(1, args.steps)
    for _ in range(W):
        step()
    barrier()
    l0 = ctx.launches
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(K):
        out = step()
    b.record()
    barrier()
    ms = max_over_ranks(a.elapsed_time(b), device=dev)
    units = float(w.nx) * w.ny * w.n_slices * w.n_frames * w.n_probes
    if rank == 0:
        print(json.dumps({
            "metric": metric, "value": units * K / (ms * 1e-3) / 1e9, "unit": unit, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "complex64 (f32)", "data": "synthetic",
            "config": {"workload": getattr(w, "label", w.name), "grid": [w.nx, w.ny], "n_slices": w.n_slices,
                       "frames": w.n_frames, "probes": w.n_probes, "atoms": int(w.n_atoms),
                       "parallelism": f"{pl.axis} shards x{world}: {pl.exchange}"},
            "gpu_launches": int(ctx.launches - l0),
            "checksum_spectrum_image": float(out["spectrum_image"].sum())}))
