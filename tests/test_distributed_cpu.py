"""World-size-2 gloo tests (CPU) of the multi-GPU host logic.

The kernels cannot run here, so each rank's device work is stood in for by the NumPy definition of the
same quantity (per-bin DFT partial sums over the rank's frames with the GLOBAL frame index; rank-local
|.|^2 for probe shards); what is under test is the sharding arithmetic and the collectives of
paper_2602_10064_b200/sharding.py: the combined result must equal the oracle on the whole problem.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import tacaw_oracle as O
from paper_2602_10064_b200 import sharding


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _exit_waves(P, F, n=6, seed=3):
    rng = np.random.default_rng(seed)
    return (rng.normal(size=(P, F, n, n)) + 1j * rng.normal(size=(P, F, n, n))) * 0.1 + (2.0 - 1.0j)


class OracleOps:
    """run_sharded's device work stood in for by the float64 oracle (the kernels cannot run here): same methods as
    sharding.LibraryOps, torch CPU tensors in and out.  The streaming accumulator follows the contract of
    include/pyslice_b200.h (global frame index in the twiddle, shared reference wave, bin 0 := 0)."""

    def __init__(self, w):
        from workloads import form_factor_coefficients
        self.w = w
        self.nl, self.ng, self.coef = form_factor_coefficients(w.elements, w.ff_kind)
        self.elem = np.searchsorted(w.elements, w.Z)
        self.pos = w.positions()

    def build_slices(self, f0, f1):
        w = self.w
        return np.stack([O.projected_potential(self.pos[f], self.elem, self.coef, self.nl, self.ng, w.cell, w.nx, w.ny,
                                               w.n_slices)[0] for f in range(f0, f1)])

    def incident(self, p0, p1):
        w = self.w
        if w.beam == "probe":
            return [O.probe_wave(w.cell, w.nx, w.ny, w.kV, w.semi_angle_mrad, x, y) for x, y in w.probe_xy[p0:p1]]
        return [O.plane_wave(w.nx, w.ny)]

    def accumulate(self, acc, part):
        acc += part
        return acc

    def multislice(self, psi0, V, tiled=False):                          # the layout is the library's business: same values
        return torch.from_numpy(np.stack([[O.multislice(p, v, self.w.cell, self.w.kV) for v in V] for p in psi0]))

    def tacaw(self, ex, bins):
        return torch.from_numpy(np.stack([O.tacaw_intensity(e, bins) for e in ex.numpy()]).astype(np.float32))

    def sdp(self, I, lo, hi):
        return torch.from_numpy(O.sdp(I.numpy().astype(np.float64), lo, min(hi, I.shape[1] - 1)).astype(np.float32))

    def spectrum_image(self, I):
        return torch.from_numpy(I.numpy().astype(np.float64).sum(axis=(2, 3)).astype(np.float32))

    def stream_begin(self, P, F, bins):
        self.F, self.bins = F, np.asarray(bins) % F
        self.acc = np.zeros((P, len(bins), self.w.ny * self.w.nx), complex)
        self.ref = None

    def stream_set_reference(self, ref):
        self.ref = ref.numpy().reshape(ref.shape[0], 1, -1)

    def stream_add(self, ex, frame0):
        x = ex.numpy().reshape(ex.shape[0], ex.shape[1], -1) - self.ref
        j = frame0 + np.arange(ex.shape[1])
        self.acc += np.einsum("bj,pjk->pbk", np.exp(-2j * np.pi * np.outer(self.bins, j) / self.F), x)

    def stream_accumulators(self):
        return torch.from_numpy(self.acc)

    def stream_finish_shard(self, acc_shard):
        I = np.abs(acc_shard.numpy()) ** 2
        I[:, self.bins == 0] = 0.0
        return torch.from_numpy(I.astype(np.float32))

    def as_images(self, I_flat):
        return I_flat.reshape(I_flat.shape[0], I_flat.shape[1], self.w.ny, self.w.nx)


def _sharded_case(case, rank, world):
    """The function bench.py --scaling strong runs (sharding.run_sharded), with the oracle as the device: the combined
    result must equal the oracle on the whole, unsharded problem."""
    from workloads import make_workload
    if case == "sharded_probe":
        w = make_workload("c3_si_probe_512", mini=True, n_frames=8, grid=32)          # 4 probes >= 2 ranks
        w.n_slices = 2
        bins = None
    else:
        w = make_workload("c1_si_128", mini=True, n_frames=13, grid=32)              # 1 probe < 2 ranks, ragged frames
        w.n_slices = 2
        bins = np.array([0, 1, 2, -1, 5, -6], dtype=np.int64)
    ops = OracleOps(w)
    out = sharding.run_sharded(ops, w.n_probes, w.n_frames, bins, rank, world, frame_chunk=3, probe_chunk=1)   # 2 chunks per rank
    assert out["plan"].axis == ("probe" if case == "sharded_probe" else "frame")
    I_all, _ = O.run_path(ops.pos, ops.elem, ops.coef, ops.nl, ops.ng, w.cell, w.nx, w.ny, w.n_slices, w.kV,
                          ops.incident(0, w.n_probes), bins)
    want_sdp = O.sdp(I_all, 1, min(4, I_all.shape[1] - 1))
    want_si = I_all.sum(axis=(2, 3))
    ok = np.allclose(out["sdp"].numpy(), want_sdp, rtol=2e-5, atol=1e-6 * want_sdp.max())
    ok = ok and np.allclose(out["spectrum_image"].numpy(), want_si, rtol=2e-5, atol=1e-6 * want_si.max())
    if case == "sharded_frame":                                                      # this rank's k-slice of I
        npix = w.nx * w.ny
        n_k = -(-npix // world)
        mine = I_all.reshape(1, len(bins), npix)[:, :, rank * n_k:(rank + 1) * n_k]
        got = out["I_local"].numpy()[:, :, :mine.shape[2]]
        ok = ok and np.allclose(got, mine, rtol=2e-5, atol=1e-6 * I_all.max())
    return ok


def _worker(rank, world, port, case, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        if case.startswith("sharded_"):
            ok = _sharded_case(case, rank, world)
        elif case == "frame":
            P, F = 1, 37                                            # P < world -> frame shards, ragged split
            bins = np.array([0, 1, -1, 5, 18, -18], dtype=np.int64)
            x = _exit_waves(P, F)
            pl = sharding.plan(P, F, rank, world)
            assert pl.axis == "frame"
            f0, f1 = pl.frames
            j = np.arange(f0, f1)
            tw = np.exp(-2j * np.pi * np.outer(bins % F, j) / F)     # [nb][f_local], global frame index
            acc = np.einsum("bj,pjyx->pbyx", tw, x[:, f0:f1])
            mean_slot = x[:, f0:f1].sum(axis=1, keepdims=True)
            acc_t = torch.from_numpy(np.concatenate([acc, mean_slot], axis=1).astype(np.complex128))
            sharding.all_reduce_sum_(acc_t)
            a = acc_t.numpy()
            nb = len(bins)
            corr = np.where((bins % F == 0)[None, :, None, None], a[:, nb:nb + 1], 0.0)   # F * mean at bin 0
            I = np.abs(a[:, :nb] - corr) ** 2
            want = np.stack([O.tacaw_intensity(x[p], bins) for p in range(P)])
            ok = np.allclose(I, want, rtol=1e-10, atol=1e-12 * want.max())
        elif case == "probe":
            P, F = 5, 16                                             # P >= world -> probe shards, ragged split
            x = _exit_waves(P, F, seed=4)
            pl = sharding.plan(P, F, rank, world)
            assert pl.axis == "probe" and pl.frames == (0, F)
            p0, p1 = pl.probes
            I_loc = np.stack([O.tacaw_intensity(x[p]) for p in range(p0, p1)])
            sdp = torch.from_numpy(O.sdp(I_loc, 1, 4))
            sharding.all_reduce_sum_(sdp)
            want = O.sdp(np.stack([O.tacaw_intensity(x[p]) for p in range(P)]), 1, 4)
            ok = np.allclose(sdp.numpy(), want, rtol=1e-12)
            counts = torch.tensor([p1 - p0])
            dist.all_reduce(counts)
            ok = ok and int(counts.item()) == P
        elif case == "trajectory":
            x = _exit_waves(1, 16, seed=10 + rank)                   # an independent trajectory per rank
            I = torch.from_numpy(O.tacaw_intensity(x[0]))
            sharding.all_reduce_sum_(I)
            want = sum(O.tacaw_intensity(_exit_waves(1, 16, seed=10 + r)[0]) for r in range(world))
            ok = np.allclose(I.numpy(), want, rtol=1e-12)
            t = sharding.max_over_ranks(1.0 + rank)
            ok = ok and t == float(world)
        else:
            ok = False
        out[rank] = bool(ok)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("case", ["frame", "probe", "trajectory", "sharded_probe", "sharded_frame"])
def test_world_size_2_gloo(case):
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), case, out), nprocs=world, join=True)
    assert dict(out) == {0: True, 1: True}


def test_shard_range_covers_everything_once():
    for n in (0, 1, 7, 16, 257):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                lo, hi = sharding.shard_range(n, r, world)
                assert 0 <= lo <= hi <= n
                got.extend(range(lo, hi))
            assert got == list(range(n))
            sizes = [sharding.shard_range(n, r, world)[1] - sharding.shard_range(n, r, world)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_plan_axes():
    assert sharding.plan(256, 1024, 3, 8).axis == "probe"
    assert sharding.plan(1, 4096, 3, 8).axis == "frame"
    assert sharding.plan(1, 4096, 0, 1).exchange == "none"


def test_probe_branch_fits_config_3_on_every_rank_count():
    """the probe branch of run_sharded holds V of all frames plus ONE 16-probe chunk of
    tiled exit waves and its I cube, whatever the number of ranks: config 3 (1024 frames x 512^2 x 80 slices, all 1024
    bins) must stay under 170 GB of a 180 GB B200, work array of the library included."""
    from workloads import make_workload
    w = make_workload("c3_si_probe_512")
    assert abs(sharding.tiled_exit_fraction(w.cell, w.nx, w.ny) - 44 / 64) < 1e-12
    need = sharding.probe_branch_bytes(w.cell, w.nx, w.ny, w.n_slices, w.n_frames, w.n_frames, probe_chunk=16)
    assert need < 170e9, need
    dense_all = 8 * 32 * w.n_frames * w.nx * w.ny + 4 * 32 * w.n_frames * w.nx * w.ny + 4 * w.n_frames * w.n_slices * w.nx * w.ny
    assert dense_all > 180e9                                            # what the unchunked dense plan needed at 8 ranks
    for world in (1, 2, 4, 8):
        for rank in range(world):
            pl = sharding.plan(w.n_probes, w.n_frames, rank, world)
            assert pl.axis == "probe" and (pl.probes[1] - pl.probes[0]) * world == w.n_probes


def test_plan_forced_axis():
    pl = sharding.plan(4, 10, 0, 1, axis="frame")
    assert pl.axis == "frame" and pl.frames == (0, 10) and pl.probes == (0, 4)
    with pytest.raises(ValueError):
        sharding.plan(1, 10, 0, 2, axis="probe")
    with pytest.raises(ValueError):
        sharding.plan(1, 10, 0, 2, axis="time")
