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


def _worker(rank, world, port, case, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        if case == "frame":
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


@pytest.mark.parametrize("case", ["frame", "probe", "trajectory"])
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
