"""Host-side sharding of the TACAW path over ranks (one process per GPU, torch.distributed).

The path partitions over independent problems: (frame, probe) pairs are independent
through ps_build_slices / ps_multislice, so

  * P >= world  -> shard probes: every rank holds all frames of its probes; ps_tacaw and the
                   spectrum image are rank-local, the spectral diffraction pattern is one all-reduce
                   of a [ny][nx] image.  No exchange of waves.
  * P <  world  -> shard frames: every rank runs the streaming per-bin DFT (ps_tacaw_begin/add) on
                   its own frames with the GLOBAL frame index in the twiddle; the accumulators
                   acc[p][b][k] (and the mean slot) are linear in the frames, so ONE all-reduce (sum)
                   of the complex accumulators followed by ps_tacaw_finish gives I(k, w).
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


def plan(n_probes: int, n_frames: int, rank: int, world: int) -> ShardPlan:
    """Pick the sharding axis for this rank (see module docstring)."""
    if world == 1:
        return ShardPlan("probe", (0, n_probes), (0, n_frames), "none")
    if n_probes >= world:
        return ShardPlan("probe", shard_range(n_probes, rank, world), (0, n_frames),
                         "all_reduce(sdp image); spectrum image rank-local")
    return ShardPlan("frame", (0, n_probes), shard_range(n_frames, rank, world),
                     "all_reduce(sum) of the per-bin DFT accumulators, then ps_tacaw_finish")


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
