"""GPU test of `ps_spectrum_image_static`, the spectrum-image reduction for callers that cannot allocate device memory.

Who needs it: a host program that has already handed all free HBM to its own memory pool (a `cudaMalloc` made by the
library would fail there), or a latency-bound serving loop that cannot accept the device-wide stall `cudaMalloc` /
`cudaFree` cause.  `ps_spectrum_image` allocates its detector mask through the ctx; the `_static` variant keeps the
mask in a 1 MiB array built into the library (grids up to 1024 x 1024) and calls no allocator.

What is checked: on the same seeded `I` cube the new entry point returns what the existing `ps_spectrum_image` path
returns, within the tolerance the reduction tests use (`TOL_RED`, relative L2), on two calls in a row with different
detectors (the shared array still holds the first call's mask when the second starts), then on a smaller grid (stale
bytes beyond the new grid must not matter); and a grid beyond the limit is refused with a clear message and no output
written.  The new entry point runs first on a fresh context, so it cannot be borrowing a mask the old path allocated.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It needs nothing from the other test files and passes alone in a fresh process as well as after them.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_RED = 1e-5          # the tolerance of the reduction checks in tests/test_gpu_parity.py


def _rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def _ctx(cell, nx, ny):
    import paper_2602_10064_b200 as ps
    ctx = ps.Context(0)
    ctx.set_geometry(np.asarray(cell, dtype=np.float64), nx, ny, cell[2])
    return ctx


def _cube(P, n_bins, ny, nx, seed):
    import torch
    g = torch.Generator(device="cpu").manual_seed(seed)
    I = torch.rand((P, n_bins, ny, nx), generator=g, dtype=torch.float32) ** 4      # non-negative, wide dynamic range
    return I.cuda()


def test_static_entry_point_matches_existing_path_on_two_calls_in_a_row():
    import torch
    import paper_2602_10064_b200 as ps

    assert ps.static_scratch_bytes() == 1024 * 1024
    cell, nx, ny = (9.0, 7.0, 4.0), 128, 64                       # non-square cell and grid
    kc = (2.0 / 3.0) * min(nx / (2 * cell[0]), ny / (2 * cell[1]))
    P, n_bins = 3, 5
    I = _cube(P, n_bins, ny, nx, seed=20260210)
    detectors = [(0.2 * kc, 0.7 * kc), (0.0, 0.0), (0.5 * kc, 0.0)]   # annulus, every pixel, outer region

    fresh = _ctx(cell, nx, ny)                                    # has never run ps_spectrum_image: owns no mask buffer
    outs = [torch.full((P, n_bins), float("nan"), device="cuda") for _ in detectors]
    for (k_in, k_out), out in zip(detectors, outs):               # back to back on one stream, no sync in between
        ps.ps_spectrum_image_static(fresh, I, out, k_in, k_out)
    torch.cuda.synchronize()

    old = _ctx(cell, nx, ny)
    for (k_in, k_out), out in zip(detectors, outs):
        want = ps.ps_spectrum_image(old, I, k_in, k_out).cpu().numpy()
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        assert _rel_l2(got, want) < TOL_RED, (k_in, k_out)
    # "every pixel" has a definition that needs no mask at all
    assert _rel_l2(outs[1].cpu().numpy(), I.double().sum(dim=(2, 3)).cpu().numpy()) < TOL_RED

    # a smaller grid next: the array still holds 8192 bytes of the 128 x 64 masks, only the first 1024 are rewritten
    cell2 = (5.0, 6.0, 3.0)
    small_new, small_old = _ctx(cell2, 32, 32), _ctx(cell2, 32, 32)
    I2 = _cube(2, 4, 32, 32, seed=7)
    kc2 = (2.0 / 3.0) * min(32 / (2 * cell2[0]), 32 / (2 * cell2[1]))
    out2 = torch.full((2, 4), float("nan"), device="cuda")
    ps.ps_spectrum_image_static(small_new, I2, out2, 0.1 * kc2, 0.9 * kc2)
    want2 = ps.ps_spectrum_image(small_old, I2, 0.1 * kc2, 0.9 * kc2).cpu().numpy()
    assert _rel_l2(out2.cpu().numpy(), want2) < TOL_RED

    # and the first grid again after that, through the first context
    again = torch.full((P, n_bins), float("nan"), device="cuda")
    ps.ps_spectrum_image_static(fresh, I, again, *detectors[0])
    assert torch.equal(again, outs[0])                            # fixed summation order: the same bits every time
    for c in (fresh, old, small_new, small_old):
        c.close()


def test_static_entry_point_refuses_grids_beyond_its_array():
    import torch
    import paper_2602_10064_b200 as ps

    ctx = _ctx((40.0, 20.0, 4.0), 2048, 1024)                     # 2 Mi pixels > the 1 Mi the array holds
    I = torch.ones((1, 1, 1024, 2048), dtype=torch.float32, device="cuda")
    out = torch.full((1, 1), -1.0, device="cuda")
    with pytest.raises(ps.PSError) as err:
        ps.ps_spectrum_image_static(ctx, I, out)
    assert err.value.status == ps.binding.PS_EUNSUPPORTED
    assert "1024 x 1024" in str(err.value) and "ps_spectrum_image" in str(err.value)
    torch.cuda.synchronize()
    assert float(out[0, 0]) == -1.0                               # nothing was launched
    assert float(ps.ps_spectrum_image(ctx, I)[0, 0]) == 2048 * 1024   # the allocating path still serves this grid

    at_limit = _ctx((20.0, 20.0, 4.0), 1024, 1024)                # exactly the maximum is accepted
    I1 = torch.ones((1, 2, 1024, 1024), dtype=torch.float32, device="cuda")
    out1 = torch.zeros((1, 2), device="cuda")
    ps.ps_spectrum_image_static(at_limit, I1, out1)
    assert out1.cpu().tolist() == [[1024.0 * 1024.0] * 2]
    ctx.close(); at_limit.close()
