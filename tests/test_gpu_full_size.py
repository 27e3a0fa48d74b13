"""GPU parity at BASELINE.json's full grid / slice / atom sizes, in the launch configuration bench.py times
(library-default chunking, whole batches per launch), on SAMPLED outputs the float64 oracle can compute one by one
(SURVEY.md §8(d) "Parity sampling"):

  * integers (slice binning) on every atom of the sampled frames: bit-exact;
  * V on sampled slices of sampled frames against the oracle's potential from positions;
  * exit waves of sampled (frame, probe) pairs against the oracle's slice loop run on the same float32 potentials
    (the CUDA potentials, which the previous bullet ties to the oracle);
  * I(k, w) on a seeded sample of k-pixels over all frames against the oracle's time transform of the same
    exit-wave columns; out-of-band pixels exactly zero;
  * properties that hold at any size: norm inside the band limit (pin P8), path-B == path-A.

Frame counts are cut where the full count would not fit the test budget (the oracle needs ~1 s per 256^2 frame,
~50 s per 512^2 x 80-slice frame); grid, slices, atoms, probes-per-launch and bins are the configs' own.
"""
import numpy as np
import pytest

from oracle import tacaw_oracle as O
from workloads import make_workload

from gpu_common import gpu_incident, make_ctx, oracle_incident, oracle_potential, rel_l2

pytestmark = pytest.mark.gpu

TOL_EXIT = 1e-4
TOL_I = 1e-3
TOL_V = 2e-5


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    return torch


def _t(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _check_tacaw_sample(torch, ps, ctx, w, ex, I, bins, n_sample, seed):
    """I[p][b][pix] against the oracle transform of the CUDA exit waves at sampled in-band pixels; zeros elsewhere."""
    A = O.aperture_mask(w.cell, w.nx, w.ny)
    iy, ix = np.nonzero(A)
    rng = np.random.default_rng(seed)
    sel = rng.choice(iy.size, size=min(n_sample, iy.size), replace=False)
    sy, sx = torch.as_tensor(iy[sel]).cuda(), torch.as_tensor(ix[sel]).cuda()
    P, F = ex.shape[0], ex.shape[1]
    for p in range(P):
        cols = ex[p][:, sy, sx].cpu().numpy().astype(np.complex128)          # [F][n_sample]
        Io = O.tacaw_intensity(cols, bins)
        Ig = I[p][:, sy, sx].cpu().numpy()
        assert rel_l2(Ig, Io) < TOL_I
    out = torch.as_tensor(~A).cuda()
    assert float(I[:, :, out].abs().max()) == 0.0, "I outside the band limit must be exactly zero"


def _check_norm(torch, ex, w):
    """P8: exp(i sigma V) is unitary and P A only removes intensity: sum_k |Psi|^2 <= nx ny, and close to it."""
    n = (ex.real.double() ** 2 + ex.imag.double() ** 2).sum(dim=(-2, -1)) / (w.nx * w.ny)
    assert float(n.max()) <= 1.0 + 1e-5
    assert float(n.min()) > 0.5


def test_c2_full_bench_configuration(torch):
    """Config 2 exactly as bench.py runs it: 1152 atoms, 256^2, 10 slices, all 512 frames, bins 0..49."""
    import paper_2602_10064_b200 as ps
    w = make_workload("c2_hbn_256")
    ctx = make_ctx(w)
    pos = w.positions()
    V, sidx = ps.ps_build_slices(ctx, _t(torch, pos), _t(torch, w.Z), want_slice_idx=True)
    ex = ps.ps_multislice(ctx, w.kV, gpu_incident(ctx, w), V)
    I = ps.ps_tacaw(ctx, ex, w.dt_fs, w.bins)
    psi0 = oracle_incident(w)[0]
    for f in (0, 257, w.n_frames - 1):
        Vo, so = oracle_potential(w, pos[f])
        assert np.array_equal(sidx[f].cpu().numpy(), so), "slice binning must be bit-exact"
        assert rel_l2(V[f].cpu().numpy(), Vo) < TOL_V
        eo = O.multislice(psi0, Vo, w.cell, w.kV)                              # positions -> exit wave, all oracle
        assert rel_l2(ex[0, f].cpu().numpy(), eo) < TOL_EXIT
    # binning of every atom of every frame
    so_all = O.slice_index(O.fixed_point(pos.reshape(-1, 3), w.cell)[:, 2], w.n_slices).reshape(pos.shape[:2])
    assert np.array_equal(sidx.cpu().numpy(), so_all)
    _check_norm(torch, ex, w)
    _check_tacaw_sample(torch, ps, ctx, w, ex, I, w.bins, 4096, 21)


def test_c3_full_grid_probe_chunk(torch):
    """Config 3 geometry (10 240 atoms, 512^2, 80 slices, 30 mrad probes), 32 frames x one 16-probe scan row."""
    import paper_2602_10064_b200 as ps
    F = 32
    w = make_workload("c3_si_probe_512", n_frames=F)
    w.probe_xy = w.probe_xy[:16]
    ctx = make_ctx(w)
    pos = w.positions()
    V, sidx = ps.ps_build_slices(ctx, _t(torch, pos), _t(torch, w.Z), want_slice_idx=True)
    psi0 = gpu_incident(ctx, w)
    ex = ps.ps_multislice(ctx, w.kV, psi0, V)
    # bench.py's default step keeps the exit waves in the tiled layout: the same bits, and I(k, w) is taken from it
    tiled = ps.ps_multislice(ctx, w.kV, psi0, V, layout=ps.PS_LAYOUT_TILED_APERTURE)
    assert torch.equal(ps.ps_exit_to_dense(ctx, tiled), ex)
    I = ps.ps_tacaw(ctx, tiled, w.dt_fs)
    f = 17
    Vo, so = oracle_potential(w, pos[f], slices=(0, 41, 79))
    assert np.array_equal(sidx[f].cpu().numpy(), so)
    Vg = V[f].cpu().numpy()
    for s in (0, 41, 79):
        assert rel_l2(Vg[s], Vo[s]) < TOL_V
    po = oracle_incident(w)
    for p, fr in ((0, 0), (15, f)):
        eo = O.multislice(po[p], V[fr].cpu().numpy().astype(np.float64), w.cell, w.kV)
        assert rel_l2(ex[p, fr].cpu().numpy(), eo) < TOL_EXIT
    _check_norm(torch, ex, w)
    _check_tacaw_sample(torch, ps, ctx, w, ex, I, None, 1024, 31)


def test_c3_bench_shape(torch):
    """The step bench.py times by default, unchanged: config 3's own 10 240 atoms, 512^2, 80 slices, ALL 1024 frames x one
    16-probe scan row, exit waves in PS_LAYOUT_TILED_APERTURE (several work-array chunks per call, library-default
    chunking), k_tacaw_tma<1024, tiled> over all 1024 bins, then the spectrum image.  127 GB resident, ~2 s of GPU time.
      (a) V from positions on 2 frames x 3 slices; slice binning of those frames bit-exact;
      (b) exit waves of 4 (probe, frame) pairs spread over the work-array chunks against the oracle's slice loop;
      (c) I(k, w) at 1024 seeded in-band pixels x all 1024 bins against the oracle transform of the same exit-wave
          columns, as a whole and bin by bin (weak bins get the fp32 floor of a length-F transform, eps log2(F) times
          the strongest line's amplitude, the elastic one included: DESIGN.md §7); out-of-band pixels exactly zero;
      (d) Parseval over the whole cube (pin P11, holds at any size): sum_{k, n} I = F sum_{k, t} |Psi - <Psi>_t|^2 per
          probe, the left side taken from ps_spectrum_image over all k — the number bench.py --full-config c3 prints as
          its checksum is the sum of exactly these."""
    import paper_2602_10064_b200 as ps
    w = make_workload("c3_si_probe_512")
    w.probe_xy = w.probe_xy[:16]
    F, S, nx, ny = w.n_frames, w.n_slices, w.nx, w.ny
    assert (F, S, nx, ny, w.n_atoms) == (1024, 80, 512, 512, 10240)
    ctx = make_ctx(w)
    pos = w.positions()
    V = torch.empty((F, S, ny, nx), dtype=torch.float32, device="cuda")
    sidx = torch.empty((F, w.n_atoms), dtype=torch.int32, device="cuda")
    ps.ps_build_slices(ctx, _t(torch, pos), _t(torch, w.Z), d_V=V, d_slice_idx=sidx)
    psi0 = gpu_incident(ctx, w)
    ex = ps.ps_multislice(ctx, w.kV, psi0, V, layout=ps.PS_LAYOUT_TILED_APERTURE)
    I = ps.ps_tacaw(ctx, ex, w.dt_fs)
    simg = ps.ps_spectrum_image(ctx, I)
    ctx.check_async()
    assert tuple(I.shape) == (16, F, ny, nx)

    # (a)
    for f in (205, 1023):
        Vo, so = oracle_potential(w, pos[f], slices=(0, 41, 79))
        assert np.array_equal(sidx[f].cpu().numpy(), so), "slice binning must be bit-exact"
        Vg = V[f].cpu().numpy()
        for s in (0, 41, 79):
            assert rel_l2(Vg[s], Vo[s]) < TOL_V

    # (b), (d): one probe at a time through the dense view (2.1 GB)
    po = oracle_incident(w)
    pairs = {0: (0,), 5: (205,), 10: (613,), 15: (1023,)}
    A = O.aperture_mask(w.cell, nx, ny)
    iy, ix = np.nonzero(A)
    sel = np.random.default_rng(1024).choice(iy.size, size=1024, replace=False)
    sy, sx = torch.as_tensor(iy[sel]).cuda(), torch.as_tensor(ix[sel]).cuda()
    eps32 = float(np.finfo(np.float32).eps)
    dense = torch.empty((1, F, ny, nx), dtype=torch.complex64, device="cuda")
    for p in range(16):
        ps.ps_exit_to_dense(ctx, ex[p:p + 1], d_dense=dense)
        for fr in pairs.get(p, ()):
            eo = O.multislice(po[p], V[fr].cpu().numpy().astype(np.float64), w.cell, w.kV)
            assert rel_l2(dense[0, fr].cpu().numpy(), eo) < TOL_EXIT, (p, fr)
        # (c)
        cols = dense[0][:, sy, sx].cpu().numpy().astype(np.complex128)            # [F][1024]
        Io = O.tacaw_intensity(cols, None)
        Ig = I[p][:, sy, sx].cpu().numpy().astype(np.float64)
        assert rel_l2(Ig, Io) < TOL_I, p
        # amplitude floor of the fp32 transform: eps log2(F) x the strongest line it carries, the elastic one (F <Psi>_t,
        # removed by the mean subtraction only up to rounding) included
        strongest = max(Io.mean(axis=1).max(), float(np.mean(np.abs(cols.sum(axis=0)) ** 2)))
        floor = eps32 * np.log2(F) * np.sqrt(strongest)
        for b in range(F):
            allowed = TOL_I * np.linalg.norm(Io[b]) + np.linalg.norm(2.0 * np.sqrt(Io[b]) * floor + floor ** 2)
            assert np.linalg.norm(Ig[b] - Io[b]) <= allowed, (p, b)
        # (d)
        if p in pairs:
            tot = 0.0
            for y0 in range(0, ny, 64):
                blk = dense[0, :, y0:y0 + 64].to(torch.complex128)
                blk = blk - blk.mean(dim=0, keepdim=True)
                tot += float((blk.real ** 2 + blk.imag ** 2).sum())
            assert abs(float(simg[p].double().sum()) - F * tot) < TOL_I * F * tot, p
    out = torch.as_tensor(~A).cuda()
    for p in range(16):
        assert float(I[p][:, out].abs().max()) == 0.0, "I outside the band limit must be exactly zero"
    del V, ex, I, dense
    torch.cuda.empty_cache()


def test_c4_full_grid_streaming_bins(torch):
    """Config 4 geometry (48 600 atoms, 1024^2, 120 slices, 200 kV), 32 frames; path B (streaming per-bin DFT, two
    chunks) against the oracle and against path A."""
    import paper_2602_10064_b200 as ps
    from paper_2602_10064_b200.binding import TacawStream
    F = 32
    w = make_workload("c4_interface_1024", n_frames=F)
    ctx = make_ctx(w)
    pos = w.positions()
    V, sidx = ps.ps_build_slices(ctx, _t(torch, pos), _t(torch, w.Z), want_slice_idx=True)
    ex = ps.ps_multislice(ctx, w.kV, gpu_incident(ctx, w), V)
    for f in (5, 27):                                                     # V on 2 frames, from positions
        Vo, so = oracle_potential(w, pos[f], slices=(3, 60, 118))
        assert np.array_equal(sidx[f].cpu().numpy(), so)
        for s in (3, 60, 118):
            assert rel_l2(V[f, s].cpu().numpy(), Vo[s]) < TOL_V
    psi0_o = oracle_incident(w)[0]
    for f in (0, 5, 19, 31):                                              # ... exit waves on 4 (frame, probe) pairs
        eo = O.multislice(psi0_o, V[f].cpu().numpy().astype(np.float64), w.cell, w.kV)
        assert rel_l2(ex[0, f].cpu().numpy(), eo) < TOL_EXIT, f
    del V
    bins = np.arange(-8, 16, dtype=np.int32)
    ts = TacawStream(ctx, 1, F, w.dt_fs, bins)
    ts.add(ex[:, :20].contiguous(), 0)
    ts.add(ex[:, 20:].contiguous(), 20)
    IB = ts.finish()
    IA = ps.ps_tacaw(ctx, ex, w.dt_fs, bins)
    _check_norm(torch, ex, w)
    _check_tacaw_sample(torch, ps, ctx, w, ex, IB, bins, 2048, 41)
    _check_tacaw_sample(torch, ps, ctx, w, ex, IA, bins, 2048, 42)
    assert rel_l2(IB.cpu().numpy(), IA.cpu().numpy()) < TOL_I


def test_c4_streaming_loop_four_chunks(torch):
    """The loop bench.py --full-config c4 runs (build V of 64 frames -> multislice -> ps_tacaw_add, buffers reused), on
    256 frames = 4 chunks at config 4's own grid, slices, atoms and its 256 bins.  The exit-wave columns of 2048 seeded
    in-band pixels are kept from every chunk; path B's I at those pixels must equal the oracle's mean-subtracted FFT of
    the columns, as a whole and bin by bin (same floor as test_c3_bench_shape); out-of-band pixels exactly zero."""
    import paper_2602_10064_b200 as ps
    from paper_2602_10064_b200.binding import TacawStream
    F, chunk = 256, 64
    w = make_workload("c4_interface_1024", n_frames=F)
    ctx = make_ctx(w)
    nx, ny, S = w.nx, w.ny, w.n_slices
    bins = np.arange(256, dtype=np.int32)
    A = O.aperture_mask(w.cell, nx, ny)
    iy, ix = np.nonzero(A)
    sel = np.random.default_rng(404).choice(iy.size, size=2048, replace=False)
    sy, sx = torch.as_tensor(iy[sel]).cuda(), torch.as_tensor(ix[sel]).cuda()
    Z_d = _t(torch, w.Z)
    V = torch.empty((chunk, S, ny, nx), dtype=torch.float32, device="cuda")
    ex = torch.empty((1, chunk, ny, nx), dtype=torch.complex64, device="cuda")
    psi0 = ps.ps_make_incident(ctx, w.kV)
    ts = TacawStream(ctx, 1, F, w.dt_fs, bins)
    cols = []
    for f0 in range(0, F, chunk):
        ps.ps_build_slices(ctx, _t(torch, w.positions(f0, f0 + chunk)), Z_d, d_V=V)
        ps.ps_multislice(ctx, w.kV, psi0, V, d_exit=ex)
        ts.add(ex, f0)
        cols.append(ex[0][:, sy, sx].cpu().numpy())
    I = ts.finish()
    ctx.check_async()
    cols = np.concatenate(cols).astype(np.complex128)                       # [256][2048]
    Io = O.tacaw_intensity(cols, bins)
    Ig = I[0][:, sy, sx].cpu().numpy().astype(np.float64)
    nz = np.asarray(bins) != 0                                              # bin 0 (the mean term) is defined as zero
    assert rel_l2(Ig[nz], Io[nz]) < TOL_I
    assert not Ig[~nz].any()
    eps32 = float(np.finfo(np.float32).eps)
    floor = eps32 * np.log2(F) * np.sqrt(max(Io[nz].mean(axis=1).max(), float(np.mean(np.abs(cols.sum(axis=0)) ** 2))))
    for b in np.nonzero(nz)[0]:
        allowed = TOL_I * np.linalg.norm(Io[b]) + np.linalg.norm(2.0 * np.sqrt(Io[b]) * floor + floor ** 2)
        assert np.linalg.norm(Ig[b] - Io[b]) <= allowed, b
    out = torch.as_tensor(~A).cuda()
    assert float(I[0][:, out].abs().max()) == 0.0


@pytest.mark.parametrize("grid", [1024, 2048])
def test_c5_large_grids_tilts(torch, grid):
    """Config 5 geometry (40 960 atoms, 80 slices, 8 tilts) at its two largest grids (8 frames at 1024^2, 2 at
    2048^2): the longest FFTs the library instantiates, on potentials built from atoms."""
    import paper_2602_10064_b200 as ps
    F = 32
    w = make_workload("c5_al_sweep", n_frames=F, grid=grid)
    ctx = make_ctx(w)
    nf = 8 if grid == 1024 else 2                                             # frames through the slice loop
    pos = w.positions(0, nf)
    V, sidx = ps.ps_build_slices(ctx, _t(torch, pos), _t(torch, w.Z), want_slice_idx=True)
    ex = ps.ps_multislice(ctx, w.kV, gpu_incident(ctx, w), V)
    v_slices = (0, 40) if grid == 1024 else (40,)                         # the 2048^2 oracle potential is ~15 s per slice
    for f in (0, nf - 1):                                                 # V on 2 frames, from positions
        Vo, so = oracle_potential(w, pos[f], slices=v_slices)
        assert np.array_equal(sidx[f].cpu().numpy(), so)
        for s in v_slices:
            assert rel_l2(V[f, s].cpu().numpy(), Vo[s]) < TOL_V
    po = oracle_incident(w)
    # exit waves of 4 (tilt, frame) pairs at 1024^2; 1 at 2048^2, where one oracle slice loop is half a minute of host FFTs
    pairs = ((7, nf - 1), (0, 0), (3, 4), (5, 2)) if grid == 1024 else ((3, 1),)
    for p, f in pairs:
        eo = O.multislice(po[p], V[f].cpu().numpy().astype(np.float64), w.cell, w.kV)
        assert rel_l2(ex[p, f].cpu().numpy(), eo) < TOL_EXIT, (p, f)
    _check_norm(torch, ex, w)
