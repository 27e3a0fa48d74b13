"""Pins P1-P14 for the float64 oracle; CPU only.

Each pin ties `oracle/tacaw_oracle.py` to something other than itself: numbers the paper prints
(tests/golden/, cited), textbook constants, closed forms (Gaussian atom, Jacobi-Anger, free-space
propagation), invariants (Parseval, norm, translation, selection rule) or brute force with explicit
DFT sums on tiny inputs.  A dropped term, a wrong sign/index or a transposed operand in the oracle
fails at least one of them.
"""
import numpy as np
import pytest
from scipy.special import jv

from oracle import tacaw_oracle as O

RNG = np.random.default_rng(12345)


def rel_l2(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel())


# ----------------------------------------------------------------------------- P1
def test_P1_grids_match_paper_worked_example(golden):
    g = golden("paper_resolution_example.txt")
    L = g["supercell_reps"] * g["a_lattice_A"]
    assert abs(L - g["L_A"]) < 0.05
    nx = int(round(L / g["sampling_A"]))
    kx, ky = O.k_grids([L, L, 27.155], nx, nx)
    assert abs(kx[1] - kx[0] - 1.0 / L) < 1e-15                  # Eq. 4, no 2 pi
    assert round(kx[1], 3) == g["dk_invA"]
    assert abs(np.abs(kx).max() - g["k_max_invA"]) < 0.01        # k_max = 1/(2 sampling)
    kX = 1.0 / (2 * g["a_lattice_A"])
    assert round(kX, 3) == g["k_X_invA"]
    path = np.linspace(0, kX, 100)
    pix = O.dispersion_pixels([L, L, 1.0], nx, nx, path, np.zeros_like(path))
    assert abs(len(np.unique(pix)) - g["n_kpoints_gamma_X"]) <= 1   # "approximately 10"
    f = O.frequencies_THz(int(g["n_frames"]), g["dt_ps"] * 1e3)
    assert abs(f[1] - g["df_THz"]) < 1e-12                        # Eq. 5
    assert abs(np.abs(f).max() - g["f_max_THz"]) < 1e-9           # Eq. 6
    assert O.frequency_bin(15.0, int(g["n_frames"]), g["dt_ps"] * 1e3) == 30


def test_fft_index_order():
    assert list(O.fft_index(8)) == [0, 1, 2, 3, -4, -3, -2, -1]
    assert np.allclose(O.fft_index(16) / 16.0, np.fft.fftfreq(16))


# ----------------------------------------------------------------------------- P2
def test_P2_wavelength_sigma_textbook(golden):
    g = golden("electron_constants.txt")
    for kV in (60, 100, 200):
        assert abs(O.wavelength_A(kV) / g[f"lambda_{kV}kV_A"] - 1) < 2e-5
        assert abs(O.sigma_rad_per_VA(kV) / g[f"sigma_{kV}kV"] - 1) < 2e-6
    assert abs(O.C_POT / g["C_pot_VA2"] - 1) < 1e-7
    assert abs(O.MEV_PER_THZ - g["meV_per_THz"]) < 1e-12
    # non-relativistic limit: lambda -> h/sqrt(2 m E) = 12.2643/sqrt(V) Angstrom
    assert abs(O.wavelength_A(1e-3) * np.sqrt(1.0) / 12.2643 - 1) < 1e-4


# ----------------------------------------------------------------------------- a0 binning
def test_binning_edges_and_wrap():
    cell = np.array([10.0, 6.0, 8.0])
    S = 16                      # dz = 0.5 and z/Lz exactly representable at the boundaries
    z = np.array([0.0, 0.49999, 0.5, 7.99999, 8.0, -0.25, 16.25, 4.0], dtype=np.float32)
    pos = np.zeros((z.size, 3), dtype=np.float32); pos[:, 2] = z
    U = O.fixed_point(pos, cell)
    s = O.slice_index(U[:, 2], S)
    assert list(s) == [0, 0, 1, 15, 0, 15, 0, 8]
    assert U.max() < 2 ** 32
    # tiny negative coordinate: u rounds to 1.0 -> clamp to the last representable fraction
    pos = np.array([[-1e-30, 0, 0]], dtype=np.float32)
    assert O.fixed_point(pos, cell)[0, 0] == 2 ** 32 - 1


def test_binning_uniform_counts():
    cell = np.array([7.0, 9.0, 11.0]); S = 7
    pos = (RNG.uniform(-2, 3, (5000, 3)) * cell).astype(np.float32)
    U = O.fixed_point(pos, cell)
    s = O.slice_index(U[:, 2], S)
    assert s.min() >= 0 and s.max() <= S - 1
    zz = np.mod(pos[:, 2].astype(np.float64), cell[2])
    ref = np.minimum(np.floor(zz / (cell[2] / S)), S - 1).astype(int)
    assert (ref != s).mean() < 2e-3       # only atoms within rounding of a boundary may differ


# ----------------------------------------------------------------------------- P3 / P4
def _rand_coef(nl, ng, dmin=0.05):
    a = RNG.uniform(0.1, 1.0, nl); b = RNG.uniform(0.2, 8.0, nl)
    c = RNG.uniform(0.1, 1.5, ng); d = RNG.uniform(dmin, dmin + 3.0, ng)
    return np.concatenate([a, b, c, d])


def test_form_factor_definition():
    coef = np.array([0.3, 0.7, 2.0, 5.0, 1.1, 0.4, 0.5, 3.0])   # nl=2, ng=2
    q2 = np.array([0.0, 1.0, 4.0])
    want = [0.3 / (x + 2.0) + 0.7 / (x + 5.0) + 1.1 * np.exp(-0.5 * x) + 0.4 * np.exp(-3.0 * x) for x in q2]
    assert np.allclose(O.form_factor(q2, coef, 2, 2), want, rtol=1e-15)


def test_P3_potential_mean_is_C_sum_f0():
    cell = np.array([9.0, 7.0, 6.0]); nx, ny, S = 48, 40, 3
    coef = np.stack([_rand_coef(3, 3), _rand_coef(3, 3)])
    Na = 23
    pos = (RNG.uniform(0, 1, (Na, 3)) * cell).astype(np.float32)
    el = RNG.integers(0, 2, Na)
    V, s_idx = O.projected_potential(pos, el, coef, 3, 3, cell, nx, ny, S)
    f0 = np.array([(c[0:3] / c[3:6]).sum() + c[6:9].sum() for c in coef])
    for s in range(S):
        want = O.C_POT * f0[el[s_idx == s]].sum()
        assert abs(V[s].mean() * cell[0] * cell[1] - want) <= 1e-12 * max(1.0, abs(want))
    assert np.all(np.bincount(s_idx, minlength=S).sum() == Na)


def test_P4_isolated_gaussian_atom_closed_form():
    # V(r) = pi C sum_i (c_i/d_i) exp(-pi^2 |r-r0|^2 / d_i): 2-D Fourier transform of the Gaussian terms.
    cell = np.array([16.293, 13.0, 5.0]); nx, ny = 128, 96          # Lx != Ly, nx != ny: catches transposes
    c = np.array([0.8, 1.7]); d = np.array([3.0, 5.5])
    coef = np.concatenate([c, d])[None, :]
    r0 = np.array([5.137, 8.291])                                     # sub-pixel, asymmetric
    pos = np.array([[r0[0], r0[1], 2.5]], dtype=np.float32)
    V, _ = O.projected_potential(pos, np.array([0]), coef, 0, 2, cell, nx, ny, 1)
    x = np.arange(nx) * cell[0] / nx; y = np.arange(ny) * cell[1] / ny
    r0q = pos[0, :2].astype(np.float64)
    want = np.zeros((ny, nx))
    for ix in (-1, 0, 1):                                             # nearest periodic images
        for iy in (-1, 0, 1):
            r2 = (x[None, :] - r0q[0] - ix * cell[0]) ** 2 + (y[:, None] - r0q[1] - iy * cell[1]) ** 2
            want += np.pi * O.C_POT * sum(ci / di * np.exp(-np.pi ** 2 * r2 / di) for ci, di in zip(c, d))
    assert rel_l2(V[0], want) < 1e-8
    iy, ix = np.unravel_index(np.argmax(V[0]), V[0].shape)
    assert abs(x[ix] - r0[0]) < cell[0] / nx and abs(y[iy] - r0[1]) < cell[1] / ny


# ----------------------------------------------------------------------------- P5 / P6 / P10
def test_P5_free_space_plane_wave_and_probe():
    cell = np.array([12.0, 10.0, 8.0]); nx, ny, S = 64, 48, 4; kV = 100.0
    V = np.zeros((S, ny, nx))
    E = O.multislice(O.plane_wave(nx, ny), V, cell, kV)
    want = np.zeros((ny, nx), complex); want[0, 0] = np.sqrt(nx * ny)
    assert np.abs(E - want).max() < 1e-12
    psi0 = O.probe_wave(cell, nx, ny, kV, 30.0, 3.3, 7.1)
    assert abs(np.sum(np.abs(psi0) ** 2) - nx * ny) < 1e-9
    E = O.multislice(psi0, V, cell, kV)
    kx, ky = O.k_grids(cell, nx, ny)
    k2 = kx[None, :] ** 2 + ky[:, None] ** 2
    lam = O.wavelength_A(kV)
    want = np.fft.fft2(psi0) / np.sqrt(nx * ny) * np.exp(-1j * np.pi * lam * cell[2] * k2)
    assert rel_l2(E, want) < 1e-12
    # probe is centred where asked: |psi0|^2 peaks at (x0,y0)
    iy, ix = np.unravel_index(np.argmax(np.abs(psi0)), psi0.shape)
    assert abs(ix * cell[0] / nx - 3.3) <= cell[0] / nx and abs(iy * cell[1] / ny - 7.1) <= cell[1] / ny
    # support: lambda |k| <= alpha
    sup = np.abs(np.fft.fft2(psi0)) > 1e-9
    assert np.array_equal(sup, (lam * np.sqrt(k2) <= 30e-3) & O.aperture_mask(cell, nx, ny))


def test_P6_constant_potential_is_global_phase():
    cell = np.array([12.0, 10.0, 8.0]); nx, ny, S = 64, 48, 5; kV = 200.0
    psi0 = O.probe_wave(cell, nx, ny, kV, 20.0, 1.0, 2.0)
    V0 = 37.5
    E0 = O.multislice(psi0, np.zeros((S, ny, nx)), cell, kV)
    E1 = O.multislice(psi0, np.full((S, ny, nx), V0), cell, kV)
    assert rel_l2(E1, E0 * np.exp(1j * O.sigma_rad_per_VA(kV) * V0 * S)) < 1e-12


def test_P10_slice_composition_and_translation():
    cell = np.array([12.0, 10.0, 8.0]); nx, ny = 64, 64; kV = 100.0
    psi0 = O.probe_wave(cell, nx, ny, kV, 25.0, 4.0, 5.0)
    E2 = O.multislice(psi0, np.zeros((2, ny, nx)), cell, kV)
    E1 = O.multislice(psi0, np.zeros((1, ny, nx)), cell, kV)
    assert rel_l2(E2, E1) < 1e-12
    coef = _rand_coef(3, 3)[None]
    pos = (RNG.uniform(0, 1, (6, 3)) * cell).astype(np.float32)
    sx, sy = 5, 9
    shift = np.array([sx * cell[0] / nx, sy * cell[1] / ny, 0.0])
    posb = (pos.astype(np.float64) + shift).astype(np.float32)
    el = np.zeros(6, int)
    Va, _ = O.projected_potential(pos, el, coef, 3, 3, cell, nx, ny, 2)
    Vb, _ = O.projected_potential(posb, el, coef, 3, 3, cell, nx, ny, 2)
    pa = O.multislice(O.plane_wave(nx, ny), Va, cell, kV, return_real_space=True)
    pb = O.multislice(O.plane_wave(nx, ny), Vb, cell, kV, return_real_space=True)
    assert rel_l2(pb, np.roll(pa, (sy, sx), axis=(0, 1))) < 1e-5      # float32 position rounding only
    assert rel_l2(pb, pa) > 1e-2


# ----------------------------------------------------------------------------- P7 / P8 / P9
def test_P7_phase_grating_jacobi_anger():
    cell = np.array([12.0, 9.0, 3.0]); nx, ny = 96, 32; kV = 100.0
    g, V0, phi0 = 3, 900.0, 0.7
    x = np.arange(nx) * cell[0] / nx
    V = np.tile(V0 * np.cos(2 * np.pi * g * x / cell[0] + phi0)[None, None, :], (1, ny, 1))
    E = O.multislice(O.plane_wave(nx, ny), V, cell, kV)
    sig = O.sigma_rad_per_VA(kV); lam = O.wavelength_A(kV)
    want = np.zeros((ny, nx), complex)
    A = O.aperture_mask(cell, nx, ny)
    for n in range(-10, 11):
        m = n * g
        if abs(m) >= nx // 2:
            continue
        coeff = (1j ** n) * jv(n, sig * V0) * np.exp(1j * n * phi0)
        want[0, m % nx] = np.sqrt(nx * ny) * coeff * np.exp(-1j * np.pi * lam * cell[2] * (m / cell[0]) ** 2) * A[0, m % nx]
    assert sig * V0 > 0.5                                              # strong phase object
    assert np.abs(E - want).max() < 1e-9 * np.sqrt(nx * ny)


def _small_system(S=3, nx=48, ny=40, Na=14, seed=3):
    rng = np.random.default_rng(seed)
    cell = np.array([9.5, 8.0, 6.0])
    coef = np.stack([_rand_coef(3, 3), _rand_coef(3, 3)])
    pos = (rng.uniform(0, 1, (Na, 3)) * cell).astype(np.float32)
    el = rng.integers(0, 2, Na)
    return cell, coef, pos, el, S, nx, ny


def test_P8_norm_nonincreasing():
    cell, coef, pos, el, S, nx, ny = _small_system()
    V, _ = O.projected_potential(pos, el, coef, 3, 3, cell, nx, ny, S)
    norms = [nx * ny]
    for s in range(1, S + 1):
        E = O.multislice(O.plane_wave(nx, ny), V[:s], np.array([cell[0], cell[1], cell[2] * s / S]), 100.0)
        norms.append(np.sum(np.abs(E) ** 2))
    assert all(norms[i + 1] <= norms[i] * (1 + 1e-12) for i in range(S))
    assert norms[-1] > 0.5 * nx * ny
    # weak, smooth potential: nothing reaches the band edge -> norm conserved
    E = O.multislice(O.plane_wave(nx, ny), 1e-3 * V, cell, 100.0)
    assert abs(np.sum(np.abs(E) ** 2) / (nx * ny) - 1) < 1e-6


def test_P9_last_propagator_does_not_change_intensity():
    cell, coef, pos, el, S, nx, ny = _small_system()
    F = 6
    traj = pos[None] + RNG.normal(0, 0.05, (F,) + pos.shape).astype(np.float32)
    A = O.aperture_mask(cell, nx, ny)
    ea, eb = [], []
    for f in range(F):
        V, _ = O.projected_potential(traj[f], el, coef, 3, 3, cell, nx, ny, S)
        ea.append(O.multislice(O.plane_wave(nx, ny), V, cell, 100.0))
        eb.append(O.multislice(O.plane_wave(nx, ny), V, cell, 100.0, last_propagator=False))
    Ia = O.tacaw_intensity(np.array(ea)); Ib = O.tacaw_intensity(np.array(eb))
    assert rel_l2(Ia[:, A], Ib[:, A]) < 1e-10
    assert np.abs(Ia[:, ~A]).max() < 1e-20 * Ia.max()          # band-limited exit wave


# ----------------------------------------------------------------------------- P11
def test_P11_parseval_dc_and_wiener_khinchin():
    F = 32
    psi = RNG.normal(size=(F, 5, 7)) + 1j * RNG.normal(size=(F, 5, 7)) + 10.0
    I = O.tacaw_intensity(psi)
    d = psi - psi.mean(axis=0)
    assert np.allclose(I.sum(axis=0), F * (np.abs(d) ** 2).sum(axis=0), rtol=1e-12)
    assert np.abs(I[0]).max() < 1e-20
    # FFT of the circular time-autocorrelation of (psi - mean) equals I  ("Time Autocorrelation ...")
    ac = np.zeros_like(d)
    for tau in range(F):
        ac[tau] = (np.conj(d) * np.roll(d, -tau, axis=0)).sum(axis=0)
    assert np.allclose(np.fft.fft(ac, axis=0).real, I, rtol=1e-10, atol=1e-10)
    # bin list mode, signed bins
    assert np.array_equal(O.tacaw_intensity(psi, [1, -1, 3]), I[[1, F - 1, 3]])
    # a pure tone exp(+2 pi i n0 j/F) lands in bin +n0 with |.|^2 = F^2
    n0 = 5
    tone = np.exp(2j * np.pi * n0 * np.arange(F) / F)[:, None, None] * np.ones((1, 2, 2))
    It = O.tacaw_intensity(tone)
    assert np.allclose(It[n0], F * F) and np.abs(np.delete(It, n0, axis=0)).max() < 1e-18


# ----------------------------------------------------------------------------- P12 / P13
def _single_mode_run(ff_scale, amp, S, F=16, n0=3, q0=(1, 0), nlat=4, nx=32, ny=32):
    a_l = 3.0
    cell = np.array([nlat * a_l, nlat * a_l, 4.0])
    ii, jj = np.meshgrid(np.arange(nlat), np.arange(nlat), indexing="ij")
    R = np.stack([ii.ravel() * a_l + 0.4, jj.ravel() * a_l + 0.9, np.full(ii.size, 1.0)], axis=1)
    if S > 1:                                     # a second plane of atoms in another slice
        R = np.concatenate([R, R + np.array([a_l / 2, a_l / 3, 2.2])])
    e = np.array([0.6, 0.8, 0.0])
    qvec = np.array([q0[0] / cell[0], q0[1] / cell[1], 0.0])
    coef = np.array([[0.9, 0.4, 1.2, 0.3]]) * np.array([ff_scale, ff_scale, 1, 1])   # (0,2): c1,c2,d1,d2
    t = np.arange(F)
    waves = []
    for j in t:
        u = amp * e[None, :] * np.cos(2 * np.pi * (R @ qvec - n0 * j / F) + 0.3)[:, None]
        pos = (R + u).astype(np.float32)
        V, _ = O.projected_potential(pos, np.zeros(len(R), int), coef, 0, 2, cell, nx, ny, S)
        waves.append(O.multislice(O.plane_wave(nx, ny), V, cell, 100.0))
    return O.tacaw_intensity(np.array(waves)), cell, e, coef, len(R), nlat


def test_P12_single_mode_selection_rule():
    F, n0, nx, ny = 16, 3, 32, 32
    I, cell, e, coef, Na, nlat = _single_mode_run(ff_scale=1.0, amp=0.08, S=2, F=F, n0=n0, nx=nx, ny=ny)
    mx = O.fft_index(nx)[None, None, :]; my = O.fft_index(ny)[None, :, None]
    nn = np.arange(F)[:, None, None]
    # allowed: n = m*n0 (mod F) and (kx + m q0x, ky + m q0y) in G (multiples of nlat); gcd(n0,F)=1 -> m unique mod F
    minv = pow(n0, -1, F)
    m = (nn * minv) % F
    allowed = ((mx + m * 1) % nlat == 0) & ((my + m * 0) % nlat == 0)
    total = I.sum()
    assert I[~np.broadcast_to(allowed, I.shape)].sum() / total < 1e-9     # float32 position rounding only
    # +f0 <-> G - q0 ; -f0 <-> G + q0  (sign convention of time vs space transforms)
    assert I[n0, 0, (-1) % nx] > 1e3 * I[n0, 0, 1]
    assert I[F - n0, 0, 1] > 1e3 * I[F - n0, 0, (-1) % nx]
    assert I[n0].sum() / total > 0.05


def test_P13_weak_phase_single_mode_amplitude():
    F, n0, nx, ny = 16, 3, 32, 32
    amp = 4e-3          # big enough for float32 positions, small enough for O((2 pi k a)^2)
    I, cell, e, coef, Na, nlat = _single_mode_run(ff_scale=1e-4, amp=amp, S=1, F=F, n0=n0, nx=nx, ny=ny)
    sig = O.sigma_rad_per_VA(100.0)
    A = O.aperture_mask(cell, nx, ny)
    kx, ky = O.k_grids(cell, nx, ny)
    checked = 0
    for gx in (-1, 0, 1):
        for gy in (-1, 0, 1):
            ix = (gx * nlat - 1) % nx; iy = (gy * nlat) % ny              # k = G - q0 at bin +n0
            if not A[iy, ix]:
                continue
            k = np.array([kx[ix], ky[iy]])
            fk = O.form_factor(np.array([k @ k]), coef[0], 0, 2)[0]
            want = sig * O.C_POT * np.sqrt(nx * ny) / (cell[0] * cell[1]) * np.pi * abs(k @ e[:2]) * amp * fk * Na * F
            assert abs(np.sqrt(I[n0, iy, ix]) / want - 1) < 2e-3
            checked += 1
    assert checked >= 5
    # zero first-order weight where k is perpendicular to the polarisation: e=(0.6,0.8) -> k=(4,-3)/L ... use ratio
    ix = (4 - 1) % nx   # k = (3,?) not perpendicular; instead verify proportionality to |k.e|^2 between two spots
    r = I[n0, (1 * nlat) % ny, (-1) % nx] / I[n0, (-1 * nlat) % ny, (-1) % nx]
    k1 = np.array([kx[(-1) % nx], ky[nlat % ny]]); k2 = np.array([kx[(-1) % nx], ky[(-nlat) % ny]])
    f1 = O.form_factor(np.array([k1 @ k1]), coef[0], 0, 2)[0]; f2 = O.form_factor(np.array([k2 @ k2]), coef[0], 0, 2)[0]
    assert abs(r / (((k1 @ e[:2]) * f1) ** 2 / ((k2 @ e[:2]) * f2) ** 2) - 1) < 5e-3


# ----------------------------------------------------------------------------- P14 brute force
def test_P14_brute_force_explicit_dft():
    nx = ny = 8; S = 2; F = 4; kV = 100.0
    cell = np.array([4.0, 5.0, 3.0])
    coef = np.array([[0.5, 0.3, 1.0, 2.0, 0.7, 0.2, 0.4, 0.1],
                     [0.2, 0.6, 0.8, 3.0, 0.3, 0.9, 0.2, 0.6]])              # nl=2, ng=2
    el = np.array([0, 1, 0])
    base = np.array([[0.7, 1.1, 0.4], [2.9, 4.2, 2.0], [1.6, 0.3, 2.9]])
    traj = (base[None] + RNG.normal(0, 0.1, (F, 3, 3))).astype(np.float32)
    I_or, exit_or = O.run_path(traj, el, coef, 2, 2, cell, nx, ny, S, kV, [O.plane_wave(nx, ny)])

    # --- everything again with explicit sums, no FFT routine, no oracle helper
    def sidx(n):
        return np.array([i if i < n // 2 else i - n for i in range(n)])
    mxs, mys = sidx(nx), sidx(ny)
    lam = 12.398419843 / np.sqrt(kV * (2 * 510.99895 + kV))
    sig = 2 * np.pi / (lam * kV * 1e3) * (510.99895 + kV) / (2 * 510.99895 + kV)
    Cp = 2 * np.pi * 0.529177211 * 14.3996455
    kc2 = ((2 / 3) * min(nx / (2 * cell[0]), ny / (2 * cell[1]))) ** 2
    dz = cell[2] / S
    Wx = np.exp(-2j * np.pi * np.outer(mxs, np.arange(nx)) / nx)           # forward DFT matrix rows = k
    Wy = np.exp(-2j * np.pi * np.outer(mys, np.arange(ny)) / ny)
    exits = np.zeros((F, ny, nx), complex)
    for f in range(F):
        psi = np.ones((ny, nx), complex)
        frac = traj[f].astype(np.float64) / cell
        frac -= np.floor(frac)
        for s in range(S):
            Vr = np.zeros((ny, nx))
            for iy in range(ny):
                for ix in range(nx):
                    acc = 0.0
                    for a_y, my in enumerate(mys):
                        for a_x, mx in enumerate(mxs):
                            kx, ky = mx / cell[0], my / cell[1]
                            q2 = kx * kx + ky * ky
                            if q2 > kc2:
                                continue
                            for j in range(3):
                                if int(np.floor(frac[j, 2] * S)) != s:
                                    continue
                                c = coef[el[j]]
                                fq = c[0] / (q2 + c[2]) + c[1] / (q2 + c[3]) + c[4] * np.exp(-c[6] * q2) + c[5] * np.exp(-c[7] * q2)
                                ph = -2 * np.pi * (kx * frac[j, 0] * cell[0] + ky * frac[j, 1] * cell[1]) \
                                     + 2 * np.pi * (mx * ix / nx + my * iy / ny)
                                acc += fq * np.cos(ph)                       # real part of the inverse sum
                    Vr[iy, ix] = Cp / (cell[0] * cell[1]) * acc
            psi = psi * np.exp(1j * sig * Vr)
            Pk = np.zeros((ny, nx), complex)
            for a_y, my in enumerate(mys):
                for a_x, mx in enumerate(mxs):
                    q2 = (mx / cell[0]) ** 2 + (my / cell[1]) ** 2
                    if q2 <= kc2:
                        Pk[a_y, a_x] = np.exp(-1j * np.pi * lam * dz * q2)
            Psi = Wy @ psi @ Wx.T
            psi = (np.conj(Wy).T @ (Pk * Psi) @ np.conj(Wx)) / (nx * ny)
        exits[f] = (Wy @ psi @ Wx.T) / np.sqrt(nx * ny)
    assert rel_l2(exit_or[0], exits) < 1e-7                                # 2^-32 position quantisation only
    d = exits - exits.mean(axis=0)
    Wt = np.exp(-2j * np.pi * np.outer(np.arange(F), np.arange(F)) / F)
    I_bf = np.abs(np.tensordot(Wt, d, axes=(1, 0))) ** 2
    assert rel_l2(I_or[0], I_bf) < 1e-6


# ----------------------------------------------------------------------------- a8 reductions, by loops
def test_reductions_brute_force():
    P, nb, ny, nx = 2, 5, 12, 16
    cell = np.array([8.0, 6.0, 1.0])
    I = RNG.uniform(0, 1, (P, nb, ny, nx))
    mxs, mys = O.fft_index(nx), O.fft_index(ny)
    assert np.allclose(O.sdp(I, 1, 3), sum(I[p, n] for p in range(P) for n in (1, 2, 3)))
    k_in, k_out = 0.3, 0.9
    si = np.zeros((P, nb))
    for iy in range(ny):
        for ix in range(nx):
            k = np.hypot(mxs[ix] / cell[0], mys[iy] / cell[1])
            if k_in <= k < k_out:
                si += I[:, :, iy, ix]
    assert np.allclose(O.spectrum_image(I, cell, k_in, k_out), si)
    kxp = np.array([0.0, 0.124, 0.126, -0.13, 0.99]); kyp = np.array([0.0, 0.0, 0.17, -0.3, 0.5])
    out, pix = O.dispersion(I, cell, kxp, kyp)
    for i in range(len(kxp)):
        ix = int(np.floor(kxp[i] * cell[0] + 0.5)) % nx; iy = int(np.floor(kyp[i] * cell[1] + 0.5)) % ny
        assert pix[i] == iy * nx + ix
        assert np.allclose(out[:, i], I[:, :, iy, ix].sum(axis=0))
    assert pix.dtype == np.int32
    dq, nq = 0.2, 4
    out, idx = O.qbin(I, cell, dq, nq)
    want = np.zeros((nb, nq))
    for iy in range(ny):
        for ix in range(nx):
            b = int(np.floor(np.hypot(mxs[ix] / cell[0], mys[iy] / cell[1]) / dq))
            assert idx[iy, ix] == (b if b < nq else -1)
            if b < nq:
                want[:, b] += I[:, :, iy, ix].sum(axis=0)
    assert np.allclose(out, want)


def test_aperture_mask_properties():
    cell = np.array([16.293, 16.293, 5.0])
    A = O.aperture_mask(cell, 128, 128)
    m = O.fft_index(128)
    r2 = m[None, :] ** 2 + m[:, None] ** 2
    assert np.array_equal(A, r2 <= (128 / 3) ** 2)                       # square grid: integer criterion
    assert abs(A.mean() - np.pi / 9) < 0.01
    assert A[0, 42] and not A[0, 43] and not A[64, 0]
    assert np.array_equal(A, A.T) and np.array_equal(A, np.roll(A[::-1, ::-1], (1, 1), (0, 1)))


# ----------------------------------------------------------------------------- HAADF / averaging
def test_haadf_closed_forms_and_brute_force():
    """Free space: the whole beam stays at k = 0, so an annulus sees nothing and a disc that holds k = 0 sees the
    whole incident intensity (fraction 1); a phase grating puts |J_n(sigma V0)|^2 on order n (Jacobi-Anger, P7);
    and on random waves the definition is a plain double loop."""
    cell = np.array([12.0, 9.0, 3.0]); nx, ny = 96, 32; kV = 100.0
    E0 = O.multislice(O.plane_wave(nx, ny), np.zeros((2, ny, nx)), cell, kV)[None, None]
    assert abs(O.haadf(E0, cell, 0.0, 0.05)[0] - 1.0) < 1e-12
    assert O.haadf(E0, cell, 0.05, 0.0)[0] < 1e-24
    g, V0 = 3, 900.0
    x = np.arange(nx) * cell[0] / nx
    V = np.tile(V0 * np.cos(2 * np.pi * g * x / cell[0])[None, None, :], (1, ny, 1))
    E = O.multislice(O.plane_wave(nx, ny), V, cell, kV)[None, None]
    sig = O.sigma_rad_per_VA(kV)
    k1 = g / cell[0]                                                    # first diffraction order at |k| = g/Lx
    got = O.haadf(E, cell, 0.5 * k1, 1.5 * k1)[0]
    assert abs(got - 2.0 * jv(1, sig * V0) ** 2) < 1e-10                # orders +1 and -1
    rng = np.random.default_rng(8)
    W = rng.normal(size=(2, 3, 6, 8)) + 1j * rng.normal(size=(2, 3, 6, 8))
    c2 = np.array([4.0, 3.0, 1.0]); kin, kout = 0.3, 0.9
    want = np.zeros(2)
    for p in range(2):
        for f in range(3):
            for iy in range(6):
                for ix in range(8):
                    kx = (ix if ix < 4 else ix - 8) / c2[0]; ky = (iy if iy < 3 else iy - 6) / c2[1]
                    if kin <= np.hypot(kx, ky) < kout:
                        want[p] += abs(W[p, f, iy, ix]) ** 2 / 3.0 / 48.0
    assert np.allclose(O.haadf(W, c2, kin, kout), want, rtol=1e-13)


def test_accumulate_intensity_running_mean():
    rng = np.random.default_rng(9)
    Is = rng.uniform(size=(5, 2, 3, 4, 4))
    acc = np.zeros_like(Is[0])
    for n, I in enumerate(Is, start=1):
        acc = O.accumulate_intensity(acc, I, (n - 1) / n, 1.0 / n)
    assert np.allclose(acc, Is.mean(axis=0), rtol=1e-13)


# ----------------------------------------------------------------------------- aberrations
def test_aberration_function_against_propagator_and_textbook():
    """(i) pure C10: exp(-i chi) = exp(-i pi lambda C10 k^2) is the free-space propagator over the distance C10, so the
    defocused probe equals the focused probe sent through one vacuum slice of that thickness (ties sign and factor
    to the propagator pinned by P5/P7); (ii) C10 + C30 against Scherzer's form pi lambda k^2 (Cs lambda^2 k^2/2 - df)
    at a hand-picked k; (iii) rotating the astigmatism axis by 90 degrees flips its sign, coma by 180 degrees;
    (iv) a pure phase: the probe keeps its norm."""
    cell = np.array([14.0, 11.0, 5.0]); nx, ny = 64, 48; kV = 100.0
    lam = O.wavelength_A(kV)
    z = np.zeros(8)
    c = z.copy(); c[0] = 37.5                                          # C10 = 37.5 A
    p_ab = O.probe_wave(cell, nx, ny, kV, 25.0, 3.0, 4.0, aberrations=c)
    p0 = O.probe_wave(cell, nx, ny, kV, 25.0, 3.0, 4.0)
    cell_dz = np.array([cell[0], cell[1], 37.5])
    via_prop = O.multislice(p0, np.zeros((1, ny, nx)), cell_dz, kV, return_real_space=True)
    assert rel_l2(p_ab, via_prop) < 1e-12
    c = z.copy(); c[0] = -120.0; c[7] = 1.3e7                          # defocus 120 A, Cs = 1.3 mm
    chi = O.aberration_function(cell, nx, ny, kV, c)
    kx, ky = O.k_grids(cell, nx, ny)
    k2 = kx[5] ** 2 + ky[3] ** 2
    assert abs(chi[3, 5] - np.pi * lam * k2 * (0.5 * 1.3e7 * lam ** 2 * k2 - 120.0)) < 1e-9 * abs(chi[3, 5])
    a = z.copy(); a[1] = 50.0; a[2] = 0.3
    b = z.copy(); b[1] = -50.0; b[2] = 0.3 + np.pi / 2
    assert np.allclose(O.aberration_function(cell, nx, ny, kV, a), O.aberration_function(cell, nx, ny, kV, b), atol=1e-9)
    a = z.copy(); a[3] = 900.0; a[4] = 0.2
    b = z.copy(); b[3] = -900.0; b[4] = 0.2 + np.pi
    assert np.allclose(O.aberration_function(cell, nx, ny, kV, a), O.aberration_function(cell, nx, ny, kV, b), atol=1e-9)
    full = np.array([30.0, 20.0, 0.4, 500.0, 1.0, 300.0, -0.7, 2.0e5])
    p = O.probe_wave(cell, nx, ny, kV, 25.0, 3.0, 4.0, aberrations=full)
    assert abs(np.sum(np.abs(p) ** 2) - nx * ny) < 1e-9 * nx * ny
    W = RNG.normal(size=(2, ny, nx)) + 1j * RNG.normal(size=(2, ny, nx))
    assert np.allclose(np.abs(O.apply_aberrations(W, cell, kV, full)), np.abs(W), rtol=1e-12)


def test_apply_aberrations_sign_tied_to_propagator_and_probe_formation():
    """PAPER.md:143 (§4 "applied either during probe formation or post-hoc to stored wavefunctions"): the post-hoc route
    must carry the same sign as the other two pinned objects.  (i) pure C10 = 37.5 A applied post-hoc to the k-space of
    the focused probe equals that probe sent through 37.5 A of vacuum by the propagator (pinned by P5/P7: exp(-i pi
    lambda dz k^2)) — the probe is band-limited, so the propagator's aperture changes nothing; (ii) for a full set of
    coefficients, post-hoc application to the unaberrated probe's k-space equals the k-space of the probe formed with
    those aberrations.  exp(+i chi) in apply_aberrations fails both."""
    cell = np.array([14.0, 11.0, 5.0]); nx, ny = 64, 48; kV = 100.0
    p0 = O.probe_wave(cell, nx, ny, kV, 25.0, 3.0, 4.0)
    c = np.zeros(8); c[0] = 37.5
    post_hoc = np.fft.ifft2(O.apply_aberrations(np.fft.fft2(p0), cell, kV, c))
    via_prop = O.multislice(p0, np.zeros((1, ny, nx)), np.array([cell[0], cell[1], 37.5]), kV, return_real_space=True)
    assert rel_l2(post_hoc, via_prop) < 1e-12
    wrong_sign = np.fft.ifft2(np.fft.fft2(p0) * np.exp(+1j * O.aberration_function(cell, nx, ny, kV, c)))
    assert rel_l2(wrong_sign, via_prop) > 0.1                         # the check can tell the two signs apart
    full = np.array([30.0, 20.0, 0.4, 500.0, 1.0, 300.0, -0.7, 2.0e5])
    formed = O.probe_wave(cell, nx, ny, kV, 25.0, 3.0, 4.0, aberrations=full)
    assert rel_l2(O.apply_aberrations(np.fft.fft2(p0), cell, kV, full), np.fft.fft2(formed)) < 1e-12
    stack = np.stack([np.fft.fft2(p0), 2.0 * np.fft.fft2(p0)])        # leading axes are carried along
    assert rel_l2(O.apply_aberrations(stack, cell, kV, full)[1], 2.0 * np.fft.fft2(formed)) < 1e-12


def test_aberration_function_hand_evaluated_C12_C21_C23():
    """Pins the 1/2, 1/3 prefactors and the cos 2(phi-phi12), cos(phi-phi21), cos 3(phi-phi23) factors of reading A24
    ("standard aberration function supporting defocus, astigmatism, coma, spherical aberration"): chi is
    hand-evaluated from the Krivanek polynomial chi = (2 pi/lambda) sum_{n,m} C_nm theta^(n+1)/(n+1) cos m(phi-phi_nm)
    at explicit grid points of a 10 x 10 A cell (k = m/10 1/A), with theta = lambda |k| and phi worked out by hand:
        lambda(100 kV) = 0.037014 A (textbook value, tests/golden/electron_constants.txt)
        (kx, ky) = (0, 0.4):     |k| = 0.4,          theta = 0.0148056,   phi = 90 deg
        (kx, ky) = (-0.2, 0):    |k| = 0.2,          theta = 0.0074028,   phi = 180 deg
        (kx, ky) = (0.3, 0.3):   |k| = 0.424264069,  theta = 0.0157037102, phi = 45 deg
        (kx, ky) = (-0.3, 0.3):  same |k|,                                phi = 135 deg
    A wrong prefactor (1/2 <-> 1/3), a wrong power of theta or a wrong angular multiplicity fails one of the lines."""
    cell = np.array([10.0, 10.0, 5.0]); nx = ny = 32; kV = 100.0
    lam = 0.037014
    two_pi_over_lam = 2.0 * np.pi / lam
    z = np.zeros(8)

    def chi_at(coef, m, n):                                            # chi[iy][ix] at kx = m/10, ky = n/10
        return O.aberration_function(cell, nx, ny, kV, coef)[n % ny, m % nx]

    def close(got, want):
        return abs(got - want) <= 1e-4 * abs(want) + 1e-12

    # ---- pure C12 = 50 A, phi12 = 0.3 rad:  chi = (2 pi/lam) * 50 * theta^2/2 * cos 2(phi - 0.3)
    c = z.copy(); c[1] = 50.0; c[2] = 0.3
    # phi = 90 deg: cos(pi - 0.6) = -cos 0.6 = -0.8253356149
    assert close(chi_at(c, 0, 4), two_pi_over_lam * 50.0 * 0.0148056 ** 2 / 2.0 * (-0.8253356149))
    # phi = 180 deg: cos(2 pi - 0.6) = +0.8253356149
    assert close(chi_at(c, -2, 0), two_pi_over_lam * 50.0 * 0.0074028 ** 2 / 2.0 * 0.8253356149)
    # phi = 45 deg: cos(pi/2 - 0.6) = sin 0.6 = 0.5646424734  (a cos(phi - phi12) would give 0.8816)
    assert close(chi_at(c, 3, 3), two_pi_over_lam * 50.0 * 0.0157037102 ** 2 / 2.0 * 0.5646424734)
    # ---- pure C21 = 900 A, phi21 = 0.2 rad:  chi = (2 pi/lam) * 900 * theta^3/3 * cos(phi - 0.2)
    c = z.copy(); c[3] = 900.0; c[4] = 0.2
    # phi = 180 deg: cos(pi - 0.2) = -0.9800665778
    assert close(chi_at(c, -2, 0), two_pi_over_lam * 900.0 * 0.0074028 ** 3 / 3.0 * (-0.9800665778))
    # phi = 90 deg: cos(pi/2 - 0.2) = sin 0.2 = 0.1986693308
    assert close(chi_at(c, 0, 4), two_pi_over_lam * 900.0 * 0.0148056 ** 3 / 3.0 * 0.1986693308)
    # ---- pure C23 = 350 A, phi23 = 0:  chi = (2 pi/lam) * 350 * theta^3/3 * cos 3 phi
    c = z.copy(); c[5] = 350.0
    # phi = 45 deg: cos 135 deg = -0.7071067812;  phi = 135 deg: cos 405 deg = +0.7071067812 (cos phi would flip both signs)
    assert close(chi_at(c, 3, 3), two_pi_over_lam * 350.0 * 0.0157037102 ** 3 / 3.0 * (-0.7071067812))
    assert close(chi_at(c, -3, 3), two_pi_over_lam * 350.0 * 0.0157037102 ** 3 / 3.0 * 0.7071067812)
    # phi = 180 deg: cos 540 deg = -1;  phi = 90 deg: cos 270 deg = 0
    assert close(chi_at(c, -2, 0), two_pi_over_lam * 350.0 * 0.0074028 ** 3 / 3.0 * (-1.0))
    assert abs(chi_at(c, 0, 4)) < 1e-9
    # ---- with phi23 = -0.7: phi = 90 deg -> cos(3 pi/2 + 2.1) = sin 2.1 = 0.8632093666
    c[6] = -0.7
    assert close(chi_at(c, 0, 4), two_pi_over_lam * 350.0 * 0.0148056 ** 3 / 3.0 * 0.8632093666)
    # ---- the terms add: everything on at once equals the sum of the single-term values at one point
    full = np.array([30.0, 50.0, 0.3, 900.0, 0.2, 350.0, -0.7, 2.0e5])
    parts = 0.0
    for idx in ((0,), (1, 2), (3, 4), (5, 6), (7,)):
        c = z.copy(); c[list(idx)] = full[list(idx)]
        parts += chi_at(c, 3, 3)
    assert abs(chi_at(full, 3, 3) - parts) < 1e-9 * abs(parts)


# ----------------------------------------------------------------------------- tilted illumination (reading A18)
def test_tilted_plane_wave_is_one_reciprocal_grid_point():
    """A18 (BASELINE.json config 5; the paper has no tilt): psi0 = exp(2 pi i (mt x/Lx + nt y/Ly)) sits on ONE point of
    the reciprocal grid: fft2(psi0) is a single delta of height nx*ny at [nt mod ny][mt mod nx] (pins sign and axis
    order), and through V = 0 it stays that plane wave times exp(-i pi lambda Lz ((mt/Lx)^2 + (nt/Ly)^2)) — the
    free-space propagator of PAPER.md:79 (pinned by P5/P7) evaluated by hand on a NON-square cell:
        lambda(100 kV) = 0.037014 A, Lx = 9, Ly = 12, Lz = 30 A, (mt, nt) = (-3, 2):
        k^2 = (3/9)^2 + (2/12)^2 = 0.1111111111 + 0.0277777778 = 0.1388888889
        phase = -pi * 0.037014 * 30 * 0.1388888889 = -0.4845121 rad."""
    nx, ny = 24, 16
    for mt, nt in ((-3, 2), (5, 0), (0, -7), (1, 1)):
        psi = O.tilted_plane_wave(nx, ny, mt, nt)
        spec = np.fft.fft2(psi)
        want = np.zeros((ny, nx), complex); want[nt % ny, mt % nx] = nx * ny
        assert np.abs(spec - want).max() < 1e-9
    cell = np.array([9.0, 12.0, 30.0])
    psi = O.tilted_plane_wave(nx, ny, -3, 2)
    ex = O.multislice(psi, np.zeros((5, ny, nx)), cell, 100.0)           # five vacuum slices of 6 A
    want = np.zeros((ny, nx), complex)
    want[2, nx - 3] = np.sqrt(nx * ny) * np.exp(1j * (-0.4845121))        # unitary k-space exit wave (A13)
    assert np.abs(ex - want).max() < 2e-5 * np.sqrt(nx * ny)
    # a tilt outside the band limit is removed by the first propagator (kc = (2/3) * min(24/18, 16/24) = 0.4444)
    out = O.multislice(O.tilted_plane_wave(nx, ny, 0, -7), np.zeros((1, ny, nx)), cell, 100.0)   # |k| = 7/12 = 0.583
    assert np.abs(out).max() < 1e-12
