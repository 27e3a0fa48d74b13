"""TEST INFRASTRUCTURE — float64 CPU oracle of the TACAW hot path (PySlice, arxiv 2602.10064).

Plain, slow, obviously-correct NumPy restatement of what the path computes, written from
/root/reference/PAPER.md before any GPU code.  It shares NO code with the CUDA library
(`paper_2602_10064_b200/`): no common kernels, headers, helpers, tables or constant
generators; neither imports the other.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` legs may import it.

TACAW is *defined* by the paper's equations (no step approximates another), so every
function below is "the equation written out, float64, library FFT as one step":

  PAPER.md:73   (§2.1)  psi~(k,w) = F_t[psi(k,t) - <psi(k,t)>_t],  I(k,w) = |psi~|^2
  PAPER.md:79   (§2.2)  t(r) = exp(i sigma V(r)),  P(k) = exp(-i pi lambda dz |k|^2),
                        psi_exit = P_{N-1} t_N ... P_1 t_2 P_0 t_1 psi_probe
  PAPER.md:81   (§2.2)  f(q) = sum_i a_i/(q^2+b_i) + c_i exp(-d_i q^2);
                        V(k) = sum_j f_Zj(k) exp(-2 pi i k.r_j) over atoms in the slice; inverse FFT
  PAPER.md:89   (§2.2)  WFData indexed (probe, time, kx, ky)  -> exit wave kept in k-space
  PAPER.md:289-301 (Suppl. Eq. 4-6)  dk = 1/L, df = 1/(N dt), f_max = 1/(2 dt)
  PAPER.md:319  (Suppl. Eq. 7)  T(r) = exp[i sigma V(r)]

Where the paper is silent the readings A1-A22 of SURVEY.md §8(c) / DESIGN.md §3 apply; each is
named at the line that uses it.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): P1 grids (PAPER.md:402 numbers), P2 lambda/sigma
textbook values, P3 potential mean = C sum f(0), P4 isolated Gaussian atom closed form, P5 free
space, P6 constant potential, P7 Jacobi-Anger phase grating, P8 norm, P9 last propagator, P10 slice
composition + translation, P11 Parseval / Wiener-Khinchin, P12 single-mode selection rule,
P13 weak-phase single-mode amplitude, P14 brute-force DFT matrices.
Parity unpinned: physical spectra of real materials (no coefficient table, MD or reference
output exists in the container) — see DESIGN.md §3.
"""
from __future__ import annotations

import numpy as np

# ----------------------------------------------------------------------------- constants
# [derived; the paper prints none — SURVEY §8(c) "Constants"]
HC_KEV_A = 12.398419843          # h c            keV Angstrom
M0C2_KEV = 510.99895             # electron rest energy, keV
A0_A = 0.529177211               # Bohr radius, Angstrom
E2_VA = 14.3996455               # e^2/(4 pi eps0) = e * (V Angstrom)
C_POT = 2.0 * np.pi * A0_A * E2_VA   # = h^2/(2 pi m0 e) = 47.8776 V Angstrom^2   (A2)
MEV_PER_THZ = 4.135667697


def wavelength_A(kV: float) -> float:
    """Relativistic de Broglie wavelength (A4): lambda = hc / sqrt(E (2 m0c^2 + E))."""
    E = float(kV)
    return HC_KEV_A / np.sqrt(E * (2.0 * M0C2_KEV + E))


def sigma_rad_per_VA(kV: float) -> float:
    """Interaction parameter sigma = 2 pi m_e e lambda / h^2 with relativistic m_e
    (A3): (2 pi / (lambda E)) (m0c^2 + E)/(2 m0c^2 + E), E in volts -> rad/(V A)."""
    E = float(kV)
    return (2.0 * np.pi / (wavelength_A(kV) * E * 1.0e3)) * (M0C2_KEV + E) / (2.0 * M0C2_KEV + E)


# ----------------------------------------------------------------------------- grids
def fft_index(n: int) -> np.ndarray:
    """Signed FFT-order indices 0..n/2-1, -n/2..-1 (A1: numpy convention)."""
    m = np.arange(n, dtype=np.int64)
    m[m >= (n + 1) // 2] -= n
    return m


def k_grids(cell, nx: int, ny: int):
    """kx[nx], ky[ny] in 1/Angstrom, k = m/L without 2 pi (Eq. 4, pinned by PAPER.md:402)."""
    return fft_index(nx) / float(cell[0]), fft_index(ny) / float(cell[1])


def k_cut(cell, nx: int, ny: int) -> float:
    """Band limit (A10): 2/3 of the smaller Nyquist frequency."""
    return (2.0 / 3.0) * min(nx / (2.0 * float(cell[0])), ny / (2.0 * float(cell[1])))


def aperture_mask(cell, nx: int, ny: int) -> np.ndarray:
    """bool [ny][nx]: kx^2 + ky^2 <= k_c^2, inclusive (A10, A11)."""
    kx, ky = k_grids(cell, nx, ny)
    kc = k_cut(cell, nx, ny)
    return (kx[None, :] * kx[None, :] + ky[:, None] * ky[:, None]) <= kc * kc


def frequencies_THz(n_frames: int, dt_fs: float) -> np.ndarray:
    """f_n = n/(F dt), n signed in FFT order (Eq. 5; THz when dt in ps)."""
    return fft_index(n_frames) / (n_frames * dt_fs * 1.0e-3)


# ----------------------------------------------------------------------------- a0: ingest + slice binning
def fixed_point(pos32: np.ndarray, cell) -> np.ndarray:
    """uint64 array (values < 2^32) of fractional coordinates in units of 2^-32 of the cell.

    SURVEY §8(c) step 3: u = pos/L - floor(pos/L) in float64 (pos upcast from float32);
    U = floor(u 2^32) clamped to 2^32-1.  Periodic wrap (A8)."""
    L = np.asarray(cell, dtype=np.float64)
    q = pos32.astype(np.float64) / L
    u = q - np.floor(q)
    U = np.floor(u * 4294967296.0)
    U = np.minimum(U, 4294967295.0)
    return U.astype(np.uint64)


def slice_index(Uz: np.ndarray, n_slices: int) -> np.ndarray:
    """s = (U_z * S) >> 32 — half-open slices [s dz, (s+1) dz), beam along +z (A8). int32."""
    return ((Uz.astype(np.uint64) * np.uint64(n_slices)) >> np.uint64(32)).astype(np.int32)


# ----------------------------------------------------------------------------- a1: form factors
def form_factor(q2: np.ndarray, coef: np.ndarray, n_lorentz: int, n_gauss: int) -> np.ndarray:
    """f(q) = sum_i a_i/(q^2+b_i) + sum_i c_i exp(-d_i q^2)  (general (nl,ng) form, A5).
    coef row layout: a_1..a_nl, b_1..b_nl, c_1..c_ng, d_1..d_ng."""
    a = coef[0:n_lorentz]; b = coef[n_lorentz:2 * n_lorentz]
    c = coef[2 * n_lorentz:2 * n_lorentz + n_gauss]; d = coef[2 * n_lorentz + n_gauss:2 * n_lorentz + 2 * n_gauss]
    f = np.zeros_like(q2, dtype=np.float64)
    for i in range(n_lorentz):
        f = f + a[i] / (q2 + b[i])
    for i in range(n_gauss):
        f = f + c[i] * np.exp(-d[i] * q2)
    return f


# ----------------------------------------------------------------------------- a2+a3: projected potential
def projected_potential(pos32_frame: np.ndarray, elem_of_atom: np.ndarray, coef: np.ndarray,
                        n_lorentz: int, n_gauss: int, cell, nx: int, ny: int, n_slices: int,
                        band_limit: bool = True, atom_chunk: int = 64, slices=None):
    """V[s][ny][nx] in V*Angstrom for one frame, and the int32 slice index of every atom.

    SURVEY §8(c) steps 3-4 / PAPER.md:81:
      V_s(k) = A(k) sum_{j in s} f_Zj(|k|) exp(-2 pi i (kx x_j + ky y_j)),
      V_s(r) = (C/(Lx Ly)) Nx Ny real(ifft2(V_s(k)))      (A1, A2; numpy ifft2 carries 1/(NxNy)).
    x_j, y_j are the fixed-point-quantised positions U/2^32 * L.  `elem_of_atom[j]` indexes rows of
    `coef`.  `band_limit=False` drops A(k) (only used by pins that need the un-truncated sum).
    `slices` (an iterable of slice numbers) restricts the work to those slices, the others stay zero: the
    full-size parity tests sample slices this way (same arithmetic, fewer of them)."""
    L = np.asarray(cell, dtype=np.float64)
    U = fixed_point(pos32_frame, L)
    s_idx = slice_index(U[:, 2], n_slices)
    x = U[:, 0].astype(np.float64) / 4294967296.0 * L[0]
    y = U[:, 1].astype(np.float64) / 4294967296.0 * L[1]
    kx, ky = k_grids(L, nx, ny)
    A = aperture_mask(L, nx, ny) if band_limit else np.ones((ny, nx), dtype=bool)
    iy, ix = np.nonzero(A)
    kxa = kx[ix]; kya = ky[iy]
    q2 = kxa * kxa + kya * kya
    n_elem = coef.shape[0]
    f_tab = np.stack([form_factor(q2, coef[e], n_lorentz, n_gauss) for e in range(n_elem)])   # [nE][nk]
    V = np.zeros((n_slices, ny, nx), dtype=np.float64)
    for s in (range(n_slices) if slices is None else slices):
        Vk_a = np.zeros(kxa.shape[0], dtype=np.complex128)
        for e in range(n_elem):
            sel = np.nonzero((s_idx == s) & (elem_of_atom == e))[0]
            for c0 in range(0, sel.size, atom_chunk):
                j = sel[c0:c0 + atom_chunk]
                phase = -2.0 * np.pi * (x[j, None] * kxa[None, :] + y[j, None] * kya[None, :])
                Vk_a += f_tab[e] * np.exp(1j * phase).sum(axis=0)
        Vk = np.zeros((ny, nx), dtype=np.complex128)
        Vk[iy, ix] = Vk_a
        V[s] = (C_POT / (L[0] * L[1])) * nx * ny * np.real(np.fft.ifft2(Vk))
    return V, s_idx


# ----------------------------------------------------------------------------- a4: incident waves
def plane_wave(nx: int, ny: int) -> np.ndarray:
    """aperture=0 => parallel beam: psi0 = 1."""
    return np.ones((ny, nx), dtype=np.complex128)


def tilted_plane_wave(nx: int, ny: int, mt: int, nt: int) -> np.ndarray:
    """exp(2 pi i (mt x/Lx + nt y/Ly)) on a reciprocal-grid point (A18)."""
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    return np.exp(2j * np.pi * (mt * i / nx + nt * j / ny))


def aberration_function(cell, nx: int, ny: int, kV: float, coef) -> np.ndarray:
    """chi(k) in radians ("the standard aberration function supporting defocus, astigmatism, coma,
    spherical aberration"; the paper prints no formula: reading A24, Krivanek-style coefficients in Angstrom):
        chi = (2 pi / lambda) [ C10 th^2/2 + C12 th^2/2 cos(2(phi - phi12)) + C21 th^3/3 cos(phi - phi21)
                                + C23 th^3/3 cos(3(phi - phi23)) + C30 th^4/4 ],
    th = lambda |k|, phi = atan2(ky, kx); coef = (C10, C12, phi12, C21, phi21, C23, phi23, C30).
    With C10 = -defocus and C30 = Cs this is the textbook chi = pi lambda k^2 (Cs lambda^2 k^2 / 2 - defocus)."""
    C10, C12, p12, C21, p21, C23, p23, C30 = [float(x) for x in coef]
    kx, ky = k_grids(cell, nx, ny)
    KX, KY = np.meshgrid(kx, ky)
    lam = wavelength_A(kV)
    th = lam * np.sqrt(KX ** 2 + KY ** 2)
    phi = np.arctan2(KY, KX)
    return (2.0 * np.pi / lam) * (0.5 * C10 * th ** 2 + 0.5 * C12 * th ** 2 * np.cos(2.0 * (phi - p12))
                                  + C21 * th ** 3 / 3.0 * np.cos(phi - p21)
                                  + C23 * th ** 3 / 3.0 * np.cos(3.0 * (phi - p23)) + 0.25 * C30 * th ** 4)


def apply_aberrations(waves_k: np.ndarray, cell, kV: float, coef) -> np.ndarray:
    """Post-hoc aberrations on stored k-space waves [..., ny, nx]: Psi(k) <- Psi(k) exp(-i chi(k))."""
    ny, nx = waves_k.shape[-2:]
    return waves_k * np.exp(-1j * aberration_function(cell, nx, ny, kV, coef))


def probe_wave(cell, nx: int, ny: int, kV: float, semi_angle_mrad: float, x0: float, y0: float,
               aberrations=None) -> np.ndarray:
    """Focused probe (A12): Psi0(k) = [lambda |k| <= alpha] A(k) exp(-i chi(k)) exp(-2 pi i k.r_p),
    psi0 = ifft2(Psi0) scaled so sum |psi0|^2 = Nx Ny; chi = 0 without `aberrations`."""
    kx, ky = k_grids(cell, nx, ny)
    lam = wavelength_A(kV)
    k2 = kx[None, :] ** 2 + ky[:, None] ** 2
    Psi0 = ((lam * np.sqrt(k2) <= semi_angle_mrad * 1.0e-3) & aperture_mask(cell, nx, ny)).astype(np.complex128)
    Psi0 = Psi0 * np.exp(-2j * np.pi * (kx[None, :] * x0 + ky[:, None] * y0))
    if aberrations is not None:
        Psi0 = Psi0 * np.exp(-1j * aberration_function(cell, nx, ny, kV, aberrations))
    psi0 = np.fft.ifft2(Psi0)
    return psi0 * np.sqrt(nx * ny / np.sum(np.abs(psi0) ** 2))


# ----------------------------------------------------------------------------- a5+a6: multislice
def propagator(cell, nx: int, ny: int, kV: float, dz: float) -> np.ndarray:
    """P(k) A(k) = exp(-i pi lambda dz |k|^2) inside the band limit, 0 outside (A10)."""
    kx, ky = k_grids(cell, nx, ny)
    k2 = kx[None, :] ** 2 + ky[:, None] ** 2
    return np.exp(-1j * np.pi * wavelength_A(kV) * dz * k2) * aperture_mask(cell, nx, ny)


def multislice(psi0: np.ndarray, V: np.ndarray, cell, kV: float, last_propagator: bool = True,
               return_real_space: bool = False) -> np.ndarray:
    """Exit wave in k-space, unitary: Psi(k) = fft2(psi)/sqrt(Nx Ny)  (A9, A13).

    for s = 0..S-1 (increasing z):  psi <- psi exp(i sigma V_s);  psi <- ifft2(P A fft2(psi)).
    S transmissions and S propagations (A9); `last_propagator=False` skips the final one (pin P9)."""
    S, ny, nx = V.shape
    sig = sigma_rad_per_VA(kV)
    PA = propagator(cell, nx, ny, kV, float(cell[2]) / S)
    psi = psi0.astype(np.complex128).copy()
    for s in range(S):
        psi = psi * np.exp(1j * sig * V[s])
        if s < S - 1 or last_propagator:
            psi = np.fft.ifft2(PA * np.fft.fft2(psi))
    if return_real_space:
        return psi
    return np.fft.fft2(psi) / np.sqrt(nx * ny)


# ----------------------------------------------------------------------------- a7: TACAW transform
def tacaw_intensity(exit_waves: np.ndarray, bins=None) -> np.ndarray:
    """I[n][...] = |sum_j (Psi_j - <Psi>_t) exp(-2 pi i n j / F)|^2 over axis 0 (A14).

    Mean over all F frames, no window, unnormalised forward FFT, both signs of omega kept.
    `bins`: list of signed FFT bins n (index n mod F) or None for all F in FFT order."""
    F = exit_waves.shape[0]
    d = exit_waves - exit_waves.mean(axis=0, keepdims=True)
    spec = np.fft.fft(d, axis=0)
    I = np.abs(spec) ** 2
    if bins is None:
        return I
    return I[np.asarray(bins, dtype=np.int64) % F]


# ----------------------------------------------------------------------------- a8: reductions
def sdp(I: np.ndarray, bin_lo: int, bin_hi: int) -> np.ndarray:
    """Spectral diffraction pattern: sum over probes and bins bin_lo..bin_hi inclusive of I[P][n][ny][nx]
    (A15 incoherent probe sum)."""
    return I[:, bin_lo:bin_hi + 1].sum(axis=(0, 1))


def detector_mask(cell, nx: int, ny: int, k_in: float, k_out: float) -> np.ndarray:
    """k_in <= |k| < k_out."""
    kx, ky = k_grids(cell, nx, ny)
    k = np.sqrt(kx[None, :] ** 2 + ky[:, None] ** 2)
    return (k >= k_in) & (k < k_out)


def spectrum_image(I: np.ndarray, cell, k_in: float, k_out: float) -> np.ndarray:
    """out[P][n] = sum_{k in detector} I[P][n][k]  (A16)."""
    P, nb, ny, nx = I.shape
    m = detector_mask(cell, nx, ny, k_in, k_out)
    return (I * m[None, None]).sum(axis=(2, 3))


def haadf(exit_waves: np.ndarray, cell, k_in: float, k_out: float) -> np.ndarray:
    """Annular detector signal per probe position ("HAADFData ... annular dark field scanning probe
    imaging", "integrates scattered intensity within configurable collection angle ranges"):
        out[p] = (1/F) sum_f sum_{k_in <= |k| < k_out} |Psi_pf(k)|^2 / (nx ny)
    for exit waves [P][F][ny][nx] in k-space, unitary (step 7): the fraction of the incident intensity (mean
    intensity 1 per pixel) that lands on the detector, averaged over the frames (frozen-phonon average).
    k_out <= 0: no outer limit.  [Reading: detector limits in 1/Angstrom like spectrum_image; theta = lambda k.]"""
    P, F, ny, nx = exit_waves.shape
    kx, ky = k_grids(cell, nx, ny)
    k = np.sqrt(kx[None, :] ** 2 + ky[:, None] ** 2)
    m = (k >= k_in) & ((k < k_out) if k_out > 0 else True)
    inten = np.abs(exit_waves) ** 2
    return (inten * m[None, None]).sum(axis=(2, 3)).mean(axis=1) / (nx * ny)


def accumulate_intensity(acc: np.ndarray, I: np.ndarray, w_acc: float, w_new: float) -> np.ndarray:
    """acc <- w_acc * acc + w_new * I: averaging |Psi(k,w)|^2 over independent trajectories or trajectory
    segments (Suppl. PAPER.md:305).  Running mean over n results: w_acc = (n-1)/n, w_new = 1/n."""
    return w_acc * acc + w_new * I


def dispersion_pixels(cell, nx: int, ny: int, kx_path, ky_path) -> np.ndarray:
    """Linear pixel index iy*nx+ix of the nearest reciprocal-grid point to each path point:
    ix = floor(kx Lx + 0.5) mod Nx (A17). int32."""
    ix = np.floor(np.asarray(kx_path, dtype=np.float64) * float(cell[0]) + 0.5).astype(np.int64) % nx
    iy = np.floor(np.asarray(ky_path, dtype=np.float64) * float(cell[1]) + 0.5).astype(np.int64) % ny
    return (iy * nx + ix).astype(np.int32)


def dispersion(I: np.ndarray, cell, kx_path, ky_path):
    """out[n][i] = sum_P I[P][n][pix_i]."""
    P, nb, ny, nx = I.shape
    pix = dispersion_pixels(cell, nx, ny, kx_path, ky_path)
    return I.reshape(P, nb, ny * nx)[:, :, pix].sum(axis=0), pix


def qbin_index(cell, nx: int, ny: int, dq: float, n_q: int) -> np.ndarray:
    """b = floor(sqrt(kx^2+ky^2)/dq), -1 if b >= n_q. int32 [ny][nx]."""
    kx, ky = k_grids(cell, nx, ny)
    b = np.floor(np.sqrt(kx[None, :] * kx[None, :] + ky[:, None] * ky[:, None]) / dq).astype(np.int64)
    b[b >= n_q] = -1
    return b.astype(np.int32)


def qbin(I: np.ndarray, cell, dq: float, n_q: int):
    """out[n][b] = sum_P sum_{k: bin(k)=b} I[P][n][k]."""
    P, nb, ny, nx = I.shape
    idx = qbin_index(cell, nx, ny, dq, n_q)
    out = np.zeros((nb, n_q), dtype=np.float64)
    Is = I.sum(axis=0).reshape(nb, ny * nx)
    flat = idx.ravel()
    for b in range(n_q):
        out[:, b] = Is[:, flat == b].sum(axis=1)
    return out, idx


def frequency_bin(f_THz: float, n_frames: int, dt_fs: float) -> int:
    """Nearest time-FFT bin: n = floor(f F dt + 0.5) (A16)."""
    return int(np.floor(f_THz * n_frames * dt_fs * 1.0e-3 + 0.5))


# ----------------------------------------------------------------------------- whole path
def run_path(pos32: np.ndarray, elem_of_atom: np.ndarray, coef, n_lorentz, n_gauss, cell, nx, ny, n_slices,
             kV, psi0_list, bins=None, frames=None):
    """positions -> I[P][n][ny][nx] for the listed frames (default all), plus exit waves [P][F][ny][nx]."""
    F = pos32.shape[0] if frames is None else len(frames)
    frames = range(pos32.shape[0]) if frames is None else frames
    P = len(psi0_list)
    exit_w = np.empty((P, F, ny, nx), dtype=np.complex128)
    for i, f in enumerate(frames):
        V, _ = projected_potential(pos32[f], elem_of_atom, coef, n_lorentz, n_gauss, cell, nx, ny, n_slices)
        for p in range(P):
            exit_w[p, i] = multislice(psi0_list[p], V, cell, kV)
    I = np.stack([tacaw_intensity(exit_w[p], bins) for p in range(P)])
    return I, exit_w
