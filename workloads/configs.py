"""Workload descriptions + seeded synthetic trajectories for BASELINE.json `configs`.

These stand in for the paper's ORB-MD trajectories, which need
ORB weights and ASE (absent).  Shapes, sizes and displacement magnitudes follow
BASELINE.json `configs` / SURVEY.md §8(d); the recipe is restated in DESIGN.md §4.

Common recipe: ideal lattice R_j, shifted by dz/2 along z so atomic planes sit at slice
centres, plus
    u_j(t) = sum_m A_mj e_m cos(2 pi (q_m . R_j - f_m t) + phi_m) + noise,
q_m = (h/Lx, k/Ly, l/Lz) with integer h,k,l (commensurate with the periodic cell),
f_m = n_m/(F dt) on the time-FFT grid, e_m uniform on the sphere, phi_m uniform.
Everything is generated in float64 and stored as float32 (the ABI's position type).

No TACAW arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

CONFIG_NAMES = ("c1_si_128", "c2_hbn_256", "c3_si_probe_512", "c4_interface_1024", "c5_al_sweep")

_AMU = 1.66053906660e-27      # kg
_HBAR = 1.054571817e-34       # J s
_KB = 1.380649e-23            # J/K
_MASS = {5: 10.81, 6: 12.011, 7: 14.007, 8: 15.999, 12: 24.305, 13: 26.982, 14: 28.086,
         22: 47.867, 32: 72.63, 38: 87.62}


@dataclass
class Workload:
    name: str
    cell: np.ndarray            # (3,) Angstrom, orthorhombic
    nx: int
    ny: int
    n_slices: int
    kV: float
    dt_fs: float
    n_frames: int
    Z: np.ndarray               # int32 [Na]
    R0: np.ndarray              # float64 [Na,3] ideal positions (already z-shifted)
    ff_kind: str
    beam: str                   # "plane" | "probe" | "tilt"
    semi_angle_mrad: float = 0.0
    probe_xy: np.ndarray | None = None      # float64 [P,2] Angstrom (beam == "probe")
    tilts: np.ndarray | None = None         # int32 [P,2] reciprocal-grid indices (beam == "tilt")
    bins: np.ndarray | None = None          # int32 list of FFT bins n, or None = all F bins
    seed: int = 0
    # displacement model
    mode_q: np.ndarray = field(default=None, repr=False)      # int [M,3]
    mode_n: np.ndarray = field(default=None, repr=False)      # int [M] time-FFT bin of f_m
    mode_e: np.ndarray = field(default=None, repr=False)      # [M,3]
    mode_phi: np.ndarray = field(default=None, repr=False)    # [M]
    mode_amp: np.ndarray = field(default=None, repr=False)    # [M,Na] Angstrom
    noise_sigma: float = 0.0
    noise_tau_fs: float = 0.0   # 0 -> white
    anharm: float = 0.0         # u <- h + anharm*|h|*h/anharm_scale
    anharm_scale: float = 1.0
    _noise_cache: np.ndarray | None = field(default=None, repr=False)

    # ---------------------------------------------------------------- derived
    @property
    def n_atoms(self) -> int:
        return int(self.Z.shape[0])

    @property
    def slice_dz(self) -> float:
        return float(self.cell[2]) / self.n_slices

    @property
    def elements(self) -> np.ndarray:
        return np.unique(self.Z).astype(np.int32)

    @property
    def n_probes(self) -> int:
        if self.beam == "probe":
            return int(self.probe_xy.shape[0])
        if self.beam == "tilt":
            return int(self.tilts.shape[0])
        return 1

    # ------------------------------------------------------------- trajectory
    def _harmonic(self, f0: int, f1: int) -> np.ndarray:
        """float64 [f1-f0, Na, 3] harmonic displacements via one GEMM (cos(a-b) identity)."""
        M = self.mode_q.shape[0]
        kq = self.mode_q / self.cell[None, :]                         # [M,3] 1/Angstrom
        alpha = 2.0 * np.pi * (self.R0 @ kq.T) + self.mode_phi[None, :]   # [Na,M]
        t = np.arange(f0, f1, dtype=np.float64)
        beta = 2.0 * np.pi * np.outer(self.mode_n / float(self.n_frames), t)  # [M,T]
        amp = self.mode_amp.T                                          # [Na,M]
        out = np.empty((f1 - f0, self.n_atoms, 3))
        H = np.concatenate([np.cos(beta), np.sin(beta)], axis=0)       # [2M,T]
        for c in range(3):
            G = np.concatenate([amp * np.cos(alpha) * self.mode_e[None, :, c],
                                amp * np.sin(alpha) * self.mode_e[None, :, c]], axis=1)  # [Na,2M]
            out[:, :, c] = (G @ H).T
        assert M == self.mode_n.shape[0]
        return out

    def _noise(self, f0: int, f1: int) -> np.ndarray:
        if self.noise_sigma == 0.0:
            return 0.0
        if self.noise_tau_fs == 0.0:
            out = np.empty((f1 - f0, self.n_atoms, 3))
            for i, f in enumerate(range(f0, f1)):
                out[i] = np.random.default_rng([self.seed, 7, f]).normal(0.0, self.noise_sigma, (self.n_atoms, 3))
            return out
        if self._noise_cache is None:                                  # AR(1), sequential
            rho = np.exp(-self.dt_fs / self.noise_tau_fs)
            x = np.empty((self.n_frames, self.n_atoms, 3), dtype=np.float32)
            cur = np.random.default_rng([self.seed, 7, 0]).normal(0.0, self.noise_sigma, (self.n_atoms, 3))
            x[0] = cur
            for f in range(1, self.n_frames):
                xi = np.random.default_rng([self.seed, 7, f]).normal(0.0, self.noise_sigma, (self.n_atoms, 3))
                cur = rho * cur + np.sqrt(1.0 - rho * rho) * xi
                x[f] = cur
            self._noise_cache = x
        return self._noise_cache[f0:f1].astype(np.float64)

    def positions(self, f0: int = 0, f1: int | None = None) -> np.ndarray:
        """float32 [f1-f0, Na, 3] Cartesian positions (Angstrom) of frames f0..f1-1."""
        f1 = self.n_frames if f1 is None else f1
        h = self._harmonic(f0, f1)
        if self.anharm != 0.0:
            h = h + self.anharm * np.abs(h) * h / self.anharm_scale
        return (self.R0[None] + h + self._noise(f0, f1)).astype(np.float32)


# ------------------------------------------------------------------ lattices
def _tile(basis_frac: np.ndarray, basis_Z, a: np.ndarray, reps) -> tuple[np.ndarray, np.ndarray]:
    nxr, nyr, nzr = reps
    i, j, k = np.meshgrid(np.arange(nxr), np.arange(nyr), np.arange(nzr), indexing="ij")
    origins = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1).astype(np.float64)   # [Nc,3]
    R = (origins[:, None, :] + basis_frac[None, :, :]) * a[None, None, :]
    Z = np.tile(np.asarray(basis_Z, dtype=np.int32), origins.shape[0])
    return R.reshape(-1, 3), Z


_FCC = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
_DIAMOND = np.concatenate([_FCC, _FCC + 0.25])


def _modes(rng, M, n_lo, n_hi, qmax):
    q = np.zeros((M, 3), dtype=np.int64)
    for m in range(M):
        while not q[m].any():
            q[m] = rng.integers(-qmax, qmax + 1, 3)
    n = rng.integers(n_lo, n_hi + 1, M)
    e = rng.normal(size=(M, 3))
    e /= np.linalg.norm(e, axis=1, keepdims=True)
    phi = rng.uniform(0.0, 2.0 * np.pi, M)
    return q, n, e, phi


def _finish(w: Workload) -> Workload:
    w.R0 = w.R0 + np.array([0.0, 0.0, 0.5 * w.slice_dz])   # planes at slice centres
    w.Z = w.Z.astype(np.int32)
    return w


# ------------------------------------------------------------------ configs
def make_workload(name: str, *, mini: bool = False, n_frames: int | None = None,
                  grid: int | None = None, n_probes_side: int | None = None) -> Workload:
    """Build config `name` (one of CONFIG_NAMES).  `mini=True` gives the small twin used by the
    end-to-end parity tests (same recipe, smaller cell/grid/frames); the keyword overrides
    change single dimensions (bench.py uses the full sizes)."""
    if name == "c1_si_128":
        # Si 3x3x3 (216 atoms, a=5.431), plane wave 100 kV, 128^2, S=12, F=64, dt=5 fs,
        # 8 modes A=0.05/sqrt(8) + white noise 0.01, 5-Gaussian form factors.
        a, reps, F, g, S = 5.431, (3, 3, 3), 64, 128, 12
        if mini:
            reps, F, g, S = (2, 2, 1), 32, 64, 4
        F = n_frames or F; g = grid or g
        rng = np.random.default_rng(1001)
        R, Z = _tile(_DIAMOND, [14] * 8, np.array([a, a, a]), reps)
        q, n, e, phi = _modes(rng, 8, 1, max(1, min(5, F // 2 - 1)), 2)
        amp = np.full((8, R.shape[0]), 0.05 / np.sqrt(8.0))
        return _finish(Workload(name, a * np.array(reps, float), g, g, S, 100.0, 5.0, F, Z, R, "gauss5",
                                "plane", seed=1001, mode_q=q, mode_n=n, mode_e=e, mode_phi=phi,
                                mode_amp=amp, noise_sigma=0.01))
    if name == "c2_hbn_256":
        # hBN-like monolayer, rectangular 4-atom cell a x sqrt(3)a, 24x12 cells = 1152 atoms,
        # 20 A vacuum box, 60 kV plane wave, 256^2, S=10, F=512, dt=2 fs, 64 modes with 300 K
        # Bose amplitudes, output bins 0..49 (0-200 meV).
        a, reps, F, g, S = 2.50, (24, 12, 1), 512, 256, 10
        if mini:
            reps, F, g, S = (6, 3, 1), 32, 64, 5
        F = n_frames or F; g = grid or g
        rng = np.random.default_rng(1002)
        b = a * np.sqrt(3.0)
        basis = np.array([[0, 0, 0.5], [0, 1 / 3, 0.5], [0.5, 0.5, 0.5], [0.5, 0.5 + 1 / 3, 0.5]])
        R, Z = _tile(basis, [5, 7, 5, 7], np.array([a, b, 20.0]), reps)
        M = 64
        dfTHz = 1.0e3 / (F * 2.0)                                     # THz per bin (dt in fs)
        n_lo = max(1, int(np.ceil(2.0 / dfTHz))); n_hi = max(n_lo, min(F // 2 - 1, int(48.0 / dfTHz)))
        q, n, e, phi = _modes(rng, M, n_lo, n_hi, 4)
        fm = n * dfTHz * 1e12                                          # Hz
        nB = 1.0 / np.expm1(_HBAR * 2 * np.pi * fm / (_KB * 300.0))
        mass = np.array([_MASS[int(z)] for z in Z]) * _AMU
        amp = np.sqrt(2.0 / M) * np.sqrt(_HBAR * (2 * nB[:, None] + 1) / (2 * mass[None, :] * 2 * np.pi * fm[:, None])) * 1e10
        nb = min(50, F)
        return _finish(Workload(name, np.array([a * reps[0], b * reps[1], 20.0]), g, g, S, 60.0, 2.0, F, Z, R,
                                "kirkland33", "plane", bins=np.arange(nb, dtype=np.int32), seed=1002,
                                mode_q=q, mode_n=n, mode_e=e, mode_phi=phi, mode_amp=amp))
    if name == "c3_si_probe_512":
        # Si 8x8x20 (10240 atoms), 30 mrad probe 100 kV, 512^2, S=80, F=1024, dt=5 fs,
        # 32 modes + quadratic distortion + AR(1) noise, 16x16 probe scan over one unit cell.
        a, reps, F, g, S, ps = 5.431, (8, 8, 20), 1024, 512, 80, 16
        if mini:
            reps, F, g, S, ps = (3, 3, 2), 32, 128, 8, 2
        F = n_frames or F; g = grid or g; ps = n_probes_side or ps
        rng = np.random.default_rng(1003)
        R, Z = _tile(_DIAMOND, [14] * 8, np.array([a, a, a]), reps)
        M = 32
        q, n, e, phi = _modes(rng, M, 1, max(1, min(F // 2 - 1, int(16.0 / (1e3 / (F * 5.0))))), 3)
        amp = np.full((M, R.shape[0]), 0.05 * np.sqrt(2.0 / M))       # total (3-D) RMS 0.05 A
        L = a * np.array(reps, float)
        off = 0.37 * a
        px = off + (np.arange(ps) + 0.0) * a / ps
        xy = np.stack(np.meshgrid(px, px, indexing="ij"), axis=-1).reshape(-1, 2)
        return _finish(Workload(name, L, g, g, S, 100.0, 5.0, F, Z, R, "kirkland33", "probe",
                                semi_angle_mrad=30.0, probe_xy=xy, seed=1003,
                                mode_q=q, mode_n=n, mode_e=e, mode_phi=phi, mode_amp=amp,
                                noise_sigma=0.02, noise_tau_fs=50.0, anharm=0.2, anharm_scale=0.05))
    if name == "c4_interface_1024":
        # SrTiO3 | rocksalt (MgO-like) interface slab, 48600 atoms, 200 kV plane wave, 1024^2,
        # S=120, F=4096, dt=2 fs, 128 Gaussian-amplitude modes (RMS 0.08 A per coordinate),
        # streaming per-omega-bin DFT into bins 0..255.
        nsto, nrs, nyc_sto, nyc_rs, nz_sto, nz_rs, F, g, S = 14, 13, 14, 13, 22, 20, 4096, 1024, 120
        if mini:
            nsto, nrs, nyc_sto, nyc_rs, nz_sto, nz_rs, F, g, S = 3, 3, 3, 3, 2, 2, 64, 128, 6
        F = n_frames or F; g = grid or g
        rng = np.random.default_rng(1004)
        a_sto = 3.905
        Lxh, Ly, Lz = nsto * a_sto, nyc_sto * a_sto, nz_sto * a_sto
        a_rs = np.array([Lxh / nrs, Ly / nyc_rs, Lz / nz_rs])
        sto_basis = np.array([[0, 0, 0], [.5, .5, .5], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]], float)
        R1, Z1 = _tile(sto_basis, [38, 22, 8, 8, 8], np.array([a_sto] * 3), (nsto, nyc_sto, nz_sto))
        rs_basis = np.concatenate([_FCC, _FCC + np.array([.5, 0, 0])]) % 1.0
        R2, Z2 = _tile(rs_basis, [12] * 4 + [8] * 4, a_rs, (nrs, nyc_rs, nz_rs))
        R2 = R2 + np.array([Lxh, 0, 0])
        R = np.concatenate([R1, R2]); Z = np.concatenate([Z1, Z2])
        M = 128
        q, n, e, phi = _modes(rng, M, 1, max(1, min(F // 2 - 1, 255)), 5)
        g_amp = np.abs(rng.normal(size=M))
        # per-coordinate RMS^2 = sum_m amp_m^2 <e_mc^2> / 2 = sum_m amp_m^2 / 6 = 0.08^2
        amp = np.tile((g_amp * 0.08 * np.sqrt(6.0 / (g_amp ** 2).sum()))[:, None], (1, R.shape[0]))
        nb = min(256, F)
        return _finish(Workload(name, np.array([2 * Lxh, Ly, Lz]), g, g, S, 200.0, 2.0, F, Z, R, "kirkland33",
                                "plane", bins=np.arange(nb, dtype=np.int32), seed=1004,
                                mode_q=q, mode_n=n, mode_e=e, mode_phi=phi, mode_amp=amp))
    if name == "c5_al_sweep":
        # Al fcc 16x16x40 (40960 atoms), 100 kV, 8 beam tilts (m_t, 0), grid 256..2048 (default 512),
        # S=80 (dz=a/2), F=2048, dt=4 fs, 64 modes 1-10 THz, RMS 0.07 A.
        a, reps, F, g, S, nt = 4.05, (16, 16, 40), 2048, 512, 80, 8
        if mini:
            reps, F, g, S, nt = (4, 4, 3), 32, 64, 6, 2
        F = n_frames or F; g = grid or g; nt = n_probes_side or nt
        rng = np.random.default_rng(1005)
        R, Z = _tile(_FCC, [13] * 4, np.array([a, a, a]), reps)
        M = 64
        dfTHz = 1.0e3 / (F * 4.0)
        n_lo = max(1, int(np.ceil(1.0 / dfTHz))); n_hi = max(n_lo, min(F // 2 - 1, int(10.0 / dfTHz)))
        q, n, e, phi = _modes(rng, M, n_lo, n_hi, 4)
        amp = np.full((M, R.shape[0]), 0.07 * np.sqrt(6.0 / M))
        tilts = np.stack([np.arange(nt), np.zeros(nt)], axis=1).astype(np.int32)
        return _finish(Workload(name, a * np.array(reps, float), g, g, S, 100.0, 4.0, F, Z, R, "kirkland33",
                                "tilt", tilts=tilts, seed=1005,
                                mode_q=q, mode_n=n, mode_e=e, mode_phi=phi, mode_amp=amp))
    raise ValueError(f"unknown workload {name!r}; choose from {CONFIG_NAMES}")
