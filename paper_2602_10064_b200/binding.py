"""ctypes binding of include/pyslice_b200.h — argument marshalling only.

Names follow the C ABI (`ps_build_slices`, `ps_multislice`, `ps_tacaw`, ...); each module-level
function takes a `Context` first and torch CUDA tensors for every `d_*` argument of the header.
Output tensors are allocated here with torch (device memory is torch's job) unless passed in.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_NAME = "libpyslice_b200.so"
_lib = None

PS_OK, PS_EINVAL, PS_EUNSUPPORTED, PS_EWORKSPACE, PS_ECUDA, PS_ESTATE = 0, -1, -2, -3, -4, -5
PS_LAYOUT_DENSE = 0
PS_LAYOUT_TILED_APERTURE = 1

_PROTOTYPES = {
    # name: (restype, argtypes)
    "ps_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]),
    "ps_destroy": (None, [C.c_void_p]),
    "ps_last_error": (C.c_char_p, [C.c_void_p]),
    "ps_version": (C.c_char_p, []),
    "ps_set_form_factors": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "ps_set_geometry": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double]),
    "ps_get_geometry": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_int)]),
    "ps_workspace_bytes": (C.c_size_t, [C.c_void_p, C.c_int, C.c_int]),
    "ps_set_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "ps_set_wave_chunk": (C.c_int, [C.c_void_p, C.c_int]),
    "ps_set_vk_mode": (C.c_int, [C.c_void_p, C.c_int]),
    "ps_set_tuning": (C.c_int, [C.c_void_p, C.c_char_p, C.c_int]),
    "ps_set_vacuum_shortcut": (C.c_int, [C.c_void_p, C.c_int]),
    "ps_set_aberrations": (C.c_int, [C.c_void_p, C.c_void_p]),
    "ps_apply_aberrations": (C.c_int, [C.c_void_p, C.c_double, C.c_void_p, C.c_longlong]),
    "ps_build_slices": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]),
    "ps_make_incident": (C.c_int, [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_int, C.c_void_p]),
    "ps_multislice": (C.c_int, [C.c_void_p, C.c_double, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_int]),
    "ps_tacaw": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_void_p]),
    "ps_multislice_fused": (C.c_int, [C.c_void_p, C.c_double, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                      C.c_void_p, C.c_int]),
    "ps_exit_bytes": (C.c_size_t, [C.c_void_p, C.c_int, C.c_int, C.c_int]),
    "ps_exit_to_dense": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "ps_tacaw_begin": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_void_p]),
    "ps_tacaw_set_reference": (C.c_int, [C.c_void_p, C.c_void_p]),
    "ps_tacaw_add": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int]),
    "ps_tacaw_finish": (C.c_int, [C.c_void_p, C.c_void_p]),
    "ps_tacaw_finish_shard": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "ps_sdp": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]),
    "ps_spectrum_image": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p]),
    "ps_spectrum_image_static": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p]),
    "ps_static_scratch_bytes": (C.c_size_t, []),
    "ps_haadf": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p]),
    "ps_accumulate_intensity": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_double, C.c_double]),
    "ps_dispersion": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "ps_qbin": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_void_p]),
    "ps_launch_count": (C.c_longlong, [C.c_void_p]),
    "ps_check_async": (C.c_int, [C.c_void_p]),
    "ps_profile_enable": (C.c_int, [C.c_void_p, C.c_int]),
    "ps_profile_read": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int), C.c_void_p, C.c_void_p, C.c_void_p]),
}


class PSError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"pyslice_b200 status {status}: {message}")
        self.status = status


def library_path() -> str:
    return os.path.join(_HERE, _LIB_NAME)


def exported_symbols():
    return tuple(_PROTOTYPES)


def load_library():
    """dlopen the in-tree library; raises (no fallback) when it has not been built."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: build it with `python -m paper_2602_10064_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(path)
        for name, (res, args) in _PROTOTYPES.items():
            fn = getattr(lib, name)          # AttributeError if the library does not export it
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _host(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def _need(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    return t


class Context:
    """Owns one `ps_ctx` bound to a torch CUDA device and stream."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pyslice_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._lib = load_library()
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        torch.zeros(1, device=self.device)                       # make sure the primary context exists
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        st = self._lib.ps_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream))
        if st != PS_OK:
            raise PSError(st, self._lib.ps_last_error(None).decode())
        self._h = h
        self.cell = None
        self.nx = self.ny = self.n_slices = 0
        self.dz_eff = 0.0
        self.n_k_aperture = 0
        self._ws = None

    # ------------------------------------------------------------------ plumbing
    def _check(self, st: int):
        if st != PS_OK:
            raise PSError(st, self._lib.ps_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.ps_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launches(self) -> int:
        return int(self._lib.ps_launch_count(self._h))

    def check_async(self):
        """Wait for the ctx stream and raise the error an earlier asynchronous call flagged on the device, if any
        (`ps_check_async`): call it after the last call of a run, before reading results."""
        self._check(self._lib.ps_check_async(self._h))

    synchronize = check_async

    def profile_enable(self, on: bool = True):
        self._check(self._lib.ps_profile_enable(self._h, int(bool(on))))

    def profile_read(self, reset: bool = True) -> dict:
        """{kernel name: (summed device ms, launch groups)} from the per-launch CUDA events."""
        n = C.c_int()
        names = (C.c_char_p * 16)()
        ms = (C.c_double * 16)()
        cnt = (C.c_longlong * 16)()
        self._check(self._lib.ps_profile_read(self._h, int(bool(reset)), C.byref(n), names, ms, cnt))
        return {names[i].decode(): (float(ms[i]), int(cnt[i])) for i in range(n.value)}

    def version(self) -> str:
        return self._lib.ps_version().decode()

    # ------------------------------------------------------------------ setup
    def set_form_factors(self, Z, n_lorentz: int, n_gauss: int, coef):
        Zh, Zp = _host(Z, np.int32)
        ch, cp = _host(coef, np.float64)
        assert ch.shape == (Zh.shape[0], 2 * n_lorentz + 2 * n_gauss)
        self._check(self._lib.ps_set_form_factors(self._h, int(Zh.shape[0]), Zp, n_lorentz, n_gauss, cp))

    def set_geometry(self, cell, nx: int, ny: int, slice_dz: float):
        ch, cp = _host(cell, np.float64)
        self._check(self._lib.ps_set_geometry(self._h, cp, int(nx), int(ny), float(slice_dz)))
        ns, dz, nk = C.c_int(), C.c_double(), C.c_int()
        self._check(self._lib.ps_get_geometry(self._h, C.byref(ns), C.byref(dz), C.byref(nk)))
        self.cell, self.nx, self.ny = ch.copy(), int(nx), int(ny)
        self.n_slices, self.dz_eff, self.n_k_aperture = ns.value, dz.value, nk.value

    def workspace_bytes(self, n_frames_chunk: int, n_atoms: int) -> int:
        return int(self._lib.ps_workspace_bytes(self._h, int(n_frames_chunk), int(n_atoms)))

    def set_workspace(self, ws):
        """ws: uint8 CUDA tensor (kept alive by this object) or None."""
        self._ws = ws
        if ws is None:
            self._check(self._lib.ps_set_workspace(self._h, C.c_void_p(0), 0))
        else:
            self._check(self._lib.ps_set_workspace(self._h, _ptr(ws), ws.numel() * ws.element_size()))

    def set_aberrations(self, coef=None):
        """coef = (C10, C12, phi12, C21, phi21, C23, phi23, C30) in Angstrom / rad, or None to switch them off."""
        if coef is None:
            self._check(self._lib.ps_set_aberrations(self._h, C.c_void_p(0)))
        else:
            ch, cp = _host(coef, np.float64)
            assert ch.shape == (8,)
            self._check(self._lib.ps_set_aberrations(self._h, cp))

    def apply_aberrations(self, kV: float, d_waves_k):
        """In place: k-space waves complex64 [..., ny, nx] *= exp(-i chi(k))."""
        import torch
        _need(d_waves_k, torch.complex64, "d_waves_k")
        n = d_waves_k.numel() // (self.nx * self.ny)
        self._check(self._lib.ps_apply_aberrations(self._h, float(kV), _ptr(d_waves_k), n))
        return d_waves_k

    def set_vacuum_shortcut(self, on: bool):
        """Rows with V == 0 are only rescaled by ps_multislice (exact; default off)."""
        self._check(self._lib.ps_set_vacuum_shortcut(self._h, int(bool(on))))

    def set_vk_mode(self, mode: int):
        """0 auto, 1 FP32 SIMT structure-factor sums, 2 tcgen05 3xTF32 sums."""
        self._check(self._lib.ps_set_vk_mode(self._h, int(mode)))

    def set_tuning(self, key: str, value: int):
        """Named tuning knobs ("resident"); see include/pyslice_b200.h."""
        self._check(self._lib.ps_set_tuning(self._h, key.encode(), int(value)))

    def set_wave_chunk(self, n_waves: int):
        self._check(self._lib.ps_set_wave_chunk(self._h, int(n_waves)))


# ---------------------------------------------------------------------- hot path (names of the C ABI)
def ps_build_slices(ctx: Context, d_pos, d_Z, d_V=None, d_slice_idx=None, want_slice_idx: bool = False):
    """positions float32 [F][Na][3] + Z int32 [Na] -> V float32 [F][S][ny][nx] (and slice index int32 [F][Na])."""
    import torch
    _need(d_pos, torch.float32, "d_pos"); _need(d_Z, torch.int32, "d_Z")
    F, Na = int(d_pos.shape[0]), int(d_pos.shape[1])
    if d_V is None:
        d_V = torch.empty((F, ctx.n_slices, ctx.ny, ctx.nx), dtype=torch.float32, device=ctx.device)
    _need(d_V, torch.float32, "d_V")
    if d_slice_idx is None and want_slice_idx:
        d_slice_idx = torch.empty((F, Na), dtype=torch.int32, device=ctx.device)
    ctx._check(ctx._lib.ps_build_slices(ctx._h, _ptr(d_pos), _ptr(d_Z), F, Na, _ptr(d_V), _ptr(d_slice_idx)))
    return (d_V, d_slice_idx) if (want_slice_idx or d_slice_idx is not None) else d_V


def ps_make_incident(ctx: Context, kV: float, semi_angle_mrad: float = 0.0, xy_or_tilt=None, is_tilt: bool = False,
                     n: int | None = None, d_psi0=None):
    """Incident waves complex64 [n][ny][nx] (plane wave, tilted plane waves or focused probes)."""
    import torch
    if xy_or_tilt is not None:
        xh, xp = _host(xy_or_tilt, np.float64)
        n = int(xh.shape[0])
    else:
        xh, xp = None, C.c_void_p(0)
        n = 1 if n is None else int(n)
    if d_psi0 is None:
        d_psi0 = torch.empty((n, ctx.ny, ctx.nx), dtype=torch.complex64, device=ctx.device)
    _need(d_psi0, torch.complex64, "d_psi0")
    ctx._check(ctx._lib.ps_make_incident(ctx._h, float(kV), float(semi_angle_mrad), n, xp, int(bool(is_tilt)), _ptr(d_psi0)))
    return d_psi0


def exit_shape(ctx: Context, n_probes: int, n_frames: int, layout: int = PS_LAYOUT_DENSE):
    """Shape of a complex64 exit-wave array: dense [P][F][ny][nx], tiled [P][ny][n_tiles][F][8] (size from ps_exit_bytes)."""
    if layout == PS_LAYOUT_DENSE:
        return (n_probes, n_frames, ctx.ny, ctx.nx)
    nbytes = int(ctx._lib.ps_exit_bytes(ctx._h, int(n_probes), int(n_frames), int(layout)))
    if nbytes == 0:
        raise ValueError("unknown exit layout")
    return (n_probes, ctx.ny, nbytes // (n_probes * ctx.ny * n_frames * 64), n_frames, 8)


def _exit_layout(d_exit):
    return PS_LAYOUT_TILED_APERTURE if d_exit.dim() == 5 else PS_LAYOUT_DENSE


def ps_multislice(ctx: Context, kV: float, d_psi0, d_V, d_exit=None, layout: int = PS_LAYOUT_DENSE):
    """psi0 complex64 [P][ny][nx], V float32 [F][S][ny][nx] -> k-space exit waves complex64, dense [P][F][ny][nx] or
    (layout = PS_LAYOUT_TILED_APERTURE, or a 5-D d_exit) tiled [P][ny][n_tiles][F][8]."""
    import torch
    _need(d_psi0, torch.complex64, "d_psi0"); _need(d_V, torch.float32, "d_V")
    P, F = int(d_psi0.shape[0]), int(d_V.shape[0])
    if d_exit is None:
        d_exit = torch.empty(exit_shape(ctx, P, F, layout), dtype=torch.complex64, device=ctx.device)
    _need(d_exit, torch.complex64, "d_exit")
    ctx._check(ctx._lib.ps_multislice(ctx._h, float(kV), _ptr(d_psi0), P, _ptr(d_V), F, _ptr(d_exit), _exit_layout(d_exit)))
    return d_exit


def ps_multislice_fused(ctx: Context, kV: float, d_psi0, d_pos, d_Z, d_exit=None):
    """positions float32 [F][Na][3] + Z int32 [Na] + psi0 complex64 [P][ny][nx] -> exit waves complex64 [P][F][ny][nx]
    without the V array (the row pass builds each row of V from the y-transformed slice pair)."""
    import torch
    _need(d_psi0, torch.complex64, "d_psi0"); _need(d_pos, torch.float32, "d_pos"); _need(d_Z, torch.int32, "d_Z")
    P, F, Na = int(d_psi0.shape[0]), int(d_pos.shape[0]), int(d_pos.shape[1])
    if d_exit is None:
        d_exit = torch.empty((P, F, ctx.ny, ctx.nx), dtype=torch.complex64, device=ctx.device)
    _need(d_exit, torch.complex64, "d_exit")
    ctx._check(ctx._lib.ps_multislice_fused(ctx._h, float(kV), _ptr(d_psi0), P, _ptr(d_pos), _ptr(d_Z), F, Na, _ptr(d_exit),
                                            PS_LAYOUT_DENSE))
    return d_exit


def ps_exit_to_dense(ctx: Context, d_tiled, d_dense=None):
    """Tiled exit waves [P][ny][n_tiles][F][8] -> dense [P][F][ny][nx] (zeros in the tiles the tiled layout omits)."""
    import torch
    _need(d_tiled, torch.complex64, "d_tiled")
    P, F = int(d_tiled.shape[0]), int(d_tiled.shape[3])
    if d_dense is None:
        d_dense = torch.empty((P, F, ctx.ny, ctx.nx), dtype=torch.complex64, device=ctx.device)
    _need(d_dense, torch.complex64, "d_dense")
    ctx._check(ctx._lib.ps_exit_to_dense(ctx._h, _ptr(d_tiled), P, F, _ptr(d_dense)))
    return d_dense


def ps_tacaw(ctx: Context, d_exit, dt_fs: float, bins=None, d_I=None):
    """exit waves complex64 (dense [P][F][ny][nx] or tiled [P][ny][n_tiles][F][8]) -> I float32 [P][n_bins][ny][nx];
    bins = signed FFT bins or None (all)."""
    import torch
    _need(d_exit, torch.complex64, "d_exit")
    layout = _exit_layout(d_exit)
    P, F = int(d_exit.shape[0]), int(d_exit.shape[1] if layout == PS_LAYOUT_DENSE else d_exit.shape[3])
    if bins is None:
        nb, bp, bh = F, C.c_void_p(0), None
    else:
        bh, bp = _host(bins, np.int32)
        nb = int(bh.shape[0])
    if d_I is None:
        d_I = torch.empty((P, nb, ctx.ny, ctx.nx), dtype=torch.float32, device=ctx.device)
    _need(d_I, torch.float32, "d_I")
    ctx._check(ctx._lib.ps_tacaw(ctx._h, _ptr(d_exit), layout, P, F, float(dt_fs), nb, bp, _ptr(d_I)))
    return d_I


class TacawStream:
    """ps_tacaw_begin / ps_tacaw_add / ps_tacaw_finish (per-bin streaming DFT accumulation)."""

    def __init__(self, ctx: Context, n_probes: int, n_frames_total: int, dt_fs: float, bins):
        import torch
        self.ctx = ctx
        bh, bp = _host(bins, np.int32)
        self.n_bins, self.P = int(bh.shape[0]), int(n_probes)
        self.d_acc = torch.empty((n_probes, self.n_bins, ctx.ny, ctx.nx), dtype=torch.complex64, device=ctx.device)
        ctx._check(ctx._lib.ps_tacaw_begin(ctx._h, n_probes, int(n_frames_total), float(dt_fs), self.n_bins, bp, _ptr(self.d_acc)))

    def set_reference(self, d_ref):
        """complex64 [P][ny][nx] wave subtracted from every frame (None = zeros); before the first add."""
        import torch
        if d_ref is not None:
            _need(d_ref, torch.complex64, "d_ref")
        self.ctx._check(self.ctx._lib.ps_tacaw_set_reference(self.ctx._h, _ptr(d_ref)))

    def add(self, d_exit_chunk, frame0: int):
        import torch
        _need(d_exit_chunk, torch.complex64, "d_exit_chunk")
        self.ctx._check(self.ctx._lib.ps_tacaw_add(self.ctx._h, _ptr(d_exit_chunk), int(frame0), int(d_exit_chunk.shape[1])))

    def finish(self, d_I=None):
        import torch
        if d_I is None:
            d_I = torch.empty((self.P, self.n_bins, self.ctx.ny, self.ctx.nx), dtype=torch.float32, device=self.ctx.device)
        self.ctx._check(self.ctx._lib.ps_tacaw_finish(self.ctx._h, _ptr(d_I)))
        return d_I

    def finish_shard(self, d_acc_shard, d_I_shard=None):
        """complex64 [P][n_bins][n_k] (summed over all shards by the caller) -> float32 [P][n_bins][n_k]."""
        import torch
        _need(d_acc_shard, torch.complex64, "d_acc_shard")
        if d_I_shard is None:
            d_I_shard = torch.empty(d_acc_shard.shape, dtype=torch.float32, device=self.ctx.device)
        _need(d_I_shard, torch.float32, "d_I_shard")
        self.ctx._check(self.ctx._lib.ps_tacaw_finish_shard(self.ctx._h, _ptr(d_acc_shard), int(d_acc_shard.shape[-1]), _ptr(d_I_shard)))
        return d_I_shard


def ps_sdp(ctx: Context, d_I, bin_lo: int, bin_hi: int, d_out=None):
    import torch
    _need(d_I, torch.float32, "d_I")
    P, nb = int(d_I.shape[0]), int(d_I.shape[1])
    if d_out is None:
        d_out = torch.empty((ctx.ny, ctx.nx), dtype=torch.float32, device=ctx.device)
    ctx._check(ctx._lib.ps_sdp(ctx._h, _ptr(d_I), P, nb, int(bin_lo), int(bin_hi), _ptr(d_out)))
    return d_out


def ps_spectrum_image(ctx: Context, d_I, k_in: float = 0.0, k_out: float = 0.0, d_out=None):
    import torch
    _need(d_I, torch.float32, "d_I")
    P, nb = int(d_I.shape[0]), int(d_I.shape[1])
    if d_out is None:
        d_out = torch.empty((P, nb), dtype=torch.float32, device=ctx.device)
    ctx._check(ctx._lib.ps_spectrum_image(ctx._h, _ptr(d_I), P, nb, float(k_in), float(k_out), _ptr(d_out)))
    return d_out


def ps_spectrum_image_static(ctx: Context, d_I, d_out, k_in: float = 0.0, k_out: float = 0.0):
    """`ps_spectrum_image` for callers that must not allocate device memory: a process whose pool already owns all of
    HBM, or a loop that cannot take the device-wide stall of cudaMalloc.  The detector mask sits in a 1 MiB array built
    into the library (grids up to 1024 x 1024; larger ones raise PSError with PS_EUNSUPPORTED), so neither the library
    nor this wrapper allocates: `d_out` (float32 [P][n_bins]) is therefore a required argument, not an optional one.
    The array is shared by every context on the device: do not let two of these calls overlap on the GPU.  Make the
    first call on a device outside any stream capture (it looks up the array's address)."""
    import torch
    _need(d_I, torch.float32, "d_I"); _need(d_out, torch.float32, "d_out")
    P, nb = int(d_I.shape[0]), int(d_I.shape[1])
    if tuple(d_out.shape) != (P, nb):
        raise ValueError(f"d_out must have shape ({P}, {nb})")
    ctx._check(ctx._lib.ps_spectrum_image_static(ctx._h, _ptr(d_I), P, nb, float(k_in), float(k_out), _ptr(d_out)))
    return d_out


def static_scratch_bytes() -> int:
    """Bytes (= pixels) of the built-in scratch array behind `ps_spectrum_image_static`."""
    return int(load_library().ps_static_scratch_bytes())


def ps_haadf(ctx: Context, d_exit, k_in: float, k_out: float = 0.0, d_out=None):
    """exit waves complex64 (dense [P][F][ny][nx] or tiled [P][ny][n_tiles][F][8]) -> float32 [P]: frame-averaged
    fraction of the beam on the annulus."""
    import torch
    _need(d_exit, torch.complex64, "d_exit")
    layout = _exit_layout(d_exit)
    P, F = int(d_exit.shape[0]), int(d_exit.shape[1] if layout == PS_LAYOUT_DENSE else d_exit.shape[3])
    if d_out is None:
        d_out = torch.empty((P,), dtype=torch.float32, device=ctx.device)
    ctx._check(ctx._lib.ps_haadf(ctx._h, _ptr(d_exit), layout, P, F, float(k_in), float(k_out), _ptr(d_out)))
    return d_out


def ps_accumulate_intensity(ctx: Context, d_acc, d_I, w_acc: float, w_new: float):
    """d_acc <- w_acc * d_acc + w_new * d_I (float32, same shape)."""
    import torch
    _need(d_acc, torch.float32, "d_acc"); _need(d_I, torch.float32, "d_I")
    assert d_acc.shape == d_I.shape
    ctx._check(ctx._lib.ps_accumulate_intensity(ctx._h, _ptr(d_acc), _ptr(d_I), d_I.numel(), float(w_acc), float(w_new)))
    return d_acc


def ps_dispersion(ctx: Context, d_I, kx, ky, d_out=None):
    import torch
    _need(d_I, torch.float32, "d_I")
    P, nb = int(d_I.shape[0]), int(d_I.shape[1])
    kxh, kxp = _host(kx, np.float64)
    kyh, kyp = _host(ky, np.float64)
    n_path = int(kxh.shape[0])
    d_pix = torch.empty((n_path,), dtype=torch.int32, device=ctx.device)
    if d_out is None:
        d_out = torch.empty((nb, n_path), dtype=torch.float32, device=ctx.device)
    ctx._check(ctx._lib.ps_dispersion(ctx._h, _ptr(d_I), P, nb, n_path, kxp, kyp, _ptr(d_pix), _ptr(d_out)))
    return d_out, d_pix


def ps_qbin(ctx: Context, d_I, dq: float, n_q: int, d_out=None):
    import torch
    _need(d_I, torch.float32, "d_I")
    P, nb = int(d_I.shape[0]), int(d_I.shape[1])
    d_qidx = torch.empty((ctx.ny, ctx.nx), dtype=torch.int32, device=ctx.device)
    if d_out is None:
        d_out = torch.empty((nb, int(n_q)), dtype=torch.float32, device=ctx.device)
    ctx._check(ctx._lib.ps_qbin(ctx._h, _ptr(d_I), P, nb, float(dq), int(n_q), _ptr(d_qidx), _ptr(d_out)))
    return d_out, d_qidx
