"""paper_2602_10064_b200 — B200-native TACAW hot path (arxiv 2602.10064, "PySlice").

A thin ctypes binding over `libpyslice_b200.so` (hand-written CUDA for sm_100a behind the C ABI of
`include/pyslice_b200.h`).  The functions here only marshal arguments: torch tensors supply device
memory and the CUDA stream; every step of the path runs in the library's kernels.  There is no CPU
fallback: importing works without a GPU (so the symbols can be checked), but creating a `Context`
without the built library or without a CUDA device raises.
"""
from .binding import (Context, PSError, library_path, load_library, exported_symbols,  # noqa: F401
                      ps_build_slices, ps_make_incident, ps_multislice, ps_tacaw, ps_sdp,
                      ps_spectrum_image, ps_spectrum_image_static, static_scratch_bytes, ps_dispersion, ps_qbin, ps_haadf, ps_accumulate_intensity,
                      ps_exit_to_dense, ps_multislice_fused, exit_shape, PS_LAYOUT_DENSE, PS_LAYOUT_TILED_APERTURE)
