"""Shared helpers of the GPU parity tests (the CUDA path on one side, the float64 oracle on the other)."""
import numpy as np

from oracle import tacaw_oracle as O
from workloads import form_factor_coefficients


def rel_l2(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def make_ctx(w, device=0):
    """Context configured for workload `w` (geometry + surrogate form factors)."""
    import paper_2602_10064_b200 as ps
    ctx = ps.Context(device)
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    ctx.set_form_factors(w.elements, nl, ng, coef)
    ctx.set_geometry(w.cell, w.nx, w.ny, w.slice_dz)
    assert ctx.n_slices == w.n_slices
    return ctx


def oracle_potential(w, pos32_frame, slices=None):
    nl, ng, coef = form_factor_coefficients(w.elements, w.ff_kind)
    elem = np.searchsorted(w.elements, w.Z)
    return O.projected_potential(pos32_frame, elem, coef, nl, ng, w.cell, w.nx, w.ny, w.n_slices, slices=slices)


def oracle_incident(w):
    """list of float64 incident waves of workload w."""
    if w.beam == "plane":
        return [O.plane_wave(w.nx, w.ny)]
    if w.beam == "tilt":
        return [O.tilted_plane_wave(w.nx, w.ny, int(m), int(n)) for m, n in w.tilts]
    return [O.probe_wave(w.cell, w.nx, w.ny, w.kV, w.semi_angle_mrad, x, y) for x, y in w.probe_xy]


def gpu_incident(ctx, w):
    import paper_2602_10064_b200 as ps
    if w.beam == "plane":
        return ps.ps_make_incident(ctx, w.kV)
    if w.beam == "tilt":
        return ps.ps_make_incident(ctx, w.kV, 0.0, w.tilts.astype(np.float64), is_tilt=True)
    return ps.ps_make_incident(ctx, w.kV, w.semi_angle_mrad, w.probe_xy)
