"""Helpers of the GPU parity tests (tolerance of DESIGN.md G10, scene variations)."""
import copy

import numpy as np

RTOL = 1e-10          # BASELINE.json north_star: "within 1e-10 relative per pixel (fp64)"
ATOL_OF_MAX = 1e-14   # DESIGN.md G10: + 1e-14 * max(frame) for the far PSF wings / truncation edge


def frame_errors(G, O):
    G = np.asarray(G, dtype=np.float64)
    O = np.asarray(O, dtype=np.float64)
    mx = float(np.abs(O).max()) if O.size else 0.0
    err = np.abs(G - O)
    tol = RTOL * np.abs(O) + ATOL_OF_MAX * mx
    ratio = float((err / np.where(tol > 0, tol, 1.0)).max()) if O.size else 0.0
    core = np.abs(O) >= 1e-4 * mx if mx > 0 else np.zeros_like(O, dtype=bool)
    rel_core = float((err[core] / np.abs(O[core])).max()) if core.any() else 0.0
    return {"max_tol_ratio": ratio, "max_rel_core": rel_core, "max_abs_over_max": float(err.max() / mx) if mx > 0 else float(err.max() if O.size else 0.0)}


def assert_frame_parity(G, O, what=""):
    e = frame_errors(G, O)
    assert np.isfinite(np.asarray(G)).all(), f"{what}: non-finite GPU pixels"
    assert e["max_tol_ratio"] <= 1.0, f"{what}: GPU frame outside rtol 1e-10 + 1e-14*max: {e}"
    return e


def photocenter_x(frame, i0=0):
    frame = np.asarray(frame)
    cols = np.arange(frame.shape[1], dtype=np.float64) + i0
    tot = frame.sum()
    return float((frame.sum(axis=0) * cols).sum() / tot)


def photocenter_y(frame, j0=0):
    frame = np.asarray(frame)
    rows = np.arange(frame.shape[0], dtype=np.float64) + j0
    tot = frame.sum()
    return float((frame.sum(axis=1) * rows).sum() / tot)


def with_psf(scene, **kw):
    s = copy.copy(scene)
    s.psf = copy.copy(scene.psf)
    for k, v in kw.items():
        setattr(s.psf, k, v)
    return s
