"""ctypes front-end of the CPU oracle (``oracle/e2e_oracle.c``, ``oracle/detector_oracle.c``).

TEST INFRASTRUCTURE ONLY: imported by ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py``.  The product package never imports it,
and this module never imports the product's CUDA binding: the two share only the seeded input
generators in ``paper_2008_05858_b200.workloads`` (which hold none of the method's arithmetic).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = [_HERE / "e2e_oracle.c", _HERE / "detector_oracle.c"]
_LIB = _HERE / "liboracle.so"


def build(force: bool = False) -> Path:
    """gcc -O2 -fopenmp -ffp-contract=off (no contraction: fma only where the source says fma)."""
    srcs = [s for s in _SRC if s.exists()]
    if not force and _LIB.exists() and all(_LIB.stat().st_mtime >= s.stat().st_mtime for s in srcs):
        return _LIB
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-o", str(_LIB)] + [str(s) for s in srcs] + ["-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


class _Format(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("n_orders", C.c_int32), ("n_fibers", C.c_int32),
                ("deg_l", C.c_int32), ("deg_m", C.c_int32),
                ("order_m", C.c_void_p), ("lam_min", C.c_void_p), ("lam_max", C.c_void_p),
                ("fiber_dx", C.c_void_p), ("fiber_dy", C.c_void_p),
                ("coef_x", C.c_void_p), ("coef_y", C.c_void_p),
                ("lam0", C.c_double), ("inv_dlam", C.c_double), ("m0", C.c_double), ("inv_dm", C.c_double),
                ("blaze_lam_c", C.c_void_p), ("blaze_amp", C.c_void_p),
                ("eff_table", C.c_void_p), ("eff_n", C.c_int64), ("eff_lam0", C.c_double), ("eff_dlam", C.c_double),
                ("samples_per_px", C.c_double)]


class _Psf(C.Structure):
    _fields_ = [("kind", C.c_int32), ("fiber_dx_px", C.c_double), ("fiber_dy_px", C.c_double),
                ("sigma_x", C.c_double), ("sigma_y", C.c_double), ("support_nsigma", C.c_double),
                ("n_nodes", C.c_int32), ("tab_npix", C.c_int32), ("tab_os", C.c_int32),
                ("tab_gx", C.c_int32), ("tab_gy", C.c_int32), ("tab", C.c_void_p),
                ("an_gx", C.c_int32), ("an_gy", C.c_int32), ("an_sigma_x", C.c_void_p), ("an_sigma_y", C.c_void_p)]


class _Spectrum(C.Structure):
    _fields_ = [("flux", C.c_void_p), ("n", C.c_int64), ("lam0", C.c_double), ("dlam", C.c_double),
                ("scale", C.c_double), ("doppler", C.c_double)]


class _Detector(C.Structure):
    _fields_ = [("gain", C.c_double), ("dark_e", C.c_double), ("ron_e", C.c_double), ("bias", C.c_double),
                ("seed", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.orc_order_nsamples.restype = C.c_int64
        L.orc_order_nsamples.argtypes = [C.c_void_p, C.c_int32]
        L.orc_samples.restype = None
        L.orc_samples.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int64] + [C.c_void_p] * 4
        L.orc_psf_pixel.restype = C.c_double
        L.orc_psf_pixel.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_psf_tab_pixel.restype = C.c_double
        L.orc_psf_tab_pixel.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_int32]
        L.orc_psf_map_pixel.restype = C.c_double
        L.orc_psf_map_pixel.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_int32]
        L.orc_footprint.restype = None
        L.orc_footprint.argtypes = [C.c_void_p, C.c_double, C.c_double] + [C.c_void_p] * 4
        L.orc_render.restype = C.c_int64
        L.orc_render.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                 C.c_void_p, C.c_int32]
        L.orc_total_weight.restype = C.c_double
        L.orc_total_weight.argtypes = [C.c_void_p, C.c_void_p]
        if hasattr(L, "orc_philox4x32_10"):
            L.orc_philox4x32_10.restype = None
            L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
            L.orc_detector.restype = None
            L.orc_detector.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
            L.orc_log.restype = C.c_double
            L.orc_log.argtypes = [C.c_double]
            L.orc_exp.restype = C.c_double
            L.orc_exp.argtypes = [C.c_double]
            L.orc_detector_draws.restype = None
            L.orc_detector_draws.argtypes = [C.c_void_p, C.c_uint64, C.c_double, C.c_void_p, C.c_void_p]
            L.orc_detector_ex.restype = C.c_int
            L.orc_detector_ex.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
            L.orc_log_series.restype = C.c_double
            L.orc_log_series.argtypes = [C.c_double]
            L.orc_sin2pi.restype = C.c_double
            L.orc_sin2pi.argtypes = [C.c_double]
            L.orc_gaussian_pair.restype = None
            L.orc_gaussian_pair.argtypes = [C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a):
    return a.ctypes.data if a is not None else None


class Handles:
    """Keeps numpy buffers alive next to the C structs that point into them."""

    def __init__(self, scene):
        self.keep = []
        s = scene

        def k(a, dt=np.float64):
            a = np.ascontiguousarray(np.asarray(a, dtype=dt))
            self.keep.append(a)
            return a.ctypes.data

        f = _Format()
        f.nx, f.ny, f.n_orders, f.n_fibers = s.nx, s.ny, s.n_orders, s.n_fibers
        f.deg_l, f.deg_m = s.deg_l, s.deg_m
        f.order_m = k(s.order_m, np.int32)
        f.lam_min, f.lam_max = k(s.lam_min), k(s.lam_max)
        f.fiber_dx, f.fiber_dy = k(s.fiber_dx), k(s.fiber_dy)
        f.coef_x, f.coef_y = k(s.coef_x), k(s.coef_y)
        f.lam0, f.inv_dlam, f.m0, f.inv_dm = s.lam0, s.inv_dlam, s.m0, s.inv_dm
        f.blaze_lam_c = k(s.blaze_lam_c)
        f.blaze_amp = k(s.blaze_amp) if s.blaze_amp is not None else None
        if s.eff_table is not None:
            f.eff_table, f.eff_n = k(s.eff_table), int(np.asarray(s.eff_table).shape[0])
            f.eff_lam0, f.eff_dlam = s.eff_lam0, s.eff_dlam
        else:
            f.eff_table, f.eff_n, f.eff_lam0, f.eff_dlam = None, 0, 0.0, 1.0
        f.samples_per_px = s.samples_per_px
        self.fmt = f

        p = _Psf()
        q = s.psf
        p.kind = q.kind
        p.fiber_dx_px, p.fiber_dy_px = q.fiber_dx_px, q.fiber_dy_px
        p.sigma_x, p.sigma_y, p.support_nsigma = q.sigma_x, q.sigma_y, q.support_nsigma
        p.n_nodes = 32                       # the oracle's own quadrature order, not the CUDA path's
        p.tab_npix, p.tab_os, p.tab_gx, p.tab_gy = q.tab_npix, q.tab_os, q.tab_gx, q.tab_gy
        p.tab = k(q.tab) if q.tab is not None else None
        if getattr(q, "an_sigma_x", None) is not None:      # G21 analytic PSF map
            p.an_gx, p.an_gy = int(q.an_gx), int(q.an_gy)
            p.an_sigma_x, p.an_sigma_y = k(q.an_sigma_x), k(q.an_sigma_y)
            assert np.asarray(q.an_sigma_x).size == p.an_gx * p.an_gy == np.asarray(q.an_sigma_y).size
        else:
            p.an_gx, p.an_gy, p.an_sigma_x, p.an_sigma_y = 0, 0, None, None
        self.psf = p

        arr = (_Spectrum * s.n_fibers)()
        for i, sp in enumerate(s.spectra):
            arr[i].flux = k(sp.flux)
            arr[i].n = int(np.asarray(sp.flux).shape[0])
            arr[i].lam0, arr[i].dlam, arr[i].scale, arr[i].doppler = sp.lam0, sp.dlam, sp.scale, sp.doppler
        self.spectra = arr


def order_nsamples(scene, order_idx: int) -> int:
    h = Handles(scene)
    return int(lib().orc_order_nsamples(C.addressof(h.fmt), order_idx))


def samples(scene, fiber: int, order_idx: int, k0: int = 0, k1: int | None = None):
    """(lam, x, y, w) of samples k0..k1 of one (fiber, order): steps a1-a3."""
    h = Handles(scene)
    n = int(lib().orc_order_nsamples(C.addressof(h.fmt), order_idx))
    if k1 is None:
        k1 = n
    m = max(0, k1 - k0)
    out = [np.zeros(m) for _ in range(4)]
    if m:
        lib().orc_samples(C.addressof(h.fmt), C.addressof(h.spectra[fiber]), fiber, order_idx, k0, k1,
                          *[o.ctypes.data for o in out])
    return tuple(out)


def psf_pixel(psf, u: float, v: float, n_nodes: int = 32) -> float:
    """P(u, v) of the analytic PSF (O4)."""
    p = _Psf()
    p.kind = 0
    p.fiber_dx_px, p.fiber_dy_px = psf.fiber_dx_px, psf.fiber_dy_px
    p.sigma_x, p.sigma_y, p.support_nsigma, p.n_nodes = psf.sigma_x, psf.sigma_y, psf.support_nsigma, n_nodes
    p.an_gx, p.an_gy, p.an_sigma_x, p.an_sigma_y = 0, 0, None, None
    return float(lib().orc_psf_pixel(C.addressof(p), u, v))


def psf_tab_pixel(scene, xk: float, yk: float, i: int, j: int) -> float:
    h = Handles(scene)
    return float(lib().orc_psf_tab_pixel(C.addressof(h.psf), scene.nx, scene.ny, xk, yk, i, j))


def psf_map_pixel(scene, xk: float, yk: float, i: int, j: int) -> float:
    """pixel (i, j) of the blended PSF of a sample at (xk, yk) for an analytic PSF map (G21)"""
    h = Handles(scene)
    return float(lib().orc_psf_map_pixel(C.addressof(h.psf), scene.nx, scene.ny, xk, yk, i, j))


def footprint(scene, xk: float, yk: float):
    h = Handles(scene)
    v = [C.c_int32() for _ in range(4)]
    lib().orc_footprint(C.addressof(h.psf), xk, yk, *[C.addressof(a) for a in v])
    return tuple(int(a.value) for a in v)


def render(scene, window=None, nthreads: int = 0) -> np.ndarray:
    """Steps a1-a5.  window = (i0, j0, wnx, wny) or None for the whole detector.  Returns [wny][wnx] float64."""
    h = Handles(scene)
    if window is None:
        window = (0, 0, scene.nx, scene.ny)
    i0, j0, wnx, wny = (int(v) for v in window)
    out = np.zeros((wny, wnx))
    r = lib().orc_render(C.addressof(h.fmt), C.addressof(h.psf), C.addressof(h.spectra), i0, j0, wnx, wny,
                         out.ctypes.data, nthreads)
    if r < 0:
        raise MemoryError("oracle render: allocation failed")
    render.last_touched = int(r)
    return out


def total_weight(scene) -> float:
    h = Handles(scene)
    return float(lib().orc_total_weight(C.addressof(h.fmt), C.addressof(h.spectra)))


# ---------------------------------------------------------------------------------------------
# detector stage (a6)
# ---------------------------------------------------------------------------------------------
def philox4x32_10(counter, key):
    c = np.ascontiguousarray(np.asarray(counter, dtype=np.uint32))
    k = np.ascontiguousarray(np.asarray(key, dtype=np.uint32))
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return o


def detector(frame: np.ndarray, det, pixel_offset: int = 0) -> np.ndarray:
    d = _Detector(det.gain, det.dark_e, det.ron_e, det.bias, det.seed)
    a = _f64(frame).reshape(-1)
    out = np.zeros_like(a)
    lib().orc_detector(a.ctypes.data, out.ctypes.data, a.shape[0], pixel_offset, C.addressof(d))
    return out.reshape(np.asarray(frame).shape)


class _DetectorEx(C.Structure):
    _fields_ = [("base", _Detector), ("prnu", C.c_void_p), ("dark", C.c_void_p),
                ("full_well", C.c_double), ("e_per_adu", C.c_double), ("adu_max", C.c_double),
                ("nx", C.c_int32), ("n_ports", C.c_int32), ("xtalk", C.c_void_p)]


def detector_ex(frame: np.ndarray, det, prnu=None, dark=None, full_well: float = 0.0, e_per_adu: float = 0.0,
                adu_max: float = 65535.0, pixel_offset: int = 0, xtalk=None) -> np.ndarray:
    """Full detector stage (detector_oracle.c orc_detector_ex): PRNU / dark maps, full-well saturation, ADC, and -- with
    xtalk = [n_ports][n_ports] coupling matrix on a 2-D frame -- cross-talk between the read-out ports (G20)."""
    a = _f64(frame).reshape(-1)
    pr = _f64(prnu).reshape(-1) if prnu is not None else None
    dk = _f64(dark).reshape(-1) if dark is not None else None
    assert pr is None or pr.shape == a.shape
    assert dk is None or dk.shape == a.shape
    xt, nx, n_ports = None, 0, 0
    if xtalk is not None:
        xt = _f64(xtalk)
        assert xt.ndim == 2 and xt.shape[0] == xt.shape[1] and np.asarray(frame).ndim == 2
        nx, n_ports = int(np.asarray(frame).shape[1]), int(xt.shape[0])
    d = _DetectorEx(_Detector(det.gain, det.dark_e, det.ron_e, det.bias, det.seed),
                    pr.ctypes.data if pr is not None else None, dk.ctypes.data if dk is not None else None,
                    float(full_well), float(e_per_adu), float(adu_max), nx, n_ports,
                    xt.ctypes.data if xt is not None else None)
    out = np.zeros_like(a)
    rc = lib().orc_detector_ex(a.ctypes.data, out.ctypes.data, a.shape[0], pixel_offset, C.addressof(d))
    if rc != 0:
        raise ValueError("oracle detector_ex: cross-talk needs whole rows and nx divisible by n_ports")
    return out.reshape(np.asarray(frame).shape)


def detector_adu16(frame: np.ndarray, det, **kw) -> np.ndarray:
    """ADC counts as uint16: detector_ex with e_per_adu > 0 and adu_max <= 65535, cast (the values are whole numbers)"""
    assert kw.get("e_per_adu", 0.0) > 0.0 and kw.get("adu_max", 65535.0) <= 65535.0
    return detector_ex(frame, det, **kw).astype(np.uint16)


def olog_series(x: float) -> float:
    return float(lib().orc_log_series(x))


def osin2pi(y: float) -> float:
    return float(lib().orc_sin2pi(y))


def gaussian_pairs(seed: int, n: int, pixel0: int = 0):
    z1, z2 = np.zeros(n), np.zeros(n)
    a, b = C.c_double(), C.c_double()
    L = lib()
    for p in range(n):
        L.orc_gaussian_pair(seed, pixel0 + p, C.byref(a), C.byref(b))
        z1[p], z2[p] = a.value, b.value
    return z1, z2


def olog(x: float) -> float:
    return float(lib().orc_log(x))


def oexp(x: float) -> float:
    return float(lib().orc_exp(x))


def cpu_threads() -> int:
    return os.cpu_count() or 1
