"""ctypes binding of ``libe2e.so`` (``include/e2e.h``): argument marshalling only.

Same names as the C entry points.  Every step of the hot path runs in the CUDA kernels of the library;
PyTorch supplies device memory (``torch.empty(..., device="cuda")``) and streams, nothing else.  There is
no CPU fallback: if the library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import List, Optional, Sequence

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libe2e.so"

E2E_OK = 0
ERROR_NAMES = {-1: "E2E_ERR_INVALID_ARG", -2: "E2E_ERR_NOT_MONOTONIC", -3: "E2E_ERR_CUDA", -4: "E2E_ERR_NOMEM",
               -5: "E2E_ERR_UNSUPPORTED", -6: "E2E_ERR_WORKSPACE"}

# every symbol include/e2e.h declares (tests/test_abi.py checks the header against this list and the .so)
SYMBOLS = ["e2e_last_error", "e2e_version", "e2e_format_create", "e2e_format_destroy", "e2e_format_num_samples",
           "e2e_psf_create", "e2e_psf_destroy", "e2e_psf_info", "e2e_render_workspace_bytes", "e2e_setup_samples", "e2e_render_frame",
           "e2e_render_host_workspace_bytes", "e2e_render_frame_host", "e2e_apply_detector", "e2e_apply_detector_ex",
           "e2e_apply_detector_adu16", "e2e_measure_fp64_peak",
           "e2e_launch_count", "e2e_profile_enable", "e2e_profile_read", "e2e_render_kernel_info",
           "e2e_render_algorithmic_fma", "e2e_render_frames_workspace_bytes", "e2e_render_frames",
           "e2e_render_frame_host_ex", "e2e_render_frame_host_adu16", "e2e_plan_check", "e2e_spectrograph_format", "e2e_probe_fp64_pipe",
           "e2e_render_frame_noalloc"]


class E2EError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{ERROR_NAMES.get(code, code)}: {msg}")
        self.code = code


class FormatDesc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("n_orders", C.c_int32), ("order_m", C.c_void_p),
                ("lam_min", C.c_void_p), ("lam_max", C.c_void_p), ("n_fibers", C.c_int32),
                ("fiber_dx", C.c_void_p), ("fiber_dy", C.c_void_p), ("deg_l", C.c_int32), ("deg_m", C.c_int32),
                ("coef_x", C.c_void_p), ("coef_y", C.c_void_p), ("lam0", C.c_double), ("inv_dlam", C.c_double),
                ("m0", C.c_double), ("inv_dm", C.c_double), ("blaze_lam_c", C.c_void_p), ("blaze_amp", C.c_void_p),
                ("eff_table", C.c_void_p), ("eff_n", C.c_int64), ("eff_lam0", C.c_double), ("eff_dlam", C.c_double),
                ("samples_per_px", C.c_double)]


class PsfDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("fiber_dx_px", C.c_double), ("fiber_dy_px", C.c_double),
                ("sigma_x", C.c_double), ("sigma_y", C.c_double), ("support_nsigma", C.c_double),
                ("n_nodes", C.c_int32), ("tab_npix", C.c_int32), ("tab_os", C.c_int32), ("tab_gx", C.c_int32),
                ("tab_gy", C.c_int32), ("tab", C.c_void_p), ("an_gx", C.c_int32), ("an_gy", C.c_int32),
                ("an_sigma_x", C.c_void_p), ("an_sigma_y", C.c_void_p)]


class SpectrumDesc(C.Structure):
    _fields_ = [("d_flux", C.c_void_p), ("n", C.c_int64), ("lam0", C.c_double), ("dlam", C.c_double),
                ("scale", C.c_double), ("doppler", C.c_double)]


class ProfileDesc(C.Structure):
    _fields_ = [("ms_zero", C.c_double), ("ms_setup", C.c_double), ("ms_render", C.c_double), ("ms_detector", C.c_double),
                ("n_setup", C.c_int64), ("n_render", C.c_int64), ("n_detector", C.c_int64), ("n_calls", C.c_int64)]


class DetectorDesc(C.Structure):
    _fields_ = [("gain", C.c_double), ("dark_e", C.c_double), ("ron_e", C.c_double), ("bias", C.c_double),
                ("seed", C.c_uint64)]


class DetectorExDesc(C.Structure):
    _fields_ = [("base", DetectorDesc), ("d_prnu", C.c_void_p), ("d_dark", C.c_void_p), ("full_well_e", C.c_double),
                ("e_per_adu", C.c_double), ("adu_max", C.c_double), ("n_ports", C.c_int32), ("xtalk", C.c_void_p)]


class SpectrographDesc(C.Structure):
    _fields_ = [("groove_um", C.c_double), ("blaze_deg", C.c_double), ("theta_deg", C.c_double), ("gamma_deg", C.c_double),
                ("xd_groove_um", C.c_double), ("xd_lam_ref", C.c_double), ("f_cam_mm", C.c_double), ("f_coll_mm", C.c_double),
                ("pixel_um", C.c_double), ("fiber_core_um", C.c_double), ("m_lo", C.c_int32), ("m_hi", C.c_int32),
                ("x_c", C.c_double), ("y_c", C.c_double), ("n_fibers", C.c_int32), ("fiber_height_um", C.c_void_p)]


class SpectrographFormatDesc(C.Structure):
    _fields_ = [("capacity_orders", C.c_int32), ("n_orders", C.c_int32), ("deg_l", C.c_int32), ("deg_m", C.c_int32),
                ("order_m", C.c_void_p), ("lam_min", C.c_void_p), ("lam_max", C.c_void_p), ("blaze_lam_c", C.c_void_p),
                ("blaze_amp", C.c_void_p), ("coef_x", C.c_void_p), ("coef_y", C.c_void_p), ("lam0", C.c_double),
                ("inv_dlam", C.c_double), ("m0", C.c_double), ("inv_dm", C.c_double), ("fiber_dx", C.c_void_p),
                ("fiber_dy", C.c_void_p), ("fiber_dx_px", C.c_double), ("fiber_dy_px", C.c_double),
                ("residual_x_px", C.c_double), ("residual_y_px", C.c_double), ("x_min", C.c_double), ("x_max", C.c_double),
                ("y_min", C.c_double), ("y_max", C.c_double), ("tilt_tan", C.c_double), ("K", C.c_double),
                ("px_per_radian", C.c_double)]


class PlanCheckDesc(C.Structure):
    _fields_ = [("n_items", C.c_int64), ("n_phases", C.c_int64), ("n_dependencies", C.c_int64), ("claimed_px", C.c_int64),
                ("phase_conflicts", C.c_int64), ("queue_conflicts", C.c_int64), ("device_band_conflicts", C.c_int64),
                ("host_band_conflicts", C.c_int64), ("host_rows_not_final", C.c_int64), ("n_host_bands", C.c_int32),
                ("n_device_bands", C.c_int32)]


_lib = None


def load():
    """dlopen libe2e.so (built in-tree by ``paper_2008_05858_b200.build``); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2008_05858_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.e2e_last_error.restype = C.c_char_p
    L.e2e_last_error.argtypes = []
    L.e2e_version.restype = C.c_char_p
    L.e2e_version.argtypes = []
    L.e2e_format_create.restype = C.c_int
    L.e2e_format_create.argtypes = [C.POINTER(vp), C.POINTER(FormatDesc)]
    L.e2e_format_destroy.restype = None
    L.e2e_format_destroy.argtypes = [vp]
    L.e2e_format_num_samples.restype = C.c_int
    L.e2e_format_num_samples.argtypes = [vp, vp, C.POINTER(i64)]
    L.e2e_psf_create.restype = C.c_int
    L.e2e_psf_create.argtypes = [C.POINTER(vp), C.POINTER(PsfDesc), i32, i32]
    L.e2e_psf_destroy.restype = None
    L.e2e_psf_destroy.argtypes = [vp]
    L.e2e_psf_info.restype = C.c_int
    L.e2e_psf_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
    L.e2e_render_workspace_bytes.restype = C.c_int
    L.e2e_render_workspace_bytes.argtypes = [vp, vp, C.POINTER(C.c_size_t)]
    L.e2e_setup_samples.restype = C.c_int
    L.e2e_setup_samples.argtypes = [vp, C.POINTER(SpectrumDesc), i32, i32, vp, vp, vp, vp, i64, vp]
    L.e2e_render_frame.restype = C.c_int
    L.e2e_render_frame.argtypes = [vp, vp, C.POINTER(SpectrumDesc), vp, i32, vp, C.c_size_t, vp]
    L.e2e_render_frame_noalloc.restype = C.c_int
    L.e2e_render_frame_noalloc.argtypes = [vp, vp, C.POINTER(SpectrumDesc), vp, i32, vp]
    L.e2e_render_host_workspace_bytes.restype = C.c_int
    L.e2e_render_host_workspace_bytes.argtypes = [vp, vp, C.POINTER(SpectrumDesc), C.POINTER(C.c_size_t)]
    L.e2e_render_frame_host.restype = C.c_int
    L.e2e_render_frame_host.argtypes = [vp, vp, C.POINTER(SpectrumDesc), C.POINTER(DetectorDesc), vp, vp, C.c_size_t, vp]
    L.e2e_render_frame_host_ex.restype = C.c_int
    L.e2e_render_frame_host_ex.argtypes = [vp, vp, C.POINTER(SpectrumDesc), C.POINTER(DetectorExDesc), vp, vp, C.c_size_t, vp]
    L.e2e_render_frame_host_adu16.restype = C.c_int
    L.e2e_render_frame_host_adu16.argtypes = [vp, vp, C.POINTER(SpectrumDesc), C.POINTER(DetectorExDesc), vp, vp, C.c_size_t, vp]
    L.e2e_plan_check.restype = C.c_int
    L.e2e_plan_check.argtypes = [vp, vp, C.POINTER(PlanCheckDesc)]
    L.e2e_spectrograph_format.restype = C.c_int
    L.e2e_spectrograph_format.argtypes = [C.POINTER(SpectrographDesc), C.POINTER(SpectrographFormatDesc)]
    L.e2e_apply_detector.restype = C.c_int
    L.e2e_apply_detector.argtypes = [vp, vp, i32, i32, C.POINTER(DetectorDesc), vp]
    L.e2e_apply_detector_ex.restype = C.c_int
    L.e2e_apply_detector_ex.argtypes = [vp, vp, i32, i32, C.POINTER(DetectorExDesc), vp]
    L.e2e_apply_detector_adu16.restype = C.c_int
    L.e2e_apply_detector_adu16.argtypes = [vp, vp, i32, i32, C.POINTER(DetectorExDesc), vp]
    L.e2e_measure_fp64_peak.restype = C.c_int
    L.e2e_measure_fp64_peak.argtypes = [i32, C.POINTER(dbl), C.POINTER(dbl)]
    L.e2e_probe_fp64_pipe.restype = C.c_int
    L.e2e_probe_fp64_pipe.argtypes = [C.POINTER(dbl)]
    L.e2e_render_kernel_info.restype = C.c_int
    L.e2e_render_kernel_info.argtypes = [vp, vp, C.POINTER(C.c_char_p), C.POINTER(dbl), C.POINTER(dbl)]
    L.e2e_render_frames_workspace_bytes.restype = C.c_int
    L.e2e_render_frames_workspace_bytes.argtypes = [vp, vp, i32, C.POINTER(C.c_size_t)]
    L.e2e_render_frames.restype = C.c_int
    L.e2e_render_frames.argtypes = [vp, vp, i32, vp, vp, i32, vp, C.c_size_t, vp]
    L.e2e_render_algorithmic_fma.restype = C.c_int
    L.e2e_render_algorithmic_fma.argtypes = [vp, vp, C.POINTER(dbl), C.POINTER(dbl)]
    L.e2e_launch_count.restype = i64
    L.e2e_launch_count.argtypes = []
    L.e2e_profile_enable.restype = C.c_int
    L.e2e_profile_enable.argtypes = [i32]
    L.e2e_profile_read.restype = C.c_int
    L.e2e_profile_read.argtypes = [C.POINTER(ProfileDesc), i32]
    _lib = L
    return L


def _check(rc: int):
    if rc != E2E_OK:
        raise E2EError(rc, load().e2e_last_error().decode())


def e2e_version() -> str:
    return load().e2e_version().decode()


def e2e_last_error() -> str:
    return load().e2e_last_error().decode()


def e2e_launch_count() -> int:
    return int(load().e2e_launch_count())


def _host(a, dt=np.float64):
    return np.ascontiguousarray(np.asarray(a, dtype=dt))


class Format:
    """Owns an ``e2e_format_t*``.  Built from a scene-like object (see ``workloads.Scene``)."""

    def __init__(self, scene):
        s = scene
        keep = []

        def k(a, dt=np.float64):
            a = _host(a, dt)
            keep.append(a)
            return a.ctypes.data

        d = FormatDesc()
        d.nx, d.ny = int(s.nx), int(s.ny)
        d.n_orders = int(np.asarray(s.order_m).shape[0])
        d.order_m = k(s.order_m, np.int32)
        d.lam_min, d.lam_max = k(s.lam_min), k(s.lam_max)
        d.n_fibers = int(np.asarray(s.fiber_dx).shape[0])
        d.fiber_dx, d.fiber_dy = k(s.fiber_dx), k(s.fiber_dy)
        d.deg_l, d.deg_m = int(s.deg_l), int(s.deg_m)
        d.coef_x, d.coef_y = k(s.coef_x), k(s.coef_y)
        d.lam0, d.inv_dlam, d.m0, d.inv_dm = float(s.lam0), float(s.inv_dlam), float(s.m0), float(s.inv_dm)
        d.blaze_lam_c = k(s.blaze_lam_c)
        d.blaze_amp = k(s.blaze_amp) if getattr(s, "blaze_amp", None) is not None else None
        if getattr(s, "eff_table", None) is not None:
            d.eff_table = k(s.eff_table)
            d.eff_n = int(np.asarray(s.eff_table).shape[0])
            d.eff_lam0, d.eff_dlam = float(s.eff_lam0), float(s.eff_dlam)
        else:
            d.eff_table, d.eff_n, d.eff_lam0, d.eff_dlam = None, 0, 0.0, 1.0
        d.samples_per_px = float(s.samples_per_px)
        self.nx, self.ny, self.n_orders, self.n_fibers = d.nx, d.ny, d.n_orders, d.n_fibers
        self.handle = C.c_void_p()
        _check(load().e2e_format_create(C.byref(self.handle), C.byref(d)))

    def num_samples(self):
        per = np.zeros(self.n_orders, dtype=np.int64)
        tot = C.c_int64()
        _check(load().e2e_format_num_samples(self.handle, per.ctypes.data, C.byref(tot)))
        return per, int(tot.value)

    def close(self):
        if getattr(self, "handle", None) is not None and self.handle.value:
            load().e2e_format_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Psf:
    """Owns an ``e2e_psf_t*``.  ``psf`` is a ``workloads.Psf``-like object."""

    def __init__(self, psf, nx: int, ny: int):
        d = PsfDesc()
        d.kind = int(psf.kind)
        d.fiber_dx_px, d.fiber_dy_px = float(psf.fiber_dx_px), float(psf.fiber_dy_px)
        d.sigma_x, d.sigma_y = float(psf.sigma_x), float(psf.sigma_y)
        d.support_nsigma = float(psf.support_nsigma)
        d.n_nodes = int(psf.n_nodes)
        d.tab_npix, d.tab_os, d.tab_gx, d.tab_gy = int(psf.tab_npix), int(psf.tab_os), int(psf.tab_gx), int(psf.tab_gy)
        tab = _host(psf.tab) if psf.tab is not None else None
        d.tab = tab.ctypes.data if tab is not None else None
        sx = _host(psf.an_sigma_x) if getattr(psf, "an_sigma_x", None) is not None else None
        sy = _host(psf.an_sigma_y) if getattr(psf, "an_sigma_y", None) is not None else None
        d.an_gx, d.an_gy = (int(psf.an_gx), int(psf.an_gy)) if sx is not None else (0, 0)
        d.an_sigma_x = sx.ctypes.data if sx is not None else None
        d.an_sigma_y = sy.ctypes.data if sy is not None else None
        self.handle = C.c_void_p()
        _check(load().e2e_psf_create(C.byref(self.handle), C.byref(d), int(nx), int(ny)))

    def info(self):
        q, c, r = C.c_int32(), C.c_int32(), C.c_int32()
        _check(load().e2e_psf_info(self.handle, C.byref(q), C.byref(c), C.byref(r)))
        return {"n_nodes": int(q.value), "footprint_cols": int(c.value), "footprint_rows": int(r.value)}

    def close(self):
        if getattr(self, "handle", None) is not None and self.handle.value:
            load().e2e_psf_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def e2e_format_create(scene) -> Format:
    return Format(scene)


def e2e_psf_create(psf, nx: int, ny: int) -> Psf:
    return Psf(psf, nx, ny)


def spectra_array(spectra: Sequence, flux_ptrs: Sequence[int]):
    """``e2e_spectrum_t[n_fibers]`` from ``workloads.Spectrum``-like objects and the addresses of their tables."""
    arr = (SpectrumDesc * len(spectra))()
    for i, (sp, ptr) in enumerate(zip(spectra, flux_ptrs)):
        arr[i].d_flux = int(ptr)
        arr[i].n = int(np.asarray(sp.flux).shape[0]) if not hasattr(sp.flux, "numel") else int(sp.flux.numel())
        arr[i].lam0, arr[i].dlam, arr[i].scale, arr[i].doppler = float(sp.lam0), float(sp.dlam), float(sp.scale), float(sp.doppler)
    return arr


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    return int(getattr(stream, "cuda_stream", stream))


def e2e_render_workspace_bytes(fmt: Format, psf: Psf) -> int:
    n = C.c_size_t()
    _check(load().e2e_render_workspace_bytes(fmt.handle, psf.handle, C.byref(n)))
    return int(n.value)


def e2e_setup_samples(fmt: Format, spectrum_desc, fiber: int, order_index: int, d_lam, d_x, d_y, d_w, capacity: int,
                      stream=None):
    def p(t):
        return None if t is None else int(t.data_ptr())
    _check(load().e2e_setup_samples(fmt.handle, C.byref(spectrum_desc), fiber, order_index, p(d_lam), p(d_x), p(d_y),
                                    p(d_w), int(capacity), _stream_ptr(stream)))


def e2e_render_frame(fmt: Format, psf: Psf, spectra_desc, d_frame, accumulate: bool, d_workspace, stream=None):
    """d_frame: float64 CUDA tensor [ny, nx]; d_workspace: uint8 CUDA tensor of e2e_render_workspace_bytes bytes."""
    _check(load().e2e_render_frame(fmt.handle, psf.handle, spectra_desc, int(d_frame.data_ptr()), int(bool(accumulate)),
                                   int(d_workspace.data_ptr()), int(d_workspace.numel() * d_workspace.element_size()),
                                   _stream_ptr(stream)))


NOALLOC_SCRATCH_BYTES = 32 << 20   # E2E_NOALLOC_SCRATCH_BYTES of include/e2e.h


def e2e_render_frame_noalloc(fmt: Format, psf: Psf, spectra_desc, d_frame, accumulate: bool, stream=None):
    """e2e_render_frame with the scratch in the library's static device array (no workspace, no allocation)."""
    _check(load().e2e_render_frame_noalloc(fmt.handle, psf.handle, spectra_desc, int(d_frame.data_ptr()), int(bool(accumulate)),
                                           _stream_ptr(stream)))


def e2e_render_frames_workspace_bytes(fmt: Format, psf: Psf, n_frames: int) -> int:
    n = C.c_size_t()
    _check(load().e2e_render_frames_workspace_bytes(fmt.handle, psf.handle, int(n_frames), C.byref(n)))
    return int(n.value)


def e2e_render_frames(fmt: Format, psf: Psf, spectra_descs: Sequence, d_frames: Sequence, accumulate: bool, d_workspace, stream=None):
    """batch render on fixed geometry: spectra_descs = one spectra_array per frame, d_frames = one CUDA tensor per frame"""
    nfr = len(d_frames)
    nfib = len(spectra_descs[0])
    flat = (SpectrumDesc * (nfr * nfib))()
    for b, desc in enumerate(spectra_descs):
        for f in range(nfib):
            C.memmove(C.byref(flat, (b * nfib + f) * C.sizeof(SpectrumDesc)), C.byref(desc, f * C.sizeof(SpectrumDesc)),
                      C.sizeof(SpectrumDesc))
    ptrs = (C.c_void_p * nfr)(*[int(t.data_ptr()) for t in d_frames])
    _check(load().e2e_render_frames(fmt.handle, psf.handle, nfr, flat, ptrs, int(bool(accumulate)), int(d_workspace.data_ptr()),
                                    int(d_workspace.numel() * d_workspace.element_size()), _stream_ptr(stream)))


def e2e_render_host_workspace_bytes(fmt: Format, psf: Psf, spectra_desc) -> int:
    n = C.c_size_t()
    _check(load().e2e_render_host_workspace_bytes(fmt.handle, psf.handle, spectra_desc, C.byref(n)))
    return int(n.value)


def e2e_render_frame_host(fmt: Format, psf: Psf, spectra_desc, h_frame_ptr: int, d_workspace, det=None, stream=None):
    """spectra_desc[f].d_flux are HOST addresses, h_frame_ptr a HOST address (pinned for full PCIe speed)."""
    d = None
    if det is not None:
        d = C.byref(DetectorDesc(float(det.gain), float(det.dark_e), float(det.ron_e), float(det.bias), int(det.seed)))
    _check(load().e2e_render_frame_host(fmt.handle, psf.handle, spectra_desc, d, int(h_frame_ptr), int(d_workspace.data_ptr()),
                                        int(d_workspace.numel() * d_workspace.element_size()), _stream_ptr(stream)))


def e2e_render_frame_host_ex(fmt: Format, psf: Psf, spectra_desc, h_frame_ptr: int, d_workspace, det_ex_desc, stream=None,
                             adu16: bool = False):
    """host path with the full detector stage; det_ex_desc from detector_ex_desc(); adu16: h_frame_ptr is a uint16 array"""
    fn = load().e2e_render_frame_host_adu16 if adu16 else load().e2e_render_frame_host_ex
    _check(fn(fmt.handle, psf.handle, spectra_desc, C.byref(det_ex_desc), int(h_frame_ptr), int(d_workspace.data_ptr()),
              int(d_workspace.numel() * d_workspace.element_size()), _stream_ptr(stream)))


def e2e_spectrograph_format(groove_um: float, blaze_deg: float, theta_deg: float, gamma_deg: float, xd_groove_um: float,
                            xd_lam_ref: float, f_cam_mm: float, f_coll_mm: float, pixel_um: float, fiber_core_um: float,
                            m_lo: int, m_hi: int, x_c: float, y_c: float, fiber_height_um: Sequence[float] = (0.0,)) -> dict:
    """parametric Spectrograph Unit (e2e.h): the arrays of a spectral format from the geometrical parameters of a
    cross-dispersed echelle spectrograph.  Host call, needs no GPU.  Returns a dict of numpy arrays / floats."""
    n = int(m_hi) - int(m_lo) + 1
    hf = _host(fiber_height_um)
    d = SpectrographDesc(groove_um, blaze_deg, theta_deg, gamma_deg, xd_groove_um, xd_lam_ref, f_cam_mm, f_coll_mm, pixel_um,
                         fiber_core_um, int(m_lo), int(m_hi), x_c, y_c, int(hf.shape[0]), hf.ctypes.data)
    arr = {"order_m": np.zeros(max(n, 1), dtype=np.int32)}
    for k in ("lam_min", "lam_max", "blaze_lam_c", "blaze_amp"):
        arr[k] = np.zeros(max(n, 1))
    arr["coef_x"], arr["coef_y"] = np.zeros(36), np.zeros(36)
    arr["fiber_dx"], arr["fiber_dy"] = np.zeros(hf.shape[0]), np.zeros(hf.shape[0])
    o = SpectrographFormatDesc()
    o.capacity_orders = max(n, 1)
    for k, a in arr.items():
        setattr(o, k, a.ctypes.data)
    _check(load().e2e_spectrograph_format(C.byref(d), C.byref(o)))
    res = {k: a[:o.n_orders] if k in ("order_m", "lam_min", "lam_max", "blaze_lam_c", "blaze_amp") else a for k, a in arr.items()}
    for k in ("n_orders", "deg_l", "deg_m", "lam0", "inv_dlam", "m0", "inv_dm", "fiber_dx_px", "fiber_dy_px", "residual_x_px",
              "residual_y_px", "x_min", "x_max", "y_min", "y_max", "tilt_tan", "K", "px_per_radian"):
        res[k] = getattr(o, k)
    return res


def e2e_plan_check(fmt: Format, psf: Psf) -> dict:
    """device-side check of the schedule invariants (test hook): every *_conflicts / host_rows_not_final must be 0"""
    d = PlanCheckDesc()
    _check(load().e2e_plan_check(fmt.handle, psf.handle, C.byref(d)))
    return {k: int(getattr(d, k)) for k, _ in PlanCheckDesc._fields_}


def e2e_apply_detector(d_in, d_out, nx: int, ny: int, det, stream=None):
    d = DetectorDesc(float(det.gain), float(det.dark_e), float(det.ron_e), float(det.bias), int(det.seed))
    _check(load().e2e_apply_detector(int(d_in.data_ptr()), int(d_out.data_ptr()), int(nx), int(ny), C.byref(d),
                                     _stream_ptr(stream)))


def detector_ex_desc(det, d_prnu=None, d_dark=None, full_well_e: float = 0.0, e_per_adu: float = 0.0,
                     adu_max: float = 65535.0, xtalk=None):
    """``e2e_detector_ex_t`` (+ the host array the xtalk pointer refers to, which the caller must keep alive)"""
    xt = _host(xtalk) if xtalk is not None else None
    d = DetectorExDesc(DetectorDesc(float(det.gain), float(det.dark_e), float(det.ron_e), float(det.bias), int(det.seed)),
                       int(d_prnu.data_ptr()) if d_prnu is not None else None,
                       int(d_dark.data_ptr()) if d_dark is not None else None,
                       float(full_well_e), float(e_per_adu), float(adu_max),
                       int(xt.shape[0]) if xt is not None else 0, xt.ctypes.data if xt is not None else None)
    return d, xt


def e2e_apply_detector_ex(d_in, d_out, nx: int, ny: int, det, d_prnu=None, d_dark=None, full_well_e: float = 0.0,
                          e_per_adu: float = 0.0, adu_max: float = 65535.0, xtalk=None, stream=None):
    """full detector stage (e2e.h): d_prnu / d_dark are device tensors [ny*nx] or None, xtalk a host [n_ports][n_ports] array"""
    d, keep = detector_ex_desc(det, d_prnu, d_dark, full_well_e, e_per_adu, adu_max, xtalk)
    _check(load().e2e_apply_detector_ex(int(d_in.data_ptr()), int(d_out.data_ptr()), int(nx), int(ny), C.byref(d),
                                        _stream_ptr(stream)))


def e2e_apply_detector_adu16(d_in, d_out_u16, nx: int, ny: int, det, d_prnu=None, d_dark=None, full_well_e: float = 0.0,
                             e_per_adu: float = 1.0, adu_max: float = 65535.0, xtalk=None, stream=None):
    """the same stage with uint16 ADC counts (d_out_u16: uint16 device tensor [ny*nx])"""
    d, keep = detector_ex_desc(det, d_prnu, d_dark, full_well_e, e_per_adu, adu_max, xtalk)
    _check(load().e2e_apply_detector_adu16(int(d_in.data_ptr()), int(d_out_u16.data_ptr()), int(nx), int(ny), C.byref(d),
                                           _stream_ptr(stream)))


def e2e_measure_fp64_peak(repeats: int = 60):
    """(burst, sustained) DFMA/s of independent fp64 FMA chains on every SM."""
    burst, sus = C.c_double(), C.c_double()
    _check(load().e2e_measure_fp64_peak(int(repeats), C.byref(burst), C.byref(sus)))
    return float(burst.value), float(sus.value)


def e2e_probe_fp64_pipe() -> dict:
    """probes of one SM's FP64 pipe (e2e.h): DMMA latency / issue interval, DMMA and scalar DFMA rates alone and mixed"""
    r = (C.c_double * 6)()
    _check(load().e2e_probe_fp64_pipe(r))
    return {"dmma_cycles_dependent_chain": r[0], "dmma_cycles_two_chains": r[1], "dmma_per_clk_sm_alone": r[2],
            "dfma_per_clk_sm_alone": r[3], "dfma_per_clk_sm_next_to_dmma": r[4], "dmma_per_clk_sm_in_mix": r[5]}


def e2e_render_kernel_info(fmt, psf) -> dict:
    """name of the a4+a5 kernel e2e_render_frame launches for (fmt, psf) and the fp64 FMAs it issues per cell / sample"""
    name, pc, ps = C.c_char_p(), C.c_double(), C.c_double()
    _check(load().e2e_render_kernel_info(fmt.handle, psf.handle, C.byref(name), C.byref(pc), C.byref(ps)))
    return {"name": name.value.decode(), "executed_fma_per_cell": float(pc.value), "executed_fma_per_sample": float(ps.value)}


def e2e_render_algorithmic_fma(fmt, psf) -> dict:
    """un-padded fp64 FMAs of the cell-moment method per footprint cell / per sample (0 for the other kernels)"""
    pc, ps = C.c_double(), C.c_double()
    _check(load().e2e_render_algorithmic_fma(fmt.handle, psf.handle, C.byref(pc), C.byref(ps)))
    return {"fma_per_cell": float(pc.value), "fma_per_sample": float(ps.value)}


def e2e_profile_enable(on: bool):
    _check(load().e2e_profile_enable(int(bool(on))))


def e2e_profile_read(reset: bool = True) -> dict:
    p = ProfileDesc()
    _check(load().e2e_profile_read(C.byref(p), int(bool(reset))))
    return {k: getattr(p, k) for k, _ in ProfileDesc._fields_}


# ---------------------------------------------------------------------------------------------------------
# convenience on top of the calls above (still marshalling only): a scene rendered with torch-owned buffers
# ---------------------------------------------------------------------------------------------------------
class Renderer:
    """Holds the handles, the device copies of the spectra and the workspace of one scene."""

    def __init__(self, scene, device="cuda:0"):
        import torch
        self.torch = torch
        self.scene = scene
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.fmt = Format(scene)
        self.psf = Psf(scene.psf, scene.nx, scene.ny)
        self.flux = [torch.from_numpy(_host(sp.flux)).to(self.device) for sp in scene.spectra]
        self.spectra = spectra_array(scene.spectra, [t.data_ptr() for t in self.flux])
        nbytes = e2e_render_workspace_bytes(self.fmt, self.psf)
        self.workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=self.device)
        self.per_order, self.n_samples = self.fmt.num_samples()

    def render(self, frame=None, accumulate=False, stream=None):
        torch = self.torch
        if frame is None:
            frame = torch.empty((self.scene.ny, self.scene.nx), dtype=torch.float64, device=self.device)
        e2e_render_frame(self.fmt, self.psf, self.spectra, frame, accumulate, self.workspace, stream)
        return frame

    def samples(self, fiber: int, order_index: int):
        torch = self.torch
        n = int(self.per_order[order_index])
        out = [torch.empty(max(n, 1), dtype=torch.float64, device=self.device) for _ in range(4)]
        e2e_setup_samples(self.fmt, self.spectra[fiber], fiber, order_index, *out, capacity=max(n, 1))
        torch.cuda.synchronize()
        return tuple(o[:n].cpu().numpy() for o in out)

    def detector(self, frame, det=None, out=None, stream=None):
        det = det if det is not None else self.scene.detector
        out = out if out is not None else self.torch.empty_like(frame)
        e2e_apply_detector(frame, out, self.scene.nx, self.scene.ny, det, stream)
        return out

    def close(self):
        self.psf.close()
        self.fmt.close()
