"""Seeded synthetic workloads (input arrays only).

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the CUDA
path: it produces *inputs* -- spectra tables, spectral-format polynomial
coefficients, blaze parameters, PSF descriptors, tabulated PSF kernels -- and holds
none of the method's arithmetic (no wavelength->pixel mapping, no PSF integration,
no accumulation, no noise).  Recipes follow SURVEY.md section 8(d); they stand in
for the paper's ESPRESSO and ELT-HIRES workloads, whose
real spectra, Zemax spectral formats and PSF maps are not available.

All randomness is ``numpy.random.default_rng(seed)``.
"""
from __future__ import annotations

import copy
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

C_LIGHT = 299_792_458.0  # m/s


@dataclass
class Spectrum:
    """Uniform-grid photon-flux table for one fiber."""
    flux: np.ndarray            # float64 [n]
    lam0: float                 # wavelength of flux[0]  (Angstrom)
    dlam: float                 # grid step
    scale: float = 1.0          # per-fiber illumination
    doppler: float = 1.0        # 1 + v/c, S'(lam) = S(lam / doppler)


@dataclass
class Psf:
    kind: int = 0               # 0 analytic (ellipse (x) gaussian), 1 tabulated
    fiber_dx_px: float = 0.0    # full widths of the geometric fiber image
    fiber_dy_px: float = 0.0
    sigma_x: float = 1.0        # optical PSF, axis-aligned gaussian
    sigma_y: float = 1.0
    support_nsigma: float = 7.5
    n_nodes: int = 0            # chord quadrature nodes for the CUDA path (0 = library default)
    tab_npix: int = 0
    tab_os: int = 0
    tab_gx: int = 0
    tab_gy: int = 0
    tab: Optional[np.ndarray] = None   # float64 [gy][gx][npix*os][npix*os]
    # analytic PSF map (G21; "PSF ... for each wavelength"): sigma_x, sigma_y at the nodes of an
    # an_gx x an_gy grid over the detector; None = one PSF for the whole frame (sigma_x, sigma_y above)
    an_gx: int = 0
    an_gy: int = 0
    an_sigma_x: Optional[np.ndarray] = None   # float64 [an_gy][an_gx]
    an_sigma_y: Optional[np.ndarray] = None


@dataclass
class Detector:
    gain: float = 1.0
    dark_e: float = 0.0
    ron_e: float = 0.0
    bias: float = 0.0
    seed: int = 0


@dataclass
class Scene:
    name: str
    nx: int
    ny: int
    order_m: np.ndarray         # int32 [n_orders]
    lam_min: np.ndarray         # float64 [n_orders]
    lam_max: np.ndarray
    fiber_dx: np.ndarray        # float64 [n_fibers]
    fiber_dy: np.ndarray
    deg_l: int
    deg_m: int
    coef_x: np.ndarray          # float64 [(deg_l+1)*(deg_m+1)], c[p*(deg_m+1)+q] * L^p M^q
    coef_y: np.ndarray
    lam0: float
    inv_dlam: float
    m0: float
    inv_dm: float
    blaze_lam_c: np.ndarray     # float64 [n_orders]
    blaze_amp: np.ndarray
    samples_per_px: float
    psf: Psf
    spectra: List[Spectrum]
    detector: Optional[Detector] = None
    eff_table: Optional[np.ndarray] = None
    eff_lam0: float = 0.0
    eff_dlam: float = 1.0
    notes: dict = field(default_factory=dict)

    @property
    def n_orders(self) -> int:
        return int(self.order_m.shape[0])

    @property
    def n_fibers(self) -> int:
        return int(self.fiber_dx.shape[0])

    def subset(self, orders=None, fibers=None) -> "Scene":
        """A copy restricted to some order indices / fiber indices (parity-test crops)."""
        s = copy.copy(self)
        if orders is not None:
            idx = np.asarray(orders, dtype=np.int64)
            s.order_m = np.ascontiguousarray(self.order_m[idx])
            s.lam_min = np.ascontiguousarray(self.lam_min[idx])
            s.lam_max = np.ascontiguousarray(self.lam_max[idx])
            s.blaze_lam_c = np.ascontiguousarray(self.blaze_lam_c[idx])
            s.blaze_amp = np.ascontiguousarray(self.blaze_amp[idx])
        if fibers is not None:
            idx = np.asarray(fibers, dtype=np.int64)
            s.fiber_dx = np.ascontiguousarray(self.fiber_dx[idx])
            s.fiber_dy = np.ascontiguousarray(self.fiber_dy[idx])
            s.spectra = [self.spectra[int(i)] for i in idx]
        return s


# --------------------------------------------------------------------------------------
# small polynomial helpers (input generation only: expand a closed-form spectral format
# into the monomial basis the C-ABI takes)
# --------------------------------------------------------------------------------------
def _pmul(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    out = np.zeros((a.shape[0] + b.shape[0] - 1, a.shape[1] + b.shape[1] - 1))
    for p in range(a.shape[0]):
        for q in range(a.shape[1]):
            if a[p, q] != 0.0:
                out[p:p + b.shape[0], q:q + b.shape[1]] += a[p, q] * b
    return out


def _padd(*terms) -> np.ndarray:
    sp = max(t.shape[0] for t in terms)
    sq = max(t.shape[1] for t in terms)
    out = np.zeros((sp, sq))
    for t in terms:
        out[:t.shape[0], :t.shape[1]] += t
    return out


def _const(c: float) -> np.ndarray:
    return np.array([[float(c)]])


def _pad_to(c: np.ndarray, deg_l: int, deg_m: int) -> np.ndarray:
    assert c.shape[0] <= deg_l + 1 and c.shape[1] <= deg_m + 1
    out = np.zeros((deg_l + 1, deg_m + 1))
    out[:c.shape[0], :c.shape[1]] = c
    return np.ascontiguousarray(out.reshape(-1))


def _gaussian_lines(lam_grid_0: float, dlam: float, n: int, centers, sigmas, amps,
                    nsig: float = 8.0) -> np.ndarray:
    """sum_l amps[l] * exp(-(lam-c_l)^2 / (2 s_l^2)) on a uniform grid, windowed at nsig."""
    out = np.zeros(n)
    for c, s, a in zip(centers, sigmas, amps):
        i0 = max(0, int(np.floor((c - nsig * s - lam_grid_0) / dlam)))
        i1 = min(n, int(np.ceil((c + nsig * s - lam_grid_0) / dlam)) + 1)
        if i1 <= i0:
            continue
        lam = lam_grid_0 + dlam * np.arange(i0, i1)
        out[i0:i1] += a * np.exp(-0.5 * ((lam - c) / s) ** 2)
    return out


# --------------------------------------------------------------------------------------
# configs[0]  Tiny
# --------------------------------------------------------------------------------------
def tiny(seed: int = 1001, samples_per_px: float = 40.0) -> Scene:
    """BASELINE.json configs[0]; SURVEY 8(d) 'Tiny'."""
    rng = np.random.default_rng(seed)
    nx, ny = 2048, 256
    # u = (lam-5025)/25 ; x = 1024 + 1000 u + u^2 ; y = 128 + 0.01 x
    coef_x = np.array([1024.0, 1000.0, 1.0, 0.0])
    coef_y = np.array([128.0 + 0.01 * 1024.0, 10.0, 0.01, 0.0])
    tab_lam0, tab_dlam = 4999.0, 0.001
    n_tab = int(round((5051.0 - 4999.0) / tab_dlam)) + 1
    depth = rng.uniform(0.1, 0.9, 50)
    sig = rng.uniform(0.02, 0.08, 50)
    cen = rng.uniform(5000.0, 5050.0, 50)
    flux = 1.0 - _gaussian_lines(tab_lam0, tab_dlam, n_tab, cen, sig, depth)
    flux = np.clip(flux, 0.0, None)
    return Scene(
        name="tiny", nx=nx, ny=ny,
        order_m=np.array([100], dtype=np.int32),
        lam_min=np.array([5000.0]), lam_max=np.array([5050.0]),
        fiber_dx=np.array([0.0]), fiber_dy=np.array([0.0]),
        deg_l=3, deg_m=0, coef_x=coef_x, coef_y=coef_y,
        lam0=5025.0, inv_dlam=1.0 / 25.0, m0=100.0, inv_dm=1.0,
        blaze_lam_c=np.array([5025.0]), blaze_amp=np.array([1.0]),
        samples_per_px=samples_per_px,
        psf=Psf(kind=0, fiber_dx_px=3.0, fiber_dy_px=3.0, sigma_x=1.0, sigma_y=1.0),
        spectra=[Spectrum(flux=flux, lam0=tab_lam0, dlam=tab_dlam, scale=1.0e4)],
        notes={"line_centers": cen, "line_sigmas": sig, "line_depths": depth},
    )


# --------------------------------------------------------------------------------------
# configs[1]  ESPRESSO-like,  configs[2] HIRES-like : shared echelle geometry recipe
# --------------------------------------------------------------------------------------
def _echelle_format(K: float, m_lo: int, m_hi: int, y0: float, dy1: float, dy2: float,
                    lam_mid: float, lam_half: float):
    """x = 4608 + 4500 u + 40 u^2, y = y0 + dy1 j + dy2 j^2 - 25 u^2 + 8 u with
    u = 2 (m^2 lam / K - m), j = m_hi - m, expanded in L=(lam-lam_mid)/lam_half,
    M=(m-m_mid)/m_half.  Returns (coef_x, coef_y, lam0, inv_dlam, m0, inv_dm) at tensor degree (5,5)."""
    m_mid = 0.5 * (m_lo + m_hi)
    m_half = 0.5 * (m_hi - m_lo)
    lam = np.array([[lam_mid], [lam_half]])           # lam = lam_mid + lam_half * L   (p index)
    m = np.array([[m_mid, m_half]])                   # m   = m_mid  + m_half  * M   (q index)
    m2 = _pmul(m, m)
    u = _padd((2.0 / K) * _pmul(m2, lam), -2.0 * m)
    u2 = _pmul(u, u)
    j = _padd(_const(float(m_hi)), -1.0 * m)
    x = _padd(_const(4608.0), 4500.0 * u, 40.0 * u2)
    y = _padd(_const(y0), dy1 * j, dy2 * _pmul(j, j), -25.0 * u2, 8.0 * u)
    return (_pad_to(x, 5, 5), _pad_to(y, 5, 5), lam_mid, 1.0 / lam_half, m_mid, 1.0 / m_half)


def _object_spectrum(rng, lam_lo, lam_hi, dlam, n_lines):
    n = int(round((lam_hi - lam_lo) / dlam)) + 1
    cen = rng.uniform(lam_lo, lam_hi, n_lines)
    sig = rng.uniform(0.02, 0.08, n_lines)
    dep = rng.uniform(0.0, 0.9, n_lines)
    flux = np.clip(1.0 - _gaussian_lines(lam_lo, dlam, n, cen, sig, dep), 0.0, None)
    return flux


def _fabry_perot(lam_lo, lam_hi, dlam, n_lines, lam_a, lam_b):
    """n_lines equal-area gaussian emission lines equally spaced in frequency between
    c/lam_b and c/lam_a, sigma_lam = lam / 1.5e6, unit area each."""
    n = int(round((lam_hi - lam_lo) / dlam)) + 1
    nu = np.linspace(1.0 / lam_b, 1.0 / lam_a, n_lines)
    cen = 1.0 / nu
    sig = cen / 1.5e6
    amp = 1.0 / (np.sqrt(2.0 * np.pi) * sig)
    return _gaussian_lines(lam_lo, dlam, n, cen, sig, amp)


def espresso_like(seed: int = 2002, samples_per_px: float = 32.0, n_obj_lines: int = 5000,
                  table_dlam: float = 0.001) -> Scene:
    """BASELINE.json configs[1]; SURVEY 8(d) 'ESPRESSO-like'."""
    rng = np.random.default_rng(seed)
    K = 614_640.0
    m_lo, m_hi = 78, 162
    orders = np.arange(m_lo, m_hi + 1, dtype=np.int32)
    cx, cy, lam0, inv_dlam, m0, inv_dm = _echelle_format(
        K, m_lo, m_hi, y0=150.0, dy1=92.0, dy2=0.18, lam_mid=5850.0, lam_half=2100.0)
    mf = orders.astype(np.float64)
    lam_min = K / (mf + 0.5)
    lam_max = K / (mf - 0.5)
    t_lo, t_hi = 3780.0, 7933.0
    obj = _object_spectrum(rng, t_lo, t_hi, table_dlam, n_obj_lines)
    fp = _fabry_perot(t_lo, t_hi, table_dlam, 2000, 3782.0, 7931.0)
    return Scene(
        name="espresso_like", nx=9216, ny=9216,
        order_m=orders, lam_min=lam_min, lam_max=lam_max,
        fiber_dx=np.array([0.0, 0.0]), fiber_dy=np.array([-2.5, 2.5]),
        deg_l=5, deg_m=5, coef_x=cx, coef_y=cy,
        lam0=lam0, inv_dlam=inv_dlam, m0=m0, inv_dm=inv_dm,
        blaze_lam_c=K / mf, blaze_amp=np.ones_like(mf),
        samples_per_px=samples_per_px,
        psf=Psf(kind=0, fiber_dx_px=4.0, fiber_dy_px=4.0, sigma_x=1.2, sigma_y=1.2),
        spectra=[Spectrum(flux=obj, lam0=t_lo, dlam=table_dlam, scale=1.0e4),
                 Spectrum(flux=fp, lam0=t_lo, dlam=table_dlam, scale=1.0e3)],
    )


def hires_like(seed: int = 3003, samples_per_px: float = 32.0, n_lines: int = 20000,
               table_dlam: float = 0.001) -> Scene:
    """BASELINE.json configs[2]; SURVEY 8(d) 'HIRES-like' (10-fiber pseudo-slit, Voigt lines)."""
    from scipy.special import voigt_profile
    rng = np.random.default_rng(seed)
    K = 553_000.0
    m_lo, m_hi = 79, 138
    orders = np.arange(m_lo, m_hi + 1, dtype=np.int32)
    cx, cy, lam0, inv_dlam, m0, inv_dm = _echelle_format(
        K, m_lo, m_hi, y0=200.0, dy1=148.0, dy2=0.1, lam_mid=5500.0, lam_half=1500.0)
    mf = orders.astype(np.float64)
    lam_min = K / (mf + 0.5)
    lam_max = K / (mf - 0.5)
    t_lo, t_hi = 3990.0, 7040.0
    n = int(round((t_hi - t_lo) / table_dlam)) + 1
    cen = rng.uniform(4000.0, 7000.0, n_lines)
    sig = rng.uniform(0.02, 0.08, n_lines)
    gam = rng.uniform(0.005, 0.02, n_lines)
    dep = rng.uniform(0.0, 0.9, n_lines)
    flux = np.ones(n)
    half = int(round(5.0 / table_dlam))
    for c, s, g, d in zip(cen, sig, gam, dep):
        ic = int(round((c - t_lo) / table_dlam))
        i0, i1 = max(0, ic - half), min(n, ic + half + 1)
        lam = t_lo + table_dlam * np.arange(i0, i1)
        flux[i0:i1] *= 1.0 - d * voigt_profile(lam - c, s, g) / voigt_profile(0.0, s, g)
    n_f = 10
    f = np.arange(n_f, dtype=np.float64)
    dy = 6.0 * (f - 4.5)
    scale = 1.0e4 * np.exp(-0.5 * ((f - 4.5) / 3.0) ** 2)      # centre fibers brighter
    return Scene(
        name="hires_like", nx=9216, ny=9216,
        order_m=orders, lam_min=lam_min, lam_max=lam_max,
        fiber_dx=np.zeros(n_f), fiber_dy=dy,
        deg_l=5, deg_m=5, coef_x=cx, coef_y=cy,
        lam0=lam0, inv_dlam=inv_dlam, m0=m0, inv_dm=inv_dm,
        blaze_lam_c=K / mf, blaze_amp=np.ones_like(mf),
        samples_per_px=samples_per_px,
        psf=Psf(kind=0, fiber_dx_px=4.0, fiber_dy_px=4.0, sigma_x=1.2, sigma_y=1.2),
        spectra=[Spectrum(flux=flux, lam0=t_lo, dlam=table_dlam, scale=float(sc)) for sc in scale],
    )


# --------------------------------------------------------------------------------------
# configs[3]  field-dependent tabulated PSF
# --------------------------------------------------------------------------------------
def tabulated_kernels(seed: int = 4004, npix: int = 11, os: int = 8, gx: int = 5, gy: int = 5) -> np.ndarray:
    """gy*gx kernels of (npix*os)^2 cell values: elliptical gaussian (sigma U[1.0,1.6], axis ratio
    >= 0.8, random orientation) x smooth low-order perturbation (<= 5 %) x cosine taper to 0 at
    r = npix/2, integrated over the 1/os-px cells (4x4 midpoint sub-samples), normalised to sum 1."""
    rng = np.random.default_rng(seed)
    n = npix * os
    sub = 4
    h = 1.0 / (os * sub)
    g = -0.5 * npix + h * (np.arange(n * sub) + 0.5)
    X, Y = np.meshgrid(g, g)
    R = np.hypot(X, Y)
    taper = np.where(R < 0.5 * npix, 0.5 * (1.0 + np.cos(np.pi * R / (0.5 * npix))), 0.0)
    out = np.zeros((gy, gx, n, n))
    for b in range(gy):
        for a in range(gx):
            s1 = rng.uniform(1.0, 1.6)
            ratio = rng.uniform(0.8, 1.0)
            s2 = s1 * ratio
            th = rng.uniform(0.0, np.pi)
            c, s = np.cos(th), np.sin(th)
            U = c * X + s * Y
            V = -s * X + c * Y
            dens = np.exp(-0.5 * ((U / s1) ** 2 + (V / s2) ** 2))
            p = rng.uniform(-0.05, 0.05, 3)
            dens = dens * (1.0 + p[0] * X / npix + p[1] * Y / npix + p[2] * (X * Y) / (npix * npix))
            dens = dens * taper
            cells = dens.reshape(n, sub, n, sub).sum(axis=(1, 3))
            out[b, a] = cells / cells.sum()
    return np.ascontiguousarray(out)


def field_psf(seed: int = 4004, samples_per_px: float = 32.0, base: Optional[Scene] = None) -> Scene:
    """BASELINE.json configs[3]: ESPRESSO-like geometry + 5x5 grid of 11x11-px, 8x kernels."""
    s = copy.copy(base) if base is not None else espresso_like(samples_per_px=samples_per_px)
    s.name = "field_psf"
    s.psf = Psf(kind=1, tab_npix=11, tab_os=8, tab_gx=5, tab_gy=5, tab=tabulated_kernels(seed))
    return s


# --------------------------------------------------------------------------------------
# configs[4]  precision / RV sweep
# --------------------------------------------------------------------------------------
def psf_map(base: Scene, gx: int = 3, gy: int = 3, seed: int = 6006, growth: float = 0.25, jitter: float = 0.03) -> Scene:
    """Analytic PSF map (G21; "evaluate the optical PSF ... for each wavelength"): the base scene with
    sigma_x, sigma_y given at the nodes of a gx x gy grid over the detector.  Input recipe only: the image quality of a camera
    degrades towards the corners of the field, so sigma grows with the squared normalised distance from the detector centre
    (by `growth` at the corners, differently in x and y) with a few per cent of node-to-node scatter."""
    rng = np.random.default_rng(seed)
    s = copy.copy(base)
    s.name = base.name + "_psf_map"
    gxs = np.linspace(-1.0, 1.0, gx) if gx > 1 else np.zeros(1)
    gys = np.linspace(-1.0, 1.0, gy) if gy > 1 else np.zeros(1)
    X, Y = np.meshgrid(gxs, gys)                                    # [gy][gx]
    r2 = 0.5 * (X * X + Y * Y)
    p = copy.copy(base.psf)
    p.an_gx, p.an_gy = gx, gy
    p.an_sigma_x = base.psf.sigma_x * (1.0 + growth * (r2 + 0.2 * X)) * (1.0 + jitter * rng.uniform(-1.0, 1.0, (gy, gx)))
    p.an_sigma_y = base.psf.sigma_y * (1.0 + 0.6 * growth * (r2 - 0.25 * Y)) * (1.0 + jitter * rng.uniform(-1.0, 1.0, (gy, gx)))
    s.psf = p
    return s


RV_SWEEP_V = (0.0, 0.01, 0.1, 1.0, 10.0)   # m/s


def rv_sweep(v_mps: float = 0.0, seed: int = 5005, samples_per_px: float = 256.0) -> Scene:
    """BASELINE.json configs[4]: Tiny geometry/PSF, 200 isolated gaussian emission lines,
    Doppler factor 1+v/c; peak scaled to ~4e4 e-/px; detector ron = 3 e-."""
    s = tiny(samples_per_px=samples_per_px)
    s.name = "rv_sweep"
    tab_lam0, tab_dlam = 4999.0, 0.0005
    n_tab = int(round((5051.0 - 4999.0) / tab_dlam)) + 1
    cen = 5000.0 + (np.arange(200) + 0.5) * 0.25
    sig = np.full(200, 0.01)
    flux = _gaussian_lines(tab_lam0, tab_dlam, n_tab, cen, sig, np.ones(200))
    # a line of unit peak and sigma 0.01 A holds sqrt(2 pi) 0.01 A of flux * blaze ~0.4-1; spread by the
    # PSF over ~ (3 px core)^2: scale so the brightest pixel is ~4e4 e-
    s.spectra = [Spectrum(flux=flux, lam0=tab_lam0, dlam=tab_dlam, scale=1.8e7,
                          doppler=1.0 + v_mps / C_LIGHT)]
    s.detector = Detector(gain=1.0, dark_e=0.0, ron_e=3.0, bias=0.0, seed=seed)
    s.notes = {"line_centers": cen, "v_mps": v_mps}
    return s


# --------------------------------------------------------------------------------------
# small special-purpose scenes used by pins / parity edge cases
# --------------------------------------------------------------------------------------
def single_line_scene(x_pos: float = 100.3173, y_pos: float = 37.8641, nx: int = 200, ny: int = 80,
                      fiber_d: float = 3.0, sigma: float = 1.0, samples: int = 1,
                      support_nsigma: float = 7.5) -> Scene:
    """One order whose `samples` wavelength samples all map to x in a tiny range around x_pos
    (samples=1: exactly one sample at x_pos); flat spectrum, flat blaze (amp 1, m=0 -> sinc(0)=1)."""
    # x = x_pos + (samples-1)/spp... we use lam in [0,1], x = x_pos + width*(L-0.5), L = lam
    spp = 1.0
    width = float(samples) if samples > 1 else 0.5
    # N = ceil(spp*|x(lmax)-x(lmin)|) = ceil(width): samples=1 -> width 0.5 -> N=1 at L=0.5 -> x = x_pos
    coef_x = np.array([x_pos - 0.5 * width, width])
    coef_y = np.array([y_pos, 0.0])
    return Scene(
        name="single_line", nx=nx, ny=ny,
        order_m=np.array([0], dtype=np.int32),
        lam_min=np.array([0.0]), lam_max=np.array([1.0]),
        fiber_dx=np.array([0.0]), fiber_dy=np.array([0.0]),
        deg_l=1, deg_m=0, coef_x=coef_x, coef_y=coef_y,
        lam0=0.0, inv_dlam=1.0, m0=0.0, inv_dm=1.0,
        blaze_lam_c=np.array([1.0]), blaze_amp=np.array([1.0]),
        samples_per_px=spp,
        psf=Psf(kind=0, fiber_dx_px=fiber_d, fiber_dy_px=fiber_d, sigma_x=sigma, sigma_y=sigma,
                support_nsigma=support_nsigma),
        spectra=[Spectrum(flux=np.ones(8), lam0=-1.0, dlam=0.5, scale=1.0)],
    )
