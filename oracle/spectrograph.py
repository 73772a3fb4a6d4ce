"""CPU oracle of the parametric Spectrograph Unit (G22).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  The closed-form relations of a cross-dispersed echelle spectrograph,
written out in plain numpy float64 -- no polynomial fit, no tables: this is what the format polynomials produced by the
library's ``e2e_spectrograph_format`` have to reproduce.  Shares no code with paper_2008_05858_b200/csrc/spectrograph.cu.

  echelle          m lam = d cos(gamma) (sin alpha + sin beta),   alpha = blaze + theta;  blaze peak at beta_c = blaze - theta
  camera           x = x_c + F tan(beta - beta_c),   F = f_cam / pixel
  cross-disperser  sin beta_x = lam / d_x - sin alpha_x,  sin alpha_x = lam_ref / (2 d_x);   y = y_c + F tan(beta_x - alpha_x)

Pins (tests/test_oracle_spectrograph.py): Littrow blaze relation m lam_c = 2 d sin(blaze); angular dispersion
d beta / d lam = m / (d cos gamma cos beta); free spectral range K / (m^2 - 1/4); every blaze peak lands on x_c; lam_ref lands
on y_c; dy / dlam = F / (d_x cos beta_x); Littrow line tilt tan chi = 2 tan(blaze) tan(gamma).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Sequence

import numpy as np


@dataclass
class Spectrograph:
    groove_um: float
    blaze_deg: float
    theta_deg: float
    gamma_deg: float
    xd_groove_um: float
    xd_lam_ref: float
    f_cam_mm: float
    f_coll_mm: float
    pixel_um: float
    fiber_core_um: float
    m_lo: int
    m_hi: int
    x_c: float
    y_c: float
    fiber_height_um: Sequence[float] = (0.0,)


def _angles(p: Spectrograph):
    tb, th, g = np.deg2rad(p.blaze_deg), np.deg2rad(p.theta_deg), np.deg2rad(p.gamma_deg)
    return tb + th, tb - th, g


def blaze_constant(p: Spectrograph) -> float:
    """K = m lam at the blaze peak (Angstrom)"""
    alpha, beta_c, g = _angles(p)
    return p.groove_um * 1e4 * np.cos(g) * (np.sin(alpha) + np.sin(beta_c))


def beta(p: Spectrograph, lam, m):
    """diffraction angle of wavelength lam (Angstrom) in order m, from the grating equation"""
    alpha, _, g = _angles(p)
    return np.arcsin(np.asarray(m, dtype=float) * np.asarray(lam, dtype=float) / (p.groove_um * 1e4 * np.cos(g)) - np.sin(alpha))


def px_per_radian(p: Spectrograph) -> float:
    return p.f_cam_mm * 1e3 / p.pixel_um


def position_x(p: Spectrograph, lam, m):
    _, beta_c, _ = _angles(p)
    return p.x_c + px_per_radian(p) * np.tan(beta(p, lam, m) - beta_c)


def beta_x(p: Spectrograph, lam):
    dx = p.xd_groove_um * 1e4
    return np.arcsin(np.asarray(lam, dtype=float) / dx - p.xd_lam_ref / (2.0 * dx))


def position_y(p: Spectrograph, lam):
    alpha_x = np.arcsin(p.xd_lam_ref / (2.0 * p.xd_groove_um * 1e4))
    return p.y_c + px_per_radian(p) * np.tan(beta_x(p, lam) - alpha_x)


def order_table(p: Spectrograph):
    """(m, lam_c, lam_min, lam_max) per order: blaze wavelength and one free spectral range around it"""
    m = np.arange(p.m_lo, p.m_hi + 1)
    K = blaze_constant(p)
    return m, K / m, K / (m + 0.5), K / (m - 0.5)


def blaze_peak_amplitude(p: Spectrograph) -> float:
    alpha, beta_c, _ = _angles(p)
    return min(1.0, np.cos(alpha) / np.cos(beta_c))


def fiber_images(p: Spectrograph):
    """(Dx, Dy, dx_f, dy_f, tan chi): full widths of the fiber image in pixels, per-fiber offsets, line tilt"""
    alpha, beta_c, g = _angles(p)
    mag = p.f_cam_mm / p.f_coll_mm / p.pixel_um
    Dy = p.fiber_core_um * mag
    Dx = Dy * np.cos(alpha) / np.cos(beta_c)
    tan_chi = np.tan(g) * (np.sin(alpha) + np.sin(beta_c)) / np.cos(beta_c)
    dy = np.asarray(p.fiber_height_um, dtype=float) * mag
    return Dx, Dy, tan_chi * dy, dy, tan_chi
