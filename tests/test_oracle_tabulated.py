"""Pins for the oracle's tabulated, field-dependent PSF (pin P10)."""
import numpy as np
import pytest
from scipy import special

import oracle
from paper_2008_05858_b200 import workloads as W


def tab_scene(tab, npix, os_, nx=200, ny=120, x_pos=60.3, y_pos=40.7):
    s = W.single_line_scene(x_pos=x_pos, y_pos=y_pos, nx=nx, ny=ny)
    gy, gx = tab.shape[:2]
    s.psf = W.Psf(kind=1, tab_npix=npix, tab_os=os_, tab_gx=gx, tab_gy=gy, tab=np.ascontiguousarray(tab))
    return s


def gaussian_cells(npix, os_, sx, sy):
    """exact cell integrals of a gaussian density over the 1/os-px cells (erf differences)"""
    e = -0.5 * npix + np.arange(npix * os_ + 1) / os_
    cx = np.diff(special.ndtr(e / sx)); cy = np.diff(special.ndtr(e / sy))
    return np.outer(cy, cx)


def test_t2_summed_area_table_form_equals_cell_overlap_sum():
    """P10a: the pixel integral of a piecewise-constant density == 4-corner difference of bilinear lookups in
    the summed-area table of the cells (computed here in numpy), for a random kernel"""
    rng = np.random.default_rng(3)
    npix, os_ = 11, 8
    n = npix * os_
    T = rng.uniform(0, 1, (n, n)); T /= T.sum()
    s = tab_scene(T[None, None], npix, os_)
    Csat = np.zeros((n + 1, n + 1)); Csat[1:, 1:] = np.cumsum(np.cumsum(T, axis=0), axis=1)

    def lookup(u, v):                       # bilinear in the SAT, kernel coords in px, clamped to the support
        a = np.clip((u + 0.5 * npix) * os_, 0, n); b = np.clip((v + 0.5 * npix) * os_, 0, n)
        a0 = min(int(np.floor(a)), n - 1); b0 = min(int(np.floor(b)), n - 1)
        fa, fb = a - a0, b - b0
        return ((1 - fb) * ((1 - fa) * Csat[b0, a0] + fa * Csat[b0, a0 + 1]) + fb * ((1 - fa) * Csat[b0 + 1, a0] + fa * Csat[b0 + 1, a0 + 1]))

    xk, yk = 60.3, 40.7
    tot = 0.0
    for i in range(54, 68):
        for j in range(34, 48):
            u, v = i - xk, j - yk
            sat = lookup(u + .5, v + .5) - lookup(u - .5, v + .5) - lookup(u + .5, v - .5) + lookup(u - .5, v - .5)
            got = oracle.psf_tab_pixel(s, xk, yk, i, j)
            assert got == pytest.approx(sat, rel=1e-12, abs=2e-16)
            tot += got
    assert tot == pytest.approx(1.0, abs=1e-14)            # P3 for the tabulated path: kernel sums to 1


def test_t1_converges_to_analytic_gaussian_as_cells_shrink():
    """P10b: cells built from an analytic gaussian reproduce the analytic pixel integrals with O(h^2) error"""
    sx, sy, npix = 0.55, 0.62, 11
    xk, yk = 60.3, 40.7
    pix = [(60, 41), (61, 40), (59, 42), (62, 41)]
    ana = W.Psf(fiber_dx_px=0, fiber_dy_px=0, sigma_x=sx, sigma_y=sy)
    errs = []
    for os_ in (4, 8, 16):
        s = tab_scene(gaussian_cells(npix, os_, sx, sy)[None, None], npix, os_)
        e = max(abs(oracle.psf_tab_pixel(s, xk, yk, i, j) - oracle.psf_pixel(ana, i - xk, j - yk)) for i, j in pix)
        errs.append(e)
    assert errs[0] < 5e-3 and errs[2] < errs[0] / 10
    # second order in the cell size h = 1/os; the constant depends on where the pixel edge falls inside a cell
    for os_, e in zip((4, 8, 16), errs):
        assert 0.03 < e * os_ ** 2 < 0.3


def test_t3_field_blend_is_bilinear_in_detector_position():
    tabs = W.tabulated_kernels(seed=11, npix=11, os=8, gx=3, gy=2)
    nx, ny = 201, 101                                        # nodes at x = 0, 100, 200 ; y = 0, 100
    one = lambda g, h: tab_scene(tabs[h:h + 1, g:g + 1], 11, 8, nx=nx, ny=ny)
    full = tab_scene(tabs, 11, 8, nx=nx, ny=ny)
    # at a node: that node's kernel
    assert oracle.psf_tab_pixel(full, 100.0, 0.0, 101, 1) == pytest.approx(oracle.psf_tab_pixel(one(1, 0), 100.0, 0.0, 101, 1), rel=1e-14)
    # in between: bilinear weights (x = 125 -> 0.75/0.25 between g=1,2 ; y = 40 -> 0.6/0.4 between h=0,1)
    xk, yk, i, j = 125.0, 40.0, 126, 39
    ref = 0.6 * (0.75 * oracle.psf_tab_pixel(one(1, 0), xk, yk, i, j) + 0.25 * oracle.psf_tab_pixel(one(2, 0), xk, yk, i, j)) \
        + 0.4 * (0.75 * oracle.psf_tab_pixel(one(1, 1), xk, yk, i, j) + 0.25 * oracle.psf_tab_pixel(one(2, 1), xk, yk, i, j))
    assert oracle.psf_tab_pixel(full, xk, yk, i, j) == pytest.approx(ref, rel=1e-14)
    # clamped outside the grid
    assert oracle.psf_tab_pixel(full, -7.0, 40.0, -6, 39) == pytest.approx(
        0.6 * oracle.psf_tab_pixel(one(0, 0), -7.0, 40.0, -6, 39) + 0.4 * oracle.psf_tab_pixel(one(0, 1), -7.0, 40.0, -6, 39), rel=1e-14)


def test_tabulated_render_footprint_and_flux():
    tabs = W.tabulated_kernels(seed=5, npix=11, os=8, gx=2, gy=2)
    s = tab_scene(tabs, 11, 8, x_pos=60.3, y_pos=40.7)
    fr = oracle.render(s)
    nz = np.nonzero(fr)
    assert (nz[1].min(), nz[1].max(), nz[0].min(), nz[0].max()) == (55, 66, 35, 46)     # 12 x 12 pixels
    assert fr.sum() == pytest.approx(1.0, abs=1e-14)
    assert oracle.footprint(s, 60.5, 40.0) == (55, 66, 34, 46)                          # degenerate phases: up to 13
    for k in tabs.reshape(-1, 88, 88):
        assert k.sum() == pytest.approx(1.0, abs=1e-14) and k.min() >= 0.0
