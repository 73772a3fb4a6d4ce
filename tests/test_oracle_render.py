"""Pins for the oracle's sample setup and frame accumulation (steps a1-a3, a5; SURVEY 8(c) O1-O3, O6,
pins P3 P5 P7 P8 P9, G9, G11, blaze / interpolation closed forms).  Small scenes only (CPU suite budget)."""
import copy

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2008_05858_b200 import workloads as W


def small_tiny(spp=1.0, lam=(5010.0, 5013.0)):
    s = W.tiny(samples_per_px=spp)
    s.lam_min = np.array([lam[0]])
    s.lam_max = np.array([lam[1]])
    return s


# ---------------------------------------------------------------- a1: sample grid
def test_a1_sample_count_and_midpoint_grid():
    s = W.tiny()
    assert oracle.order_nsamples(s, 0) == 80000          # ceil(40 * |x(5050) - x(5000)|) = 40 * 2000
    lam, x, y, w = oracle.samples(s, 0, 0, 0, 5)
    dl = 50.0 / 80000
    assert np.allclose(lam, 5000.0 + (np.arange(5) + 0.5) * dl, rtol=0, atol=1e-12)
    lam, x, y, w = oracle.samples(s, 0, 0, 79999, 80000)
    assert lam[0] == pytest.approx(5050.0 - 0.5 * dl, abs=1e-11)


# ---------------------------------------------------------------- a3: positions
def test_a3_positions_closed_form_tiny():
    """Tiny recipe: x = 1024 + 1000 u + u^2, y = 128 + 0.01 x, u = (lam - 5025)/25"""
    s = W.tiny()
    lam, x, y, w = oracle.samples(s, 0, 0, 1234, 1300)
    u = (lam - 5025.0) / 25.0
    assert np.allclose(x, 1024 + 1000 * u + u * u, rtol=0, atol=2e-12)
    assert np.allclose(y, 128 + 0.01 * (1024 + 1000 * u + u * u), rtol=0, atol=2e-13)


def test_a3_positions_vs_mpmath_and_recipe_espresso():
    """O2/G8: the (5,5) monomial expansion evaluated by fma-Horner reproduces the closed-form echelle recipe
    x = 4608 + 4500 u + 40 u^2, y = 150 + 92 j + 0.18 j^2 - 25 u^2 + 8 u (u = 2(m^2 lam/K - m), j = 162 - m)
    to the fp64 evaluation noise of G8 (<= 2e-9 px), and a 40-digit evaluation of the same coefficients closer still."""
    s = W.espresso_like(n_obj_lines=10, table_dlam=0.05)
    K = 614640.0
    for o in (0, 41, 84):
        n = oracle.order_nsamples(s, o)
        assert abs(n - 32 * 9016) < 32 * 40               # x spans ~[162, 9178]
        for fiber in (0, 1):
            lam, x, y, w = oracle.samples(s, fiber, o, n // 3, n // 3 + 4)
            m = float(s.order_m[o])
            u = 2 * (m * m * lam / K - m)
            j = 162 - m
            assert np.allclose(x, 4608 + 4500 * u + 40 * u * u + s.fiber_dx[fiber], rtol=0, atol=2e-9)
            assert np.allclose(y, 150 + 92 * j + 0.18 * j * j - 25 * u * u + 8 * u + s.fiber_dy[fiber], rtol=0, atol=2e-9)
            # the same double coefficients in 40-digit arithmetic: |x_fp64 - x_exact| is pure evaluation noise
            mp.mp.dps = 40
            L = (mp.mpf(float(lam[0])) - mp.mpf(s.lam0)) * mp.mpf(s.inv_dlam)
            M = (mp.mpf(m) - mp.mpf(s.m0)) * mp.mpf(s.inv_dm)
            xe = sum(mp.mpf(float(s.coef_x[p * 6 + q])) * L ** p * M ** q for p in range(6) for q in range(6))
            assert abs(float(xe + mp.mpf(float(s.fiber_dx[fiber])) - mp.mpf(float(x[0])))) < 2e-9


def test_format_is_monotone_and_orders_separated():
    s = W.espresso_like(n_obj_lines=10, table_dlam=0.05)
    ys = []
    for o in range(0, 85, 12):
        n = oracle.order_nsamples(s, o)
        xs = np.concatenate([oracle.samples(s, 0, o, k, k + 2)[1] for k in range(0, n - 2, n // 50)])
        assert np.all(np.diff(xs) > 0)
        assert xs.min() > 150 and xs.max() < 9216 - 30
        ys.append(oracle.samples(s, 0, o, n // 2, n // 2 + 1)[2][0])
    assert np.all(np.abs(np.diff(ys)) >= 12 * 40)          # inter-order spacing >= 40 px (BASELINE.json configs[1])


# ---------------------------------------------------------------- a2: flux
def test_a2_blaze_closed_forms():
    """E(lam_c) = A; at the free-spectral-range edges lam = lam_c m/(m -+ 1/2): E = A (2/pi)^2 = 0.405285 A"""
    s = W.single_line_scene()
    s.order_m = np.array([100], dtype=np.int32)
    s.blaze_lam_c = np.array([5025.0]); s.blaze_amp = np.array([1.7])
    s.spectra = [W.Spectrum(flux=np.ones(4), lam0=0.0, dlam=4000.0, scale=1.0)]
    for lam_t, expect in [(5025.0, 1.7), (5025.0 * 100 / 99.5, 1.7 * (2 / np.pi) ** 2), (5025.0 * 100 / 100.5, 1.7 * (2 / np.pi) ** 2),
                          (5025.0 * 100 / 99.0, 0.0)]:
        s.lam_min = np.array([lam_t - 0.5]); s.lam_max = np.array([lam_t + 0.5])   # one sample at the midpoint lam_t
        s.lam0 = lam_t - 0.5
        lam, x, y, w = oracle.samples(s, 0, 0)
        assert len(w) == 1 and lam[0] == pytest.approx(lam_t, abs=1e-12)
        assert w[0] == pytest.approx(expect, rel=1e-12, abs=1e-28)                 # dlam = 1, S = 1, scale = 1


def test_a2_linear_interpolation_and_doppler_and_photons_per_bin():
    s = small_tiny(spp=3.0)
    n = oracle.order_nsamples(s, 0)
    lam_tab0, dl_tab = 5000.0, 0.37
    tab = 2.0 + 0.5 * (lam_tab0 + dl_tab * np.arange(60) - 5000.0)      # S(lam) = 2 + 0.5 (lam - 5000): linear -> interpolation exact
    s.spectra = [W.Spectrum(flux=tab, lam0=lam_tab0, dlam=dl_tab, scale=3.0, doppler=1.0)]
    s.blaze_lam_c = np.array([1.0]); s.order_m = np.array([0], dtype=np.int32)     # m = 0 -> sinc(0) = 1
    s.m0 = 0.0
    lam, x, y, w = oracle.samples(s, 0, 0)
    dlam = 3.0 / n
    assert np.allclose(w, 3.0 * (2.0 + 0.5 * (lam - 5000.0)) * dlam, rtol=1e-13)
    d = 1.0 + 3.0e-5
    s.spectra[0].doppler = d
    lam, x, y, w2 = oracle.samples(s, 0, 0)
    assert np.allclose(w2, 3.0 * (2.0 + 0.5 * (lam / d - 5000.0)) * dlam, rtol=1e-13)    # G13: S'(lam) = S(lam/(1+v/c))
    # outside the table -> 0
    s.spectra = [W.Spectrum(flux=np.ones(5), lam0=5011.0, dlam=0.25, scale=1.0)]
    lam, x, y, w3 = oracle.samples(s, 0, 0)
    inside = (lam >= 5011.0) & (lam < 5012.0)
    assert np.all(w3[~inside] == 0.0) and np.all(w3[inside] > 0.0)


def test_a2_efficiency_table():
    s = small_tiny(spp=2.0)
    lam, x, y, w0 = oracle.samples(s, 0, 0)
    s.eff_table = np.array([0.5, 0.5, 0.9]); s.eff_lam0 = 5000.0; s.eff_dlam = 10.0
    lam, x, y, w1 = oracle.samples(s, 0, 0)
    T = np.where(lam < 5010, 0.5, 0.5 + 0.4 * (lam - 5010.0) / 10.0)
    assert np.allclose(w1, w0 * T, rtol=1e-13)


# ---------------------------------------------------------------- a5 / P3: flux conservation
def test_p3_frame_flux_conservation():
    """frame sum == injected photons to 1e-12 relative (BASELINE.json north_star)"""
    s = small_tiny(spp=4.0)
    fr = oracle.render(s)
    tot = oracle.total_weight(s)
    lam, x, y, w = oracle.samples(s, 0, 0)
    assert tot == pytest.approx(float(np.sum(w)), rel=1e-14)
    assert float(np.sum(fr)) == pytest.approx(tot, rel=1e-12)
    assert abs(float(np.sum(fr)) / tot - 1.0) < 2e-13       # the G9 tail, <= 1.3e-13 per axis pair


# ---------------------------------------------------------------- P5: photocenter of a rendered line
def test_p5_isolated_line_photocenter():
    """photocenter of a rendered isolated line == flux-weighted mean of the mapped sample positions (1e-7 px;
    paper requires < 1e-5 px), in x and in y"""
    s = small_tiny(spp=40.0, lam=(5011.0, 5012.5))
    tab0, dtab = 5010.0, 0.001
    lamt = tab0 + dtab * np.arange(4000)
    s.spectra = [W.Spectrum(flux=np.exp(-0.5 * ((lamt - 5011.7) / 0.05) ** 2), lam0=tab0, dlam=dtab, scale=1e4)]
    fr = oracle.render(s, window=(400, 100, 120, 80))
    lam, x, y, w = oracle.samples(s, 0, 0)
    ii = 400 + np.arange(120); jj = 100 + np.arange(80)
    cx = float(np.sum(fr * ii[None, :]) / np.sum(fr)); cy = float(np.sum(fr * jj[:, None]) / np.sum(fr))
    assert abs(cx - float(np.sum(w * x) / np.sum(w))) < 1e-7
    assert abs(cy - float(np.sum(w * y) / np.sum(w))) < 1e-7
    # delta-like line (one sample): photocenter == polynomial-mapped position itself
    d = W.single_line_scene(x_pos=100.3173, y_pos=37.8641)
    fr = oracle.render(d)
    cx = float(np.sum(fr * np.arange(d.nx)[None, :]) / np.sum(fr)); cy = float(np.sum(fr * np.arange(d.ny)[:, None]) / np.sum(fr))
    assert abs(cx - 100.3173) < 1e-9 and abs(cy - 37.8641) < 1e-9


# ---------------------------------------------------------------- G9 / G11 footprint and detector edge
def test_g9_footprint_box_is_part_of_the_definition():
    d = W.single_line_scene(x_pos=100.3173, y_pos=37.8641)             # R = 1.5, sigma = 1, t = 7.5 -> H = 9
    fr = oracle.render(d)
    nz = np.nonzero(fr)
    assert nz[1].min() == int(np.ceil(100.3173 - 9.5)) and nz[1].max() == int(np.floor(100.3173 + 9.5))
    assert nz[0].min() == int(np.ceil(37.8641 - 9.5)) and nz[0].max() == int(np.floor(37.8641 + 9.5))
    assert oracle.footprint(d, 100.3173, 37.8641) == (91, 109, 29, 47)
    assert oracle.footprint(d, 100.5, 37.0) == (91, 110, 28, 46)        # half-integer: 20 columns
    # values inside are the PSF itself
    assert fr[38, 100] == pytest.approx(oracle.psf_pixel(d.psf, 100 - 100.3173, 38 - 37.8641), rel=1e-15)


def test_g11_detector_edge_drops_flux():
    big = W.single_line_scene(x_pos=104.25, y_pos=43.75, nx=200, ny=80)
    fr_big = oracle.render(big)
    # same sample, but on a detector whose origin is shifted by (100, 40): the sample sits 4.25 / 3.75 px (binary-exact, so both renders see the same sub-pixel phase) from the corner
    small = W.single_line_scene(x_pos=4.25, y_pos=3.75, nx=60, ny=40)
    fr_small = oracle.render(small)
    assert np.allclose(fr_small[:30, :50], fr_big[40:70, 100:150], rtol=1e-13, atol=1e-30)
    assert fr_small.sum() < 0.9999 * fr_big.sum()            # flux beyond the edge is lost, not wrapped
    # completely off-detector sample contributes nothing
    off = W.single_line_scene(x_pos=-30.0, y_pos=3.7, nx=60, ny=40)
    assert oracle.render(off).sum() == 0.0


def test_window_render_is_a_crop():
    s = small_tiny(spp=2.0)
    full = oracle.render(s)
    lam, x, y, w = oracle.samples(s, 0, 0)
    i0 = int(x.mean()) - 10; j0 = int(y.mean()) - 6
    win = oracle.render(s, window=(i0, j0, 33, 17))
    assert np.array_equal(win, full[j0:j0 + 17, i0:i0 + 33])
    assert np.count_nonzero(win) > 100


# ---------------------------------------------------------------- P7 symmetries
def test_p7_trace_symmetry_and_reflection():
    d = W.single_line_scene(x_pos=100.3, y_pos=40.0, samples=6)          # flat trace at integer y, symmetric PSF
    fr = oracle.render(d)
    peak = fr.max()
    for dlt in range(1, 10):
        assert np.max(np.abs(fr[40 + dlt] - fr[40 - dlt])) < 1e-15 * peak
    d2 = W.single_line_scene(x_pos=100.3, y_pos=39.5, samples=6)         # half-integer y: symmetric about 39.5
    fr2 = oracle.render(d2)
    for dlt in range(0, 9):
        assert np.max(np.abs(fr2[40 + dlt] - fr2[39 - dlt])) < 1e-15 * fr2.max()
    # reflecting Y -> (ny-1) - Y flips the frame vertically
    r = copy.copy(d); r.coef_y = np.array([(d.ny - 1) - 37.2, 0.0]); d3 = copy.copy(d); d3.coef_y = np.array([37.2, 0.0])
    a, b = oracle.render(d3), oracle.render(r)
    assert np.allclose(b[::-1], a, rtol=1e-10, atol=1e-14 * a.max())
    # reflecting X
    rx = copy.copy(d3); rx.coef_x = (d.nx - 1) - d3.coef_x[0] - np.array([0.0, 0.0]); rx.coef_x = np.array([(d.nx - 1) - d3.coef_x[0], -d3.coef_x[1]])
    c = oracle.render(rx)
    assert np.allclose(c[:, ::-1], a, rtol=1e-10, atol=1e-14 * a.max())


# ---------------------------------------------------------------- P8 linearity / superposition
def test_p8_linearity_and_fiber_superposition():
    s = small_tiny(spp=1.0)
    s.fiber_dx = np.array([0.0, 0.3]); s.fiber_dy = np.array([-2.5, 2.5])
    rng = np.random.default_rng(7)
    t1 = rng.uniform(0.2, 1.0, 300); t2 = rng.uniform(0.2, 1.0, 300)
    mk = lambda t, sc: W.Spectrum(flux=t, lam0=5009.0, dlam=0.02, scale=sc)
    win = (380, 100, 180, 80)
    s.spectra = [mk(t1, 1.0), mk(t2, 0.0)]
    A = oracle.render(s, window=win)                       # fiber 0 alone
    s.spectra = [mk(t1, 0.0), mk(t2, 1.0)]
    B = oracle.render(s, window=win)                       # fiber 1 alone
    s.spectra = [mk(t1, 1.0), mk(t2, 1.0)]
    AB = oracle.render(s, window=win)
    assert np.allclose(AB, A + B, rtol=1e-14, atol=1e-16 * AB.max())
    s.spectra = [mk(2.0 * t1 + 3.0 * t2, 1.0), mk(t2, 0.0)]
    lin = oracle.render(s, window=win)
    s.spectra = [mk(t2, 1.0), mk(t2, 0.0)]
    A2 = oracle.render(s, window=win)
    assert np.allclose(lin, 2.0 * A + 3.0 * A2, rtol=1e-13, atol=1e-16 * lin.max())
    assert A.max() > 0 and B.max() > 0 and not np.allclose(A, B)


# ---------------------------------------------------------------- P9 integer translation
def test_p9_integer_translation():
    s = small_tiny(spp=1.0)
    a = oracle.render(s, window=(380, 100, 180, 80))
    t = copy.copy(s); t.coef_x = s.coef_x.copy(); t.coef_y = s.coef_y.copy()
    t.coef_x[0] += 7.0; t.coef_y[0] -= 3.0
    b = oracle.render(t, window=(387, 97, 180, 80))
    assert np.allclose(a, b, rtol=1e-10, atol=1e-14 * a.max())
    assert a.max() > 0


# ---------------------------------------------------------------- G14: RV sweep ("cm/s")
def _rv_crop(v):
    s = W.rv_sweep(v)
    s.lam_min = np.array([5010.0]); s.lam_max = np.array([5014.0])       # 16 of the 200 lines, 256 samples/px
    return s


def test_g14_rv_sweep_photocenter_linear_in_velocity():
    """BASELINE.json configs[4] on a crop of the RV-sweep scene, oracle only.  DESIGN.md G14 (re-read in round 2):
    (i) P5 at every velocity: the frame's global photocenter is the flux-weighted mean of the mapped samples (1e-9 px);
    (ii) it moves linearly with v: residual against a least-squares line through the 5 velocities < 1e-6 px, globally and per
    line (Voronoi windows of integer columns between line positions);
    (iii) the slope is the closed form of the line list: with W_l = E(lam_l), X_l = X(lam_l), xbar = sum W X / sum W,
          d xbar / d beta = [ sum_l W_l lam_l X'(lam_l)  +  sum_l E'(lam_l) lam_l (X_l - xbar) ] / sum_l W_l ,   beta = v / c.
    The second sum is the blaze-slope term: a Doppler shift moves every line along the blaze function, so the lines'
    relative weights change and the *global* centroid moves even where no line moved.  SURVEY 8(c) G14 wrote the slope
    without it (sum w X' lam / c); on this crop that formula is off by 5.9e-5 px at 10 m/s, the full one by < 2e-8 px."""
    v = np.array(W.RV_SWEEP_V)
    beta = v / W.C_LIGHT
    xc, xs, frames = [], [], []
    for vv in W.RV_SWEEP_V:
        s = _rv_crop(vv)
        lam, x, y, w = oracle.samples(s, 0, 0)
        i0 = int(x.min()) - 12
        wn = int(x.max()) + 12 - i0
        fr = oracle.render(s, window=(i0, 100, wn, 80))
        cols = i0 + np.arange(wn)
        xc.append(float((fr.sum(axis=0) * cols).sum() / fr.sum()))
        xs.append(float((w * x).sum() / w.sum()))
        frames.append(fr)
    xc, xs = np.array(xc), np.array(xs)
    assert np.max(np.abs(xc - xs)) < 1e-9                                       # (i)
    A = np.vstack([v, np.ones_like(v)]).T
    coef, *_ = np.linalg.lstsq(A, xc, rcond=None)
    assert np.max(np.abs(xc - A @ coef)) < 1e-6                                 # (ii) global
    cen = W.rv_sweep(0.0).notes["line_centers"]
    cen = cen[(cen > 5010.0) & (cen < 5014.0)]
    assert len(cen) == 16
    X = lambda l: 1024 + 1000 * ((l - 5025) / 25) + ((l - 5025) / 25) ** 2      # Tiny recipe
    Xp = lambda l: (1000 + 2 * ((l - 5025) / 25)) / 25

    def E(l):                                                                  # G7 blaze, m = 100, lam_c = 5025
        a = np.pi * 100 * (5025.0 / l - 1)
        return (np.sin(a) / a) ** 2
    edges = np.round(0.5 * (X(cen)[1:] + X(cen)[:-1])).astype(int) - i0
    for ell in (1, 7, 14):                                                      # (ii) per line
        c0, c1 = edges[ell - 1], edges[ell]
        pcs = np.array([float((f[:, c0:c1].sum(axis=0) * np.arange(c0, c1)).sum() / f[:, c0:c1].sum()) for f in frames])
        coef, *_ = np.linalg.lstsq(A, pcs, rcond=None)
        assert np.max(np.abs(pcs - A @ coef)) < 1e-6
        assert 5e-3 < pcs[-1] - pcs[0] < 8e-3                                   # ~ lam X' beta = 6.7e-3 px at 10 m/s
    h = 1e-4
    Ep = (E(cen + h) - E(cen - h)) / (2 * h)
    Wl = E(cen)
    xbar = (Wl * X(cen)).sum() / Wl.sum()
    slope = ((Wl * cen * Xp(cen)).sum() + (Ep * cen * (X(cen) - xbar)).sum()) / Wl.sum()
    assert np.max(np.abs((xc - xc[0]) - slope * beta)) < 1e-7                   # (iii) full closed form
    naive = (Wl * cen * Xp(cen)).sum() / Wl.sum()
    assert abs((xc[-1] - xc[0]) - naive * beta[-1]) > 1e-5                      # the survey's formula misses the blaze term
