"""Parametric Spectrograph Unit (G22).

(1) the oracle's closed forms (oracle/spectrograph.py) against textbook echelle relations;
(2) the library's e2e_spectrograph_format (host code of libe2e.so, no GPU needed) against the oracle: the degree-(5,5)
    format polynomials reproduce the closed-form positions within the residual the call reports, the per-order tables and
    fiber images agree to rounding."""
import numpy as np
import pytest

from oracle import spectrograph as OS

R2 = dict(groove_um=1000.0 / 52.6, blaze_deg=63.4, theta_deg=0.7, gamma_deg=0.9, xd_groove_um=1000.0 / 300.0, xd_lam_ref=5500.0,
          f_cam_mm=300.0, f_coll_mm=1200.0, pixel_um=15.0, fiber_core_um=200.0, m_lo=50, m_hi=90, x_c=2048.0, y_c=2048.0,
          fiber_height_um=(-300.0, 0.0, 300.0))
R4 = dict(groove_um=1000.0 / 31.6, blaze_deg=76.0, theta_deg=0.8, gamma_deg=1.2, xd_groove_um=1000.0 / 400.0, xd_lam_ref=5500.0,
          f_cam_mm=460.0, f_coll_mm=1500.0, pixel_um=10.0, fiber_core_um=130.0, m_lo=78, m_hi=162, x_c=4608.0, y_c=4608.0,
          fiber_height_um=(-80.0, 80.0))


def test_oracle_echelle_closed_forms():
    p = OS.Spectrograph(**R2)
    d = p.groove_um * 1e4
    # Littrow (theta = gamma = 0): the classic blaze relation m lam_c = 2 d sin(blaze)
    lit = OS.Spectrograph(**{**R2, "theta_deg": 0.0, "gamma_deg": 0.0})
    assert OS.blaze_constant(lit) == pytest.approx(2.0 * d * np.sin(np.deg2rad(63.4)), rel=1e-15)
    m, lam_c, lmin, lmax = OS.order_table(p)
    K = OS.blaze_constant(p)
    assert np.allclose(m * lam_c, K, rtol=1e-15)
    assert np.allclose(lmax - lmin, K / (m * m - 0.25), rtol=1e-13)              # free spectral range
    assert np.allclose(lmin[:-1], lmax[1:], rtol=1e-15)                          # orders tile the spectrum
    # every blaze peak lands on x_c, whatever the order; the grating equation holds for the returned angle
    assert np.allclose(OS.position_x(p, lam_c, m), p.x_c, atol=1e-8)
    lam = np.linspace(lmin[7], lmax[7], 11)
    b = OS.beta(p, lam, m[7])
    alpha = np.deg2rad(63.4 + 0.7)
    assert np.allclose(m[7] * lam, d * np.cos(np.deg2rad(0.9)) * (np.sin(alpha) + np.sin(b)), rtol=1e-14)
    # angular dispersion d beta / d lam = m / (d cos gamma cos beta)  ->  linear dispersion at the blaze peak
    h = 1e-3
    num = (OS.position_x(p, lam_c + h, m) - OS.position_x(p, lam_c - h, m)) / (2 * h)
    beta_c = np.deg2rad(63.4 - 0.7)
    assert np.allclose(num, OS.px_per_radian(p) * m / (d * np.cos(np.deg2rad(0.9)) * np.cos(beta_c)), rtol=1e-8)
    # x grows with wavelength inside an order and spans about F * FSR * dispersion
    assert np.all(np.diff(OS.position_x(p, lam, m[7])) > 0)


def test_oracle_cross_disperser_and_fibers():
    p = OS.Spectrograph(**R2)
    dx = p.xd_groove_um * 1e4
    assert OS.position_y(p, p.xd_lam_ref) == pytest.approx(p.y_c, abs=1e-9)      # Littrow wavelength on row y_c
    lam = np.linspace(4000.0, 7000.0, 13)
    assert np.all(np.diff(OS.position_y(p, lam)) > 0)
    h = 1e-3
    num = (OS.position_y(p, p.xd_lam_ref + h) - OS.position_y(p, p.xd_lam_ref - h)) / (2 * h)
    assert num == pytest.approx(OS.px_per_radian(p) / (dx * np.cos(OS.beta_x(p, p.xd_lam_ref))), rel=1e-8)
    Dx, Dy, dxf, dyf, tan_chi = OS.fiber_images(p)
    assert Dy == pytest.approx(200.0 * 300.0 / 1200.0 / 15.0)
    assert 0.9 * Dy < Dx < Dy                                                    # anamorphic demagnification for alpha > beta
    assert np.allclose(dyf, np.array([-300.0, 0.0, 300.0]) * 300.0 / 1200.0 / 15.0)
    assert np.allclose(dxf, tan_chi * dyf)
    lit = OS.Spectrograph(**{**R2, "theta_deg": 0.0})
    assert OS.fiber_images(lit)[4] == pytest.approx(2.0 * np.tan(np.deg2rad(63.4)) * np.tan(np.deg2rad(0.9)), rel=1e-14)
    assert OS.blaze_peak_amplitude(p) == pytest.approx(np.cos(np.deg2rad(64.1)) / np.cos(np.deg2rad(62.7)))


def _poly(c, L, M):
    import mpmath as mp
    acc = mp.mpf(0)
    for pp in range(5, -1, -1):
        inner = mp.mpf(0)
        for q in range(5, -1, -1):
            inner = inner * M + mp.mpf(float(c[pp * 6 + q]))
        acc = acc * L + inner
    return acc


@pytest.mark.parametrize("case,rx_max,ry_max", [("R2", 2e-4, 2e-3), ("R4", 0.1, 2e-3)])
def test_library_format_reproduces_the_closed_forms(case, rx_max, ry_max):
    """e2e_spectrograph_format (libe2e.so host code) against the oracle: per-order tables to rounding, positions from the
    stored degree-(5,5) polynomials (evaluated here in 30-digit arithmetic) within the residual the call itself reports"""
    import mpmath as mp
    from paper_2008_05858_b200 import binding as B, build
    build.build()
    mp.mp.dps = 30
    kw = R2 if case == "R2" else R4
    p = OS.Spectrograph(**kw)
    r = B.e2e_spectrograph_format(**kw)
    m, lam_c, lmin, lmax = OS.order_table(p)
    assert r["n_orders"] == len(m) and np.array_equal(r["order_m"], m) and (r["deg_l"], r["deg_m"]) == (5, 5)
    for got, want in ((r["blaze_lam_c"], lam_c), (r["lam_min"], lmin), (r["lam_max"], lmax)):
        assert np.allclose(got, want, rtol=1e-14, atol=0.0)
    assert np.allclose(r["blaze_amp"], OS.blaze_peak_amplitude(p), rtol=1e-14)
    assert r["K"] == pytest.approx(OS.blaze_constant(p), rel=1e-14)
    Dx, Dy, dxf, dyf, tan_chi = OS.fiber_images(p)
    assert r["fiber_dx_px"] == pytest.approx(Dx, rel=1e-13) and r["fiber_dy_px"] == pytest.approx(Dy, rel=1e-13)
    assert np.allclose(r["fiber_dx"], dxf, rtol=1e-13, atol=1e-15) and np.allclose(r["fiber_dy"], dyf, rtol=1e-13, atol=1e-15)
    assert r["tilt_tan"] == pytest.approx(tan_chi, rel=1e-13)
    assert r["residual_x_px"] < rx_max and r["residual_y_px"] < ry_max
    worst_x = worst_y = 0.0
    rng = np.random.default_rng(4)
    for o in list(range(0, len(m), max(1, len(m) // 9))) + [len(m) - 1]:
        for lam in np.concatenate([[lmin[o], lmax[o], lam_c[o]], rng.uniform(lmin[o], lmax[o], 4)]):
            L = (mp.mpf(float(lam)) - mp.mpf(r["lam0"])) * mp.mpf(r["inv_dlam"])
            M = (mp.mpf(int(m[o])) - mp.mpf(r["m0"])) * mp.mpf(r["inv_dm"])
            worst_x = max(worst_x, abs(float(_poly(r["coef_x"], L, M)) - float(OS.position_x(p, lam, m[o]))))
            worst_y = max(worst_y, abs(float(_poly(r["coef_y"], L, M)) - float(OS.position_y(p, lam))))
    assert worst_x <= r["residual_x_px"] * 1.05 + 1e-6 and worst_y <= r["residual_y_px"] * 1.05 + 1e-6
    assert r["x_min"] == pytest.approx(float(OS.position_x(p, lmin, m).min()), abs=1e-6)
    assert r["x_max"] == pytest.approx(float(OS.position_x(p, lmax, m).max()), abs=1e-6)


def test_library_rejects_bad_parameters():
    from paper_2008_05858_b200 import binding as B, build
    build.build()
    with pytest.raises(B.E2EError):
        B.e2e_spectrograph_format(**{**R2, "groove_um": -1.0})
    with pytest.raises(B.E2EError):
        B.e2e_spectrograph_format(**{**R2, "m_lo": 90, "m_hi": 50})
    with pytest.raises(B.E2EError):
        B.e2e_spectrograph_format(**{**R2, "blaze_deg": 89.5, "theta_deg": 0.0, "m_lo": 2, "m_hi": 3})   # beta reaches 90 degrees
