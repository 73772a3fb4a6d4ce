"""Pins for the oracle's pixel-integrated PSF (step a4, pins P1 P2 P3 P4 P6 P11).
Every expected value here comes from something other than the oracle: mpmath brute force (golden file),
scipy closed forms, analytic moments, Poisson-summation closed form, the paper's own sub-pixel scheme."""
from pathlib import Path

import numpy as np
import pytest
from scipy import special

import oracle
from paper_2008_05858_b200 import workloads as W
from paper_2008_05858_b200.workloads import Psf

GOLD = Path(__file__).parent / "golden"


def _stamp(psf, xk, yk, t=7.5):
    """all pixels of the G9 footprint of a sample at (xk, yk): returns (i, j, P[j][i])"""
    Hx = 0.5 * psf.fiber_dx_px + t * psf.sigma_x
    Hy = 0.5 * psf.fiber_dy_px + t * psf.sigma_y
    i = np.arange(int(np.ceil(xk - Hx - 0.5)), int(np.floor(xk + Hx + 0.5)) + 1)
    j = np.arange(int(np.ceil(yk - Hy - 0.5)), int(np.floor(yk + Hy + 0.5)) + 1)
    P = np.array([[oracle.psf_pixel(psf, float(ii - xk), float(jj - yk)) for ii in i] for jj in j])
    return i, j, P


def test_p1_polar_quadrature_golden():
    """P1: oracle == 30-digit 2-D polar quadrature of the definition, incl. an asymmetric PSF."""
    rows = [l.split() for l in (GOLD / "p1_polar_quadrature.txt").read_text().splitlines() if not l.startswith("#")]
    assert len(rows) == 12
    for Dx, Dy, sx, sy, xk, yk, i, j, val in rows:
        psf = Psf(fiber_dx_px=float(Dx), fiber_dy_px=float(Dy), sigma_x=float(sx), sigma_y=float(sy))
        got = oracle.psf_pixel(psf, int(i) - float(xk), int(j) - float(yk))
        # far-wing pixels (1e-7 of the peak) carry ~4e-14 relative rounding from the double special functions
        assert got == pytest.approx(float(val), rel=2e-14, abs=1e-21), (Dx, Dy, sx, sy, i, j)


def test_p2_pure_gaussian_is_erf_product():
    """P2: Dx = Dy = 0 reduces to the textbook product of two erf differences (scipy.special.ndtr)."""
    psf = Psf(fiber_dx_px=0.0, fiber_dy_px=0.0, sigma_x=0.8, sigma_y=1.3)
    for u, v in [(0.2, -0.4), (3.3, 1.1), (-2.6, 4.9), (6.1, -7.7)]:
        ref = (special.ndtr((u + 0.5) / 0.8) - special.ndtr((u - 0.5) / 0.8)) * \
              (special.ndtr((v + 0.5) / 1.3) - special.ndtr((v - 0.5) / 1.3))
        assert oracle.psf_pixel(psf, u, v) == pytest.approx(ref, rel=1e-11, abs=1e-17)


def test_small_fiber_limit_approaches_gaussian():
    """a vanishing fiber (D -> 0) must approach the pure gaussian: P_D - P_0 = O(D^2)"""
    u, v = 0.7, -1.2
    p0 = oracle.psf_pixel(Psf(fiber_dx_px=0, fiber_dy_px=0, sigma_x=1.0, sigma_y=1.0), u, v)
    d1 = oracle.psf_pixel(Psf(fiber_dx_px=0.02, fiber_dy_px=0.02, sigma_x=1.0, sigma_y=1.0), u, v) - p0
    d2 = oracle.psf_pixel(Psf(fiber_dx_px=0.01, fiber_dy_px=0.01, sigma_x=1.0, sigma_y=1.0), u, v) - p0
    assert abs(d1) < 1e-4 and d1 / d2 == pytest.approx(4.0, rel=1e-2)


@pytest.mark.parametrize("D,sigma", [(3.0, 1.0), (4.0, 1.2)])
def test_p3_single_sample_flux(D, sigma):
    """P3: sum of P over the footprint = 1 - tail, tail <= 1.3e-13 at t = 7.5 (G9)."""
    psf = Psf(fiber_dx_px=D, fiber_dy_px=D, sigma_x=sigma, sigma_y=sigma)
    _, _, P = _stamp(psf, 10.3173, 7.8641)
    tot = float(np.sum(np.sort(P.ravel())))
    assert 0.0 <= 1.0 - tot < 1.5e-13


def _epsilon(xk, R, sigma, nmax=6):
    """photocenter offset of a pixel-sampled, pixel-integrated profile (Poisson summation):
    eps = (1/pi) sum_n ((-1)^n / n) phat(n) sin(2 pi n xk), phat(n) = exp(-2 pi^2 sigma^2 n^2) 2 J1(2 pi R n)/(2 pi R n)"""
    n = np.arange(1, nmax + 1)
    arg = 2 * np.pi * R * n
    phat = np.exp(-2 * np.pi ** 2 * sigma ** 2 * n ** 2) * 2 * special.j1(arg) / arg
    return float(np.sum(((-1.0) ** n / n) * phat * np.sin(2 * np.pi * n * xk)) / np.pi)


@pytest.mark.parametrize("D,sigma,amp", [(3.0, 0.7, 7.5e-7), (3.0, 1.0, 3.2e-11)])
def test_p4_photocenter_of_one_sample(D, sigma, amp):
    """P4: photocenter lands on x_k up to the closed-form aliasing term (< 1e-5 px required)."""
    psf = Psf(fiber_dx_px=D, fiber_dy_px=D, sigma_x=sigma, sigma_y=sigma)
    worst = 0.0
    for xk, yk in [(10.3173, 7.8641), (10.25, 8.0), (10.6, 7.4)]:
        i, j, P = _stamp(psf, xk, yk)
        cx = float(np.sum(P * i[None, :]) / P.sum())
        cy = float(np.sum(P * j[:, None]) / P.sum())
        ex, ey = _epsilon(xk, D / 2, sigma), _epsilon(yk, D / 2, sigma)
        assert abs(cx - xk - ex) < 3e-12 and abs(cy - yk - ey) < 3e-12
        worst = max(worst, abs(cx - xk))
        assert abs(cx - xk) < 1e-5 and abs(cy - yk) < 1e-5
    assert worst == pytest.approx(amp, rel=0.35)       # the aliasing term has the magnitude the closed form predicts


def test_p6_second_moments_asymmetric():
    """P6: sum (i - x_k)^2 P = sigma_x^2 + a^2/4 + 1/12 and likewise in y with sigma_y, b (catches x/y swaps)."""
    psf = Psf(fiber_dx_px=5.0, fiber_dy_px=2.0, sigma_x=0.9, sigma_y=1.4)
    xk, yk = 20.75, 15.125
    i, j, P = _stamp(psf, xk, yk)
    mx = float(np.sum(P * (i[None, :] - xk) ** 2))
    my = float(np.sum(P * (j[:, None] - yk) ** 2))
    assert mx == pytest.approx(0.9 ** 2 + 2.5 ** 2 / 4 + 1 / 12, abs=5e-10)
    assert my == pytest.approx(1.4 ** 2 + 1.0 ** 2 / 4 + 1 / 12, abs=5e-10)


def test_quadrature_order_converged():
    """the chord quadrature is converged at the oracle's Q = 32: Q = 48 changes nothing at 1e-15 of the peak"""
    psf = Psf(fiber_dx_px=4.0, fiber_dy_px=4.0, sigma_x=1.2, sigma_y=1.2)
    peak = oracle.psf_pixel(psf, 0.0, 0.0)
    for u, v in [(0.3, -0.1), (2.7, 1.9), (-5.2, 6.3), (9.9, 0.4)]:
        assert abs(oracle.psf_pixel(psf, u, v, 32) - oracle.psf_pixel(psf, u, v, 48)) < 2e-15 * peak


def test_p11_papers_subpixel_scheme():
    """P11: the paper's own discretisation (0.1-px sub-pixels, one thread each, summed per pixel)
    applied to the fiber (x) PSF *density* agrees with the exact pixel integral to <= 4e-3 per pixel,
    ~1e-14 in total flux and < 1e-11 px in photocenter.  The density is computed here with Gauss-Legendre in the
    ellipse angle (numpy/scipy only), independently of the oracle."""
    R, sigma = 1.5, 1.0
    psf = Psf(fiber_dx_px=2 * R, fiber_dy_px=2 * R, sigma_x=sigma, sigma_y=sigma)
    xk, yk = 10.3173, 7.8641
    i, j, P = _stamp(psf, xk, yk)
    # density(x, y) = 1/(pi R^2) int_{-R}^{R} g(x - s) [Phi((y + c(s))/sig) - Phi((y - c(s))/sig)] ds, s = R sin(phi)
    gl_x, gl_w = np.polynomial.legendre.leggauss(96)
    phi = 0.5 * np.pi * gl_x
    s = R * np.sin(phi)
    c = R * np.cos(phi)
    ws = gl_w * 0.5 * np.pi * R * np.cos(phi)
    sub = (np.arange(10) + 0.5) / 10.0 - 0.5                 # 0.1-px midpoints inside a pixel
    xs = (i[:, None] + sub[None, :]).ravel() - xk            # all sub-pixel abscissae
    ys = (j[:, None] + sub[None, :]).ravel() - yk
    gx = np.exp(-0.5 * ((xs[:, None] - s[None, :]) / sigma) ** 2) / (np.sqrt(2 * np.pi) * sigma)      # [nxs, nodes]
    fy = special.ndtr((ys[:, None] + c[None, :]) / sigma) - special.ndtr((ys[:, None] - c[None, :]) / sigma)
    dens = (fy * ws[None, :]) @ gx.T / (np.pi * R * R)                                                # [nys, nxs]
    papers = dens.reshape(len(j), 10, len(i), 10).sum(axis=(1, 3)) * 0.01
    big = P > 1e-3 * P.max()
    assert np.max(np.abs(papers[big] / P[big] - 1.0)) < 4e-3
    assert np.max(np.abs(papers[big] / P[big] - 1.0)) > 1e-5     # it IS a different (2nd-order) method
    assert abs(papers.sum() - P.sum()) < 1e-13
    cx_p = np.sum(papers * i[None, :]) / papers.sum()
    cx_o = np.sum(P * i[None, :]) / P.sum()
    assert abs(cx_p - cx_o) < 1e-11


# ------------------------------------------------------------------------------------------ G21: analytic PSF map
def _map_scene(gx=3, gy=2, nx=200, ny=80, x_pos=100.3173, y_pos=37.8641):
    d = W.single_line_scene(x_pos=x_pos, y_pos=y_pos, nx=nx, ny=ny)
    return W.psf_map(d, gx=gx, gy=gy, seed=6)


def _bilinear_nodes(gx, gy, nx, ny, x, y):
    """independent restatement of the node rule (T3 / G21): nodes at g (nx-1)/(gx-1), weights clamped outside"""
    tx = min(max(x * (gx - 1) / (nx - 1), 0.0), gx - 1.0) if gx > 1 else 0.0
    ty = min(max(y * (gy - 1) / (ny - 1), 0.0), gy - 1.0) if gy > 1 else 0.0
    g0 = min(int(np.floor(tx)), max(gx - 2, 0)); h0 = min(int(np.floor(ty)), max(gy - 2, 0))
    fx, fy = tx - g0, ty - h0
    g1, h1 = (g0 + 1 if gx > 1 else g0), (h0 + 1 if gy > 1 else h0)
    return [((h0, g0), (1 - fy) * (1 - fx)), ((h0, g1), (1 - fy) * fx), ((h1, g0), fy * (1 - fx)), ((h1, g1), fy * fx)]


def test_g21_map_pixel_is_the_mixture_of_the_pinned_constant_psfs():
    """G21: the blended PSF = sum over the 4 surrounding nodes of beta_c P(u, v; sigma_c).  Right-hand side: the constant-sigma
    pixel integral (pinned by P1, P2, P6) per node and bilinear weights restated here in numpy.  Asymmetric maps (sigma_x !=
    sigma_y, gx != gy): a transposed grid, swapped weights or a swapped axis fails"""
    import copy
    for (xp, yp) in [(100.3173, 37.8641), (12.9, 70.2), (199.0, 0.0), (150.0, 79.0), (-3.5, 40.0), (57.25, 95.0)]:
        d = _map_scene(x_pos=xp, y_pos=yp)
        q = d.psf
        nodes = _bilinear_nodes(q.an_gx, q.an_gy, d.nx, d.ny, xp, yp)
        assert abs(sum(b for _, b in nodes) - 1.0) < 1e-15
        for (i, j) in [(int(round(xp)), int(round(yp))), (int(round(xp)) + 3, int(round(yp)) - 2), (int(round(xp)) - 6, int(round(yp)) + 1)]:
            want = 0.0
            for (h, g), beta in nodes:
                c = copy.copy(q)
                c.an_sigma_x = c.an_sigma_y = None
                c.sigma_x, c.sigma_y = float(q.an_sigma_x[h, g]), float(q.an_sigma_y[h, g])
                want += beta * oracle.psf_pixel(c, i - xp, j - yp)
            assert oracle.psf_map_pixel(d, xp, yp, i, j) == pytest.approx(want, rel=2e-15, abs=1e-300)


def test_g21_map_with_equal_nodes_is_the_constant_psf():
    d = W.single_line_scene(x_pos=100.3173, y_pos=37.8641)
    m = W.psf_map(d, gx=3, gy=3, growth=0.0, jitter=0.0)
    assert np.all(m.psf.an_sigma_x == d.psf.sigma_x) and np.all(m.psf.an_sigma_y == d.psf.sigma_y)
    A, Bm = oracle.render(d), oracle.render(m)
    assert A.max() > 0 and np.allclose(Bm, A, rtol=1e-15, atol=0.0)


def test_g21_map_moments_box_and_flux():
    """per-sample second moments of a mixture = sum beta (sigma^2) + a^2/4 + 1/12 per axis (P6 for every node), the footprint box
    comes from the LARGEST node sigma (one box for the frame), flux = 1 - tail"""
    d = _map_scene(gx=3, gy=2)
    q = d.psf
    xp, yp = 100.3173, 37.8641
    fr = oracle.render(d)
    w = oracle.total_weight(d)
    P = fr / w
    assert abs(P.sum() - 1.0) < 2e-13
    jj, ii = np.mgrid[0:d.ny, 0:d.nx]
    nodes = _bilinear_nodes(q.an_gx, q.an_gy, d.nx, d.ny, xp, yp)
    a = 0.5 * q.fiber_dx_px
    vx = sum(b * q.an_sigma_x[h, g] ** 2 for (h, g), b in nodes) + a * a / 4 + 1 / 12
    vy = sum(b * q.an_sigma_y[h, g] ** 2 for (h, g), b in nodes) + (0.5 * q.fiber_dy_px) ** 2 / 4 + 1 / 12
    assert abs((P * (ii - xp) ** 2).sum() - vx) < 1e-9
    assert abs((P * (jj - yp) ** 2).sum() - vy) < 1e-9
    assert abs(vx - vy) > 1e-3                                         # the map is asymmetric: an x/y swap would show
    hbx = 0.5 * q.fiber_dx_px + q.support_nsigma * q.an_sigma_x.max() + 0.5
    hby = 0.5 * q.fiber_dy_px + q.support_nsigma * q.an_sigma_y.max() + 0.5
    nz = np.nonzero(fr)
    assert (nz[1].min(), nz[1].max()) == (int(np.ceil(xp - hbx)), int(np.floor(xp + hbx)))
    assert (nz[0].min(), nz[0].max()) == (int(np.ceil(yp - hby)), int(np.floor(yp + hby)))
    assert oracle.footprint(d, xp, yp) == (int(np.ceil(xp - hbx)), int(np.floor(xp + hbx)), int(np.ceil(yp - hby)), int(np.floor(yp + hby)))


def test_g21_map_render_is_linear_in_the_node_psfs():
    """frame(map) = sum_c frame(weights beta_c, constant sigma_c): checked by rendering a multi-sample strip whose samples
    cross a node boundary, against the per-pixel mixture"""
    s = W.tiny(samples_per_px=2.0)
    s.lam_min = np.array([5020.0]); s.lam_max = np.array([5030.0])          # x = 824 .. 1224: crosses the node at x = 1023.5
    m = W.psf_map(s, gx=3, gy=2, seed=9)
    fr = oracle.render(m)
    lam, x, y, w = oracle.samples(m, 0, 0)
    g0s = {_bilinear_nodes(3, 2, m.nx, m.ny, xx, yy)[0][0][1] for xx, yy in zip(x, y)}
    assert g0s == {0, 1}
    rng = np.random.default_rng(0)
    for _ in range(6):
        i = int(rng.integers(int(x.min()) + 12, int(x.max()) - 12)); j = int(round(128 + 0.01 * i)) + int(rng.integers(-3, 4))
        want = sum(wk * oracle.psf_map_pixel(m, xk, yk, i, j) for xk, yk, wk in zip(x, y, w)
                   if oracle.footprint(m, xk, yk)[0] <= i <= oracle.footprint(m, xk, yk)[1])
        assert fr[j, i] == pytest.approx(want, rel=1e-13)
