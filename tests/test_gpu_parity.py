"""-m gpu: the CUDA path (through the C ABI of include/e2e.h) against the CPU oracle, element by element, on the
same seeded inputs.  Bars (BASELINE.json north_star, G8/G10/G12):
  * a1/a3  lam_k, x_k, y_k : bit-exact (the footprint boxes depend on them)
  * a2     w_k             : 4e-15 relative (libm sin vs CUDA sin differ in the last ulp)
  * a4/a5  frame           : |G - O| <= 1e-10 |O| + 1e-14 max(O) per pixel
  * a6     detector        : bit-exact
"""
import copy

import numpy as np
import pytest

import oracle
from paper_2008_05858_b200 import workloads as W
from parity_util import assert_frame_parity, frame_errors, photocenter_x, photocenter_y, with_psf

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2008_05858_b200 import build, binding
    build.build()
    binding.load()
    return binding


def gpu_render(B, scene, **kw):
    r = B.Renderer(scene)
    try:
        fr = r.render(**kw)
        r.torch.cuda.synchronize()
        return fr.cpu().numpy()
    finally:
        r.close()


def small_tiny(spp=4.0, lam=(5010.0, 5013.0)):
    s = W.tiny(samples_per_px=spp)
    s.lam_min = np.array([lam[0]])
    s.lam_max = np.array([lam[1]])
    return s


# ------------------------------------------------------------------------------------------ a1-a3
@pytest.mark.parametrize("which", ["tiny", "espresso"])
def test_setup_samples_positions_bit_exact(B, which):
    if which == "tiny":
        s = W.tiny()
        pairs = [(0, 0)]
    else:
        s = W.espresso_like(n_obj_lines=200, table_dlam=0.01).subset(orders=[0, 41, 84])
        pairs = [(0, 0), (1, 1), (1, 2)]
    r = B.Renderer(s)
    try:
        per, tot = r.fmt.num_samples()
        for o in range(s.n_orders):
            assert int(per[o]) == oracle.order_nsamples(s, o)
        assert tot == int(per.sum()) * s.n_fibers
        for fiber, o in pairs:
            lam, x, y, w = r.samples(fiber, o)
            ol, ox, oy, ow = oracle.samples(s, fiber, o)
            assert np.array_equal(lam, ol)
            assert np.array_equal(x, ox)
            assert np.array_equal(y, oy)
            assert np.allclose(w, ow, rtol=4e-15, atol=0.0)
            assert np.count_nonzero(w) > (0.9 if fiber == 0 else 0.01) * len(w)      # fiber 1 is the Fabry-Perot comb
    finally:
        r.close()


def test_setup_samples_doppler_and_efficiency_table(B):
    s = small_tiny(spp=3.0)
    s.spectra[0].doppler = 1.0 + 10.0 / W.C_LIGHT
    s.eff_table = np.array([0.5, 0.55, 0.9, 0.7])
    s.eff_lam0, s.eff_dlam = 5005.0, 4.0
    r = B.Renderer(s)
    try:
        lam, x, y, w = r.samples(0, 0)
        ol, ox, oy, ow = oracle.samples(s, 0, 0)
        assert np.array_equal(x, ox) and np.array_equal(y, oy)
        assert np.allclose(w, ow, rtol=4e-15, atol=0.0)
    finally:
        r.close()


# ------------------------------------------------------------------------------------------ a4/a5 analytic
def test_render_tiny_full_parity(B):
    """BASELINE.json configs[0]: 80 000 samples, 19x19 footprints, whole 2048x256 frame element by element"""
    s = W.tiny()
    G = gpu_render(B, s)
    O = oracle.render(s)
    e = assert_frame_parity(G, O, "tiny")
    assert e["max_rel_core"] < 1e-11
    tot = oracle.total_weight(s)
    assert abs(G.sum() / tot - 1.0) < 1e-12                       # flux conservation on the GPU frame
    assert abs(photocenter_x(G) - photocenter_x(O)) < 1e-9
    assert abs(photocenter_y(G) - photocenter_y(O)) < 1e-9


@pytest.mark.parametrize("psf_kw", [
    dict(fiber_dx_px=0.0, fiber_dy_px=0.0, sigma_x=0.9, sigma_y=1.3),      # pure asymmetric gaussian: one term, 3 power tiles
    dict(fiber_dx_px=4.0, fiber_dy_px=4.0, sigma_x=1.2, sigma_y=1.2),      # ESPRESSO-like PSF: 2 power tiles
    dict(fiber_dx_px=5.0, fiber_dy_px=2.0, sigma_x=0.8, sigma_y=1.5),      # elliptical fiber image, asymmetric PSF
    dict(fiber_dx_px=3.0, fiber_dy_px=0.0, sigma_x=1.0, sigma_y=1.0),      # degenerate ellipse: Dy = 0
    dict(fiber_dx_px=8.0, fiber_dy_px=8.0, sigma_x=2.5, sigma_y=2.5),      # footprint 47 px: 6 x 6 tiles per window
    dict(fiber_dx_px=2.0, fiber_dy_px=2.0, sigma_x=0.45, sigma_y=0.45),    # narrow PSF: fine y-phase windows
])
def test_render_psf_variants_dense_sampling(B, psf_kw):
    """the PSF variants under dense sampling, where the two-kernel cell-moment path renders (the sparse-sampling test below takes
    the per-sample polynomial kernel): whole small frame against the oracle, kernel asserted by name"""
    s = with_psf(small_tiny(spp=16.0, lam=(5010.0, 5012.0)), **psf_kw)
    r = B.Renderer(s)
    try:
        assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"].startswith("cell_flush_wide_kernel<")
        G = r.render().cpu().numpy()
    finally:
        r.close()
    O = oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, str(psf_kw))


def test_render_three_power_tiles_on_a_frame_that_fills_the_gpu(B):
    """cell_flush_kernel<3> (x degree above 15, single-warp CTAs): a 44-strip frame with a pure asymmetric gaussian PSF,
    windows of fiber 1 against the oracle"""
    s = with_psf(W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=list(range(0, 85, 4))),
                 fiber_dx_px=0.0, fiber_dy_px=0.0, sigma_x=0.9, sigma_y=1.3)
    r = B.Renderer(s)
    try:
        assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"] == "cell_flush_kernel<3>"
        G = r.render().cpu().numpy()
    finally:
        r.close()
    for o, frac in ((0, 0.2), (10, 0.5), (21, 0.9)):
        n = oracle.order_nsamples(s, o)
        k = int(frac * (n - 1))
        lam, x, y, w = oracle.samples(s, 1, o, k, k + 1)
        i0, j0 = max(0, int(x[0]) - 24), max(0, int(y[0]) - 20)
        O = oracle.render(s, window=(i0, j0, 48, 40))
        assert O.max() > 0
        assert_frame_parity(G[j0:j0 + 40, i0:i0 + 48], O, f"window {i0},{j0}")


def test_render_is_deterministic_and_accumulates(B):
    s = small_tiny(spp=8.0, lam=(5010.0, 5020.0))
    r = B.Renderer(s)
    try:
        a = r.render().cpu().numpy()
        b = r.render().cpu().numpy()
        assert np.array_equal(a, b)
        f = r.render()
        r.render(frame=f, accumulate=True)              # adds chunk by chunk: same value up to summation order
        assert np.allclose(f.cpu().numpy(), a + a, rtol=1e-14, atol=1e-16 * a.max())
        g = r.render()
        r.render(frame=g, accumulate=True)
        assert np.array_equal(f.cpu().numpy(), g.cpu().numpy())
    finally:
        r.close()


def test_render_overwrites_a_dirty_frame_on_every_zero_fill_path(B):
    """accumulate = 0 must not depend on what the frame held.  Large frames of the two-kernel path are zero-filled inside
    cell_moment_kernel (16-byte stores, grid-stride), small ones, frames that are not 16-byte aligned and every other kernel by
    a memset: a NaN-poisoned frame must come out equal, bit for bit, to a render on top of an explicitly zeroed frame"""
    import torch
    big = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    for name, s in (("two-kernel path, fused zero-fill", big), ("small frame, memset", small_tiny(spp=8.0, lam=(5010.0, 5020.0)))):
        r = B.Renderer(s)
        try:
            n = s.nx * s.ny
            ref = torch.zeros((s.ny, s.nx), dtype=torch.float64, device="cuda")
            r.render(frame=ref, accumulate=True)
            buf = torch.full((n + 1,), float("nan"), dtype=torch.float64, device="cuda")
            aligned = buf[:n].view(s.ny, s.nx)
            r.render(frame=aligned)
            assert torch.equal(aligned, ref), name
            assert torch.isnan(buf[n]).item(), name                  # nothing written past the frame
            buf.fill_(float("nan"))
            odd = buf[1:].view(s.ny, s.nx)                           # 8-byte aligned only
            r.render(frame=odd)
            assert torch.equal(odd, ref), name + " (8-byte aligned frame)"
            assert torch.isnan(buf[0]).item(), name
        finally:
            r.close()


@pytest.mark.parametrize("psf_kw", [
    dict(fiber_dx_px=0.0, fiber_dy_px=0.0, sigma_x=0.9, sigma_y=1.3),      # P2: pure asymmetric gaussian
    dict(fiber_dx_px=4.0, fiber_dy_px=4.0, sigma_x=1.2, sigma_y=1.2),      # ESPRESSO-like PSF
    dict(fiber_dx_px=5.0, fiber_dy_px=2.0, sigma_x=0.8, sigma_y=1.5),      # elliptical fiber image, asymmetric PSF
    dict(fiber_dx_px=3.0, fiber_dy_px=0.0, sigma_x=1.0, sigma_y=1.0),      # degenerate ellipse: Dy = 0
    dict(fiber_dx_px=6.6, fiber_dy_px=6.6, sigma_x=1.0, sigma_y=1.0),      # R/sigma = 3.3: needs the larger auto Q
    dict(fiber_dx_px=3.0, fiber_dy_px=3.0, sigma_x=1.0, sigma_y=1.0, support_nsigma=4.0),   # narrow truncation box
    dict(fiber_dx_px=8.0, fiber_dy_px=8.0, sigma_x=2.5, sigma_y=2.5),      # footprint 47 px: multi-panel windows
])
def test_render_psf_variants(B, psf_kw):
    s = with_psf(small_tiny(spp=3.0, lam=(5010.0, 5012.0)), **psf_kw)
    r = B.Renderer(s)
    try:
        assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"].startswith("render_poly_kernel<")      # sparse sampling
    finally:
        r.close()
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, str(psf_kw))


def test_render_narrow_sigma_reaches_the_direct_kernel(B):
    """sigma = 0.2 px: no polynomial degree up to 24 reproduces the pixel-phase factors to 1e-17, so e2e_psf_create builds no
    tables and e2e_render_frame launches render_analytic_kernel (direct erfc / Psi evaluation) -- the kernel name is
    asserted, so this test really covers that fallback.  Dense and sparse sampling, pure gaussian and with a fiber image"""
    for spp, kw in ((6.0, dict(fiber_dx_px=0.0, fiber_dy_px=0.0, sigma_x=0.2, sigma_y=0.25)),
                    (0.7, dict(fiber_dx_px=2.0, fiber_dy_px=2.0, sigma_x=0.22, sigma_y=0.22))):
        s = with_psf(small_tiny(spp=spp, lam=(5010.0, 5012.0)), **kw)
        r = B.Renderer(s)
        try:
            assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"] == "render_analytic_kernel"
            G = r.render().cpu().numpy()
        finally:
            r.close()
        O = oracle.render(s)
        assert O.max() > 0
        assert_frame_parity(G, O, f"direct kernel {kw}")
        assert abs(G.sum() / oracle.total_weight(s) - 1.0) < 1e-12


@pytest.mark.parametrize("grid", [(2, 2), (3, 2), (1, 3), (4, 1)])
def test_render_psf_map(B, grid):
    """S8(f) 3 / DESIGN.md G21 (P:61 'PSF ... for each wavelength'): analytic PSF map, the PSF of a sample = bilinear blend of
    the 4 surrounding node PSFs.  Whole frame against the oracle per pixel: strips that cross node boundaries in x, a steep
    two-fiber scene that crosses them in y, and the single-sample scene (box from the largest node sigma)"""
    gx, gy = grid
    s = small_tiny(spp=8.0, lam=(5010.0, 5030.0))                      # x = 424 .. 1224 on 2048 columns
    s.fiber_dx = np.array([0.0, 0.4]); s.fiber_dy = np.array([-30.0, 41.5])
    s.spectra = [s.spectra[0], s.spectra[0]]
    s.coef_y = np.array([128.0, 150.0, 0.0, 0.0])                      # rows 68 .. 158 (+ fibers): crosses the y node at 127.5
    m = W.psf_map(s, gx=gx, gy=gy, seed=60 + gx)
    r = B.Renderer(m)
    try:
        assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"].endswith("map>")
        G = r.render().cpu().numpy()
        again = r.render().cpu().numpy()
        c = B.e2e_plan_check(r.fmt, r.psf)
    finally:
        r.close()
    assert np.array_equal(G, again)
    assert c["queue_conflicts"] == 0 and c["phase_conflicts"] == 0
    O = oracle.render(m)
    assert O.max() > 0
    e = assert_frame_parity(G, O, f"psf map {grid}")
    assert e["max_rel_core"] < 1e-11
    assert abs(G.sum() / oracle.total_weight(m) - 1.0) < 1e-12
    d = W.psf_map(W.single_line_scene(x_pos=100.3173, y_pos=37.8641), gx=gx, gy=gy, seed=6)
    Gd, Od = gpu_render(B, d), oracle.render(d)
    assert_frame_parity(Gd, Od, "psf map, single sample")
    assert np.array_equal(Gd != 0.0, Od != 0.0)                        # the common box (largest node sigma)


def test_render_psf_map_espresso_windows(B):
    """the ESPRESSO-like frame (7 orders of it) with a 3 x 3 PSF map: oracle windows at strip ends and inside, both fibers"""
    s = W.psf_map(W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 40, 41, 42, 83, 84]), gx=3, gy=3)
    G = gpu_render(B, s)
    assert np.isfinite(G).all()
    for o, frac in ((0, 0.002), (1, 0.5), (3, 0.4999), (4, 0.75), (6, 0.998)):
        n = oracle.order_nsamples(s, o)
        k = int(frac * (n - 1))
        lam, x, y, w = oracle.samples(s, 0, o, k, k + 1)
        i0, j0 = max(0, int(x[0]) - 16), max(0, int(y[0]) - 22)
        O = oracle.render(s, window=(i0, j0, 32, 44))
        assert O.max() > 0
        assert_frame_parity(G[j0:j0 + 44, i0:i0 + 32], O, f"psf map window {i0},{j0}")
    assert abs(float(G.sum(dtype=np.longdouble)) / oracle.total_weight(s) - 1.0) < 1e-12


def test_render_single_sample_is_the_psf_itself(B):
    d = W.single_line_scene(x_pos=100.3173, y_pos=37.8641)
    G = gpu_render(B, d)
    O = oracle.render(d)
    assert_frame_parity(G, O, "single sample")
    nz = np.nonzero(G)
    assert (nz[1].min(), nz[1].max(), nz[0].min(), nz[0].max()) == (91, 109, 29, 47)      # G9 box
    assert abs(photocenter_x(G) - 100.3173) < 1e-9 and abs(photocenter_y(G) - 37.8641) < 1e-9
    # tests/golden P1 value (mpmath polar quadrature of the definition)
    assert G[38, 100] == pytest.approx(oracle.psf_pixel(d.psf, 100 - 100.3173, 38 - 37.8641), rel=1e-12)


def test_render_detector_edges_and_offdetector(B):
    """G11: pixels outside the detector are dropped.  The clipped GPU frame is checked against the crop of an
    oracle frame rendered on a padded detector (same sub-pixel phases: the shift is a whole number of pixels),
    with the G10 tolerance taken from the unclipped frame's maximum."""
    for xp, yp in [(4.25, 3.75), (55.5, 36.0), (-30.0, 3.7), (0.0, 0.0), (59.0, 39.0), (-9.375, 20.0), (30.0, 48.25)]:
        d = W.single_line_scene(x_pos=xp, y_pos=yp, nx=60, ny=40, samples=3)
        G = gpu_render(B, d)
        O = oracle.render(d)
        pad = W.single_line_scene(x_pos=xp + 32.0, y_pos=yp + 32.0, nx=60 + 64, ny=40 + 64, samples=3)
        OP = oracle.render(pad)
        assert np.allclose(OP[32:72, 32:92], O, rtol=1e-12, atol=1e-30)
        if O.max() == 0.0:
            assert G.max() == 0.0 and G.min() == 0.0
        else:
            tol = 1e-10 * np.abs(O) + 1e-14 * OP.max()
            assert np.all(np.abs(G - O) <= tol), f"edge {xp},{yp}: {np.max(np.abs(G - O) / tol)}"


def test_render_overlapping_fibers_and_orders(B):
    """two fibers 5 px apart (overlapping strips) and two orders crossing the same columns 12 px apart:
    the schedule must serialise them; result == oracle, and == sum of single-fiber renders"""
    s = small_tiny(spp=4.0, lam=(5010.0, 5014.0))
    s.order_m = np.array([100, 101], dtype=np.int32)
    s.lam_min = np.array([5010.0, 5010.0]); s.lam_max = np.array([5014.0, 5014.0])
    s.blaze_lam_c = np.array([5025.0, 5015.0]); s.blaze_amp = np.array([1.0, 0.7])
    s.deg_m = 1
    s.coef_x = np.array([1024.0, 3.0, 1000.0, 0.0, 1.0, 0.0, 0.0, 0.0])          # c[p*2+q]
    s.coef_y = np.array([138.24, 12.0, 10.0, 0.0, 0.01, 0.0, 0.0, 0.0])
    s.fiber_dx = np.array([0.0, 0.3, -0.2]); s.fiber_dy = np.array([-5.0, 0.0, 5.0])
    sp = s.spectra[0]
    s.spectra = [sp, W.Spectrum(flux=sp.flux[::-1].copy(), lam0=sp.lam0, dlam=sp.dlam, scale=3e3), copy.copy(sp)]
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert_frame_parity(G, O, "3 fibers x 2 orders")
    parts = np.zeros_like(G)
    for f in range(3):
        parts += gpu_render(B, s.subset(fibers=[f]))
    assert np.allclose(G, parts, rtol=1e-13, atol=1e-16 * G.max())


def test_render_steep_and_reversed_traces(B):
    """x decreasing with lambda (monotone either way is legal) and a steep trace (dy/dx = 0.6)"""
    s = small_tiny(spp=5.0, lam=(5010.0, 5012.0))
    s.coef_x = np.array([1024.0, -1000.0, 1.0, 0.0])
    s.coef_y = np.array([128.0, 600.0, 0.0, 0.0])
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert_frame_parity(G, O, "reversed steep")


def test_render_sparse_sampling(B):
    """samples 2.5 px apart (spp = 0.4): chunk windows far wider than one panel"""
    s = small_tiny(spp=0.4, lam=(5005.0, 5045.0))
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert_frame_parity(G, O, "sparse")


def test_render_zero_and_negative_flux(B):
    s = small_tiny(spp=2.0)
    s.spectra = [W.Spectrum(flux=np.zeros(16), lam0=5000.0, dlam=4.0, scale=1.0)]
    assert np.all(gpu_render(B, s) == 0.0)
    rng = np.random.default_rng(3)
    s.spectra = [W.Spectrum(flux=rng.normal(size=400), lam0=5009.0, dlam=0.01, scale=1.0)]     # linear: negative flux legal
    G, O = gpu_render(B, s), oracle.render(s)
    e = frame_errors(G, O)
    assert e["max_abs_over_max"] < 1e-12


def test_format_rejects_non_monotone_x(B):
    s = small_tiny(spp=2.0, lam=(5000.0, 5050.0))
    s.coef_x = np.array([1024.0, 10.0, -600.0, 0.0])            # x = 1024 + 10 u - 600 u^2 turns over inside the order
    with pytest.raises(B.E2EError) as ei:
        B.Format(s)
    assert ei.value.code == -2


def test_workspace_errors(B):
    import torch
    s = small_tiny(spp=2.0)
    r = B.Renderer(s)
    try:
        fr = torch.empty((s.ny, s.nx), dtype=torch.float64, device="cuda")
        small = torch.empty(256, dtype=torch.uint8, device="cuda")
        with pytest.raises(B.E2EError) as ei:
            B.e2e_render_frame(r.fmt, r.psf, r.spectra, fr, False, small)
        assert ei.value.code == -6
    finally:
        r.close()


# ------------------------------------------------------------------------------------------ full-size ESPRESSO-like
@pytest.fixture(scope="module")
def espresso_gpu(B):
    s = W.espresso_like()
    r = B.Renderer(s)
    fr = r.render()
    r.torch.cuda.synchronize()
    G = fr.cpu().numpy()
    # full size, bench launch configuration: the frame is bit-reproducible render to render (the L2 reductions of one
    # pixel are ordered by the schedule and the warp barriers)
    for _ in range(2):
        again = r.render()
        r.torch.cuda.synchronize()
        assert r.torch.equal(again, r.torch.from_numpy(G).to(again.device))
    r.close()
    return s, G


def test_render_espresso_full_frame_windows(B, espresso_gpu):
    """BASELINE.json configs[1] at full size in the launch configuration bench.py times; the oracle computes
    sampled windows (both fibers, blue / middle / red orders, frame edges and the centre)"""
    s, G = espresso_gpu
    assert np.isfinite(G).all()
    rng = np.random.default_rng(11)
    wins = []
    for o in (0, 1, 40, 84):
        n = oracle.order_nsamples(s, o)
        for frac in (0.0005, rng.uniform(0.1, 0.9), 0.9995):
            k = int(frac * (n - 1))
            lam, x, y, w = oracle.samples(s, 0, o, k, k + 1)
            wins.append((max(0, int(x[0]) - 24), max(0, int(y[0]) - 20), 48, 40))
    # windows centred on the Fabry-Perot fiber (fiber 1), on one of its lines: found from the oracle's own weights
    for o in (17, 63):
        lam, x, y, w = oracle.samples(s, 1, o)
        k = int(np.argmax(w[len(w) // 3:]) + len(w) // 3)
        assert w[k] > 0
        wins.append((max(0, int(x[k]) - 24), max(0, int(y[k]) - 20), 48, 40))
    worst = 0.0
    for (i0, j0, wnx, wny) in wins:
        O = oracle.render(s, window=(i0, j0, wnx, wny))
        assert O.max() > 0
        e = assert_frame_parity(G[j0:j0 + wny, i0:i0 + wnx], O, f"window {i0},{j0}")
        worst = max(worst, e["max_tol_ratio"])
    assert worst <= 1.0


def test_render_espresso_whole_order_both_fibers(B, espresso_gpu):
    """one whole order (index 40, both fibers, all 9216 columns, every row either fiber touches) of the full-size frame
    against the oracle, element by element: ~577 k samples, several thousand footprint cells, both strip ends"""
    s, G = espresso_gpu
    o = 40
    n = oracle.order_nsamples(s, o)
    ys = np.concatenate([oracle.samples(s, f, o, k, k + 1)[2] for f in (0, 1) for k in range(0, n, n // 64)] +
                        [oracle.samples(s, f, o, n - 1, n)[2] for f in (0, 1)])
    j0, j1 = int(np.floor(ys.min())) - 16, int(np.ceil(ys.max())) + 16
    O = oracle.render(s, window=(0, j0, s.nx, j1 - j0))
    assert oracle.render.last_touched == 2 * n                      # every sample of both fibers is inside the window
    assert np.all(O[0] == 0.0) and np.all(O[-1] == 0.0)             # and nothing else reaches it (orders are 92 px apart)
    e = assert_frame_parity(G[j0:j1], O, "order 40, both fibers, full x range")
    assert e["max_rel_core"] < 1e-11


def test_render_espresso_flux_conservation_and_gaps(B, espresso_gpu):
    s, G = espresso_gpu
    tot = oracle.total_weight(s)
    assert abs(float(G.sum(dtype=np.longdouble)) / tot - 1.0) < 1e-12
    # between orders nothing is written: row 117 - 40 and the last rows are exactly zero
    assert np.all(G[:60] == 0.0)
    assert G.min() >= 0.0


def test_render_hires_full_frame_windows(B):
    """BASELINE.json configs[2] at full size (10 fibers x 60 orders, 173 M samples) in the launch configuration
    bench.py times; oracle on sampled windows that span several fibers of the pseudo-slit"""
    s = W.hires_like()
    G = gpu_render(B, s)
    assert np.isfinite(G).all()
    for o, f, frac in ((0, 0, 0.0008), (30, 4, 0.41), (59, 9, 0.9992), (12, 9, 0.27), (45, 0, 0.66), (58, 5, 0.05)):
        n = oracle.order_nsamples(s, o)
        k = int(frac * (n - 1))
        lam, x, y, w = oracle.samples(s, f, o, k, k + 1)
        i0, j0 = max(0, int(x[0]) - 12), max(0, int(y[0]) - 24)
        wnx, wny = min(24, s.nx - i0), min(48, s.ny - j0)
        O = oracle.render(s, window=(i0, j0, wnx, wny))
        assert O.max() > 0
        assert_frame_parity(G[j0:j0 + wny, i0:i0 + wnx], O, f"hires window {i0},{j0}")
    # the outer fibers of the last orders leave the detector (G11: dropped), so the frame holds a bit less than was injected
    ratio = float(G.sum(dtype=np.longdouble)) / oracle.total_weight(s)
    assert 0.9 < ratio <= 1.0 + 1e-12


# ------------------------------------------------------------------------------------------ a4/a5 tabulated
def small_field_scene(gx=3, gy=2, npix=7, os=4, seed=77, nx=300, ny=120):
    s = small_tiny(spp=3.0, lam=(5010.0, 5013.0))
    s.nx, s.ny = nx, ny
    s.coef_x = np.array([1590.0, 2400.0, 1.0, 0.0])       # x = 1590 + 2400 u: u = -0.6 -> 150.4 ; u = -0.48 -> 438
    s.lam_max = np.array([5012.5])                        # u = -0.5 -> 390 - ... keeps part of the trace off the detector (G11)
    s.coef_y = np.array([60.0, 40.0, 0.0, 0.0])
    tab = W.tabulated_kernels(seed=seed, npix=npix, os=os, gx=gx, gy=gy)
    s.psf = W.Psf(kind=1, tab_npix=npix, tab_os=os, tab_gx=gx, tab_gy=gy, tab=tab)
    return s


@pytest.mark.parametrize("grid", [(1, 1), (3, 2), (5, 5)])
def test_render_tabulated_small(B, grid):
    s = small_field_scene(gx=grid[0], gy=grid[1])
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, f"tabulated {grid}")


def test_render_tabulated_11px_8x(B):
    s = small_field_scene(gx=2, gy=2, npix=11, os=8)
    s.lam_max = np.array([5010.6])
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert_frame_parity(G, O, "tabulated 11 px x 8")


@pytest.mark.parametrize("npix,os", [(6, 3), (5, 16), (9, 1), (5, 20)])
def test_render_tabulated_shapes(B, npix, os):
    """even / odd kernel widths, non-power-of-two and unit oversampling (cell-deposit kernel), and an oversampling
    beyond its weight array (os = 20 -> per-sample lattice kernel)"""
    s = small_field_scene(gx=3, gy=3, npix=npix, os=os, seed=78)
    r = B.Renderer(s)
    try:
        assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"] == ("render_tabulated_kernel" if os > 16 else "render_tabcell_kernel")
        G = r.render().cpu().numpy()
    finally:
        r.close()
    O = oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, f"tabulated npix={npix} os={os}")


def test_render_tabulated_steep_trace_and_fibers(B):
    """cells that change row every few samples (steep trace) and two overlapping fibers through the tabulated path"""
    s = small_field_scene(gx=2, gy=3, npix=7, os=4, seed=79)
    s.coef_y = np.array([560.0, 900.0, 0.0, 0.0])         # y = 20 .. 128 over x = 150 .. 438: ~0.4 px of y per px of x
    s.fiber_dx = np.array([0.0, 0.3])
    s.fiber_dy = np.array([0.0, 2.5])
    s.spectra = [s.spectra[0], s.spectra[0]]
    G = gpu_render(B, s)
    O = oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, "tabulated steep trace, 2 fibers")


def test_render_field_psf_full_frame_windows(B):
    """BASELINE.json configs[3] at full size; oracle on sampled windows"""
    s = W.field_psf()                                             # the scene bench.py --workload field_psf times
    G = gpu_render(B, s)
    assert np.isfinite(G).all()
    for o, frac in ((0, 0.3), (42, 0.77), (84, 0.5), (21, 0.0007), (66, 0.9993)):
        n = oracle.order_nsamples(s, o)
        k = int(frac * (n - 1))
        lam, x, y, w = oracle.samples(s, 0, o, k, k + 1)
        i0, j0 = int(x[0]) - 8, int(y[0]) - 10
        O = oracle.render(s, window=(i0, j0, 16, 20))
        assert O.max() > 0
        assert_frame_parity(G[j0:j0 + 20, i0:i0 + 16], O, f"field window {i0},{j0}")
    tot = oracle.total_weight(s)
    assert abs(float(G.sum(dtype=np.longdouble)) / tot - 1.0) < 1e-11


# ------------------------------------------------------------------------------------------ host entry point
def test_render_frame_host_matches_device_path(B):
    import torch
    s = small_tiny(spp=4.0)
    r = B.Renderer(s)
    try:
        dev = r.render().cpu().numpy()
        host_tabs = [np.ascontiguousarray(sp.flux, dtype=np.float64) for sp in s.spectra]
        desc = B.spectra_array(s.spectra, [t.ctypes.data for t in host_tabs])
        nbytes = B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc)
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        out = torch.empty((s.ny, s.nx), dtype=torch.float64).pin_memory()
        B.e2e_render_frame_host(r.fmt, r.psf, desc, out.data_ptr(), ws)
        assert np.array_equal(out.numpy(), dev)
    finally:
        r.close()


def test_render_frame_host_banded_pipeline(B):
    """host entry point on a multi-order, two-fiber frame: rows travel to the host band by band while later bands
    render.  Every row must arrive; the frame equals the device path up to the order of the additions, and the
    detector stage (keyed by the pixel's index in the whole frame) matches the one-pass result"""
    import torch
    s = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    det = W.Detector(gain=1.0, dark_e=0.5, ron_e=3.0, bias=100.0, seed=424242)
    r = B.Renderer(s)
    try:
        d_frame = r.render()
        dev = d_frame.cpu().numpy()
        d_noisy = torch.empty_like(d_frame)
        B.e2e_apply_detector(d_frame, d_noisy, s.nx, s.ny, det)
        dev_noisy = d_noisy.cpu().numpy()
        host_tabs = [np.ascontiguousarray(sp.flux, dtype=np.float64) for sp in s.spectra]
        desc = B.spectra_array(s.spectra, [t.ctypes.data for t in host_tabs])
        nbytes = B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc)
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        out = torch.full((s.ny, s.nx), float("nan"), dtype=torch.float64).pin_memory()
        B.e2e_render_frame_host(r.fmt, r.psf, desc, out.data_ptr(), ws)
        H = out.numpy().copy()
        assert np.isfinite(H).all()                                   # every row was copied
        mx = dev.max()
        assert np.abs(H - dev).max() <= 1e-13 * mx
        assert np.array_equal(H == 0.0, dev == 0.0)
        # the host path against the ORACLE (not only against the device path): windows at strip ends, fiber overlaps, band seams
        for o, frac in ((0, 0.001), (1, 0.5), (3, 0.25), (4, 0.999), (6, 0.6)):
            n = oracle.order_nsamples(s, o)
            k = int(frac * (n - 1))
            lam, x, y, w = oracle.samples(s, 0, o, k, k + 1)
            i0, j0 = max(0, int(x[0]) - 24), max(0, int(y[0]) - 20)
            O = oracle.render(s, window=(i0, j0, 48, 40))
            assert O.max() > 0
            assert_frame_parity(H[j0:j0 + 40, i0:i0 + 48], O, f"host path window {i0},{j0}")
        out.fill_(float("nan"))
        B.e2e_render_frame_host(r.fmt, r.psf, desc, out.data_ptr(), ws, det=det)
        Hn = out.numpy()
        assert np.isfinite(Hn).all()
        # a6 of the host path is bit-exact against the oracle's detector stage applied to the host path's own noise-free frame
        assert np.array_equal(Hn, oracle.detector(H, det))
        # identical draws; a last-bit difference of mu can move a Poisson count only at a rounding boundary
        assert (Hn == dev_noisy).mean() > 0.9999
        assert np.abs(Hn - dev_noisy).max() <= 2.0
        # and the result is reproducible call to call
        again = torch.empty_like(out)
        B.e2e_render_frame_host(r.fmt, r.psf, desc, again.data_ptr(), ws, det=det)
        assert torch.equal(again, out)
    finally:
        r.close()


def test_render_frame_host_uploads_every_table_element_a_band_reads(B):
    """the host path sends the spectrum tables piece by piece, in the order the row bands read them, and a band waits only
    for its own wavelength range.  The workspace is poisoned with NaN before every call, so a band that read an element
    before it arrived (or one that never travelled) shows up as NaN; cases: fibers that share one host table under
    different Doppler factors, a table that covers only part of an order, a table shorter than any band's range, and a
    Doppler factor that moves every sample off the table"""
    import copy
    import torch
    base = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    sp0 = base.spectra[0]
    n = sp0.flux.shape[0]
    cases = []
    # one host table, two Doppler factors (+-300 km/s).  A 33-MB table (the bench's grid step): the part no band reads travels
    # last and takes ~0.6 ms, so an element a band needs that was left to that part is still NaN when the band reads it
    big = W.espresso_like(n_obj_lines=300).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    a = copy.copy(big)
    a.spectra = [Spectrum_like(big.spectra[0], doppler=1.0 + 1e-3), Spectrum_like(big.spectra[0], doppler=1.0 - 1e-3)]
    cases.append(("shared table, two doppler factors", a))
    b = copy.copy(base)                                              # tables that start / end inside the format's range
    cut = n // 3
    b.spectra = [Spectrum_like(sp0, flux=sp0.flux[cut:], lam0=sp0.lam0 + cut * sp0.dlam),
                 Spectrum_like(base.spectra[1], flux=base.spectra[1].flux[:2 * cut])]
    cases.append(("partial tables", b))
    c = copy.copy(base)                                              # 2-element table; every sample of fiber 1 off its table
    c.spectra = [Spectrum_like(sp0, flux=np.array([3.0, 5.0]), lam0=float(base.lam_min[3]), dlam=float(base.lam_max[3] - base.lam_min[3])),
                 Spectrum_like(base.spectra[1], doppler=3.0)]
    cases.append(("two-element table, fiber off its table", c))
    for name, s in cases:
        r = B.Renderer(s)
        try:
            dev = r.render().cpu().numpy()
            tabs = {}
            for sp in s.spectra:
                tabs.setdefault(id(sp.flux), torch.from_numpy(np.ascontiguousarray(sp.flux, dtype=np.float64)).pin_memory())
            desc = B.spectra_array(s.spectra, [tabs[id(sp.flux)].data_ptr() for sp in s.spectra])
            ws = torch.empty(B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc), dtype=torch.uint8, device="cuda")
            for rep in range(2):
                ws.view(torch.float64).fill_(float("nan"))
                out = torch.full((s.ny, s.nx), float("nan"), dtype=torch.float64).pin_memory()
                B.e2e_render_frame_host(r.fmt, r.psf, desc, out.data_ptr(), ws)
                H = out.numpy()
                assert np.isfinite(H).all(), name
                assert np.abs(H - dev).max() <= 1e-13 * max(dev.max(), 1e-300), name
                assert np.array_equal(H == 0.0, dev == 0.0), name
            if name.startswith("two-element"):
                assert dev.max() > 0                                 # order 3 of fiber 0 is lit, nothing else
        finally:
            r.close()


def Spectrum_like(sp, **kw):
    d = dict(flux=sp.flux, lam0=sp.lam0, dlam=sp.dlam, scale=sp.scale, doppler=sp.doppler)
    d.update(kw)
    return W.Spectrum(**d)


def test_render_frame_host_on_a_frame_that_fills_the_gpu(B):
    """the banded host path with the single-warp flush kernel (the 7-order scenes above are small frames and take the wide kernel):
    44 strips, host frame against the device path and against oracle windows at band seams, detector stage bit-exact"""
    import torch
    s = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=list(range(0, 85, 4)))
    det = W.Detector(gain=1.0, dark_e=0.5, ron_e=3.0, bias=100.0, seed=99)
    r = B.Renderer(s)
    try:
        assert B.e2e_render_kernel_info(r.fmt, r.psf)["name"] == "cell_flush_kernel<2>"
        assert B.e2e_plan_check(r.fmt, r.psf)["n_host_bands"] >= 4
        dev = r.render().cpu().numpy()
        host_tabs = [np.ascontiguousarray(sp.flux, dtype=np.float64) for sp in s.spectra]
        desc = B.spectra_array(s.spectra, [t.ctypes.data for t in host_tabs])
        ws = torch.empty(B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc), dtype=torch.uint8, device="cuda")
        ws.view(torch.float64).fill_(float("nan"))
        out = torch.full((s.ny, s.nx), float("nan"), dtype=torch.float64).pin_memory()
        B.e2e_render_frame_host(r.fmt, r.psf, desc, out.data_ptr(), ws)
        H = out.numpy().copy()
        assert np.isfinite(H).all()
        assert np.abs(H - dev).max() <= 1e-13 * dev.max()
        assert np.array_equal(H == 0.0, dev == 0.0)
        for o, frac in ((0, 0.5), (7, 0.01), (14, 0.99), (21, 0.4)):
            n = oracle.order_nsamples(s, o)
            k = int(frac * (n - 1))
            lam, x, y, w = oracle.samples(s, 0, o, k, k + 1)
            i0, j0 = max(0, int(x[0]) - 24), max(0, int(y[0]) - 20)
            O = oracle.render(s, window=(i0, j0, 48, 40))
            assert O.max() > 0
            assert_frame_parity(H[j0:j0 + 40, i0:i0 + 48], O, f"host path window {i0},{j0}")
        B.e2e_render_frame_host(r.fmt, r.psf, desc, out.data_ptr(), ws, det=det)
        assert np.array_equal(out.numpy(), oracle.detector(H, det))
    finally:
        r.close()


def test_render_frame_host_adu16_raw_frame(B):
    """e2e_render_frame_host_adu16 / _ex: the host path with the full detector stage (PRNU + dark maps, full well, cross-talk,
    ADC) delivering uint16 counts.  Bit-exact against the oracle's detector stage applied to the host path's own noise-free
    frame, band by band (the stream is keyed by the pixel's index in the whole frame)"""
    import torch
    s = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    for sp in s.spectra:
        sp.scale = sp.scale * 400.0                                   # bright enough to reach the well in line cores
    rng = np.random.default_rng(12)
    prnu = rng.normal(1.0, 0.02, (s.ny, s.nx))
    dark = rng.uniform(0.0, 2.0, (s.ny, s.nx))
    X = rng.uniform(0.0, 5e-4, (16, 16))
    det = W.Detector(gain=1.0, dark_e=0.5, ron_e=3.0, bias=1000.0, seed=777)
    r = B.Renderer(s)
    try:
        host_tabs = [np.ascontiguousarray(sp.flux, dtype=np.float64) for sp in s.spectra]
        desc = B.spectra_array(s.spectra, [t.ctypes.data for t in host_tabs])
        ws = torch.empty(B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc), dtype=torch.uint8, device="cuda")
        clean = torch.empty((s.ny, s.nx), dtype=torch.float64).pin_memory()
        B.e2e_render_frame_host(r.fmt, r.psf, desc, clean.data_ptr(), ws)
        H = clean.numpy().copy()
        assert H.max() > 1e3
        d_pr, d_dk = torch.from_numpy(prnu).cuda(), torch.from_numpy(dark).cuda()
        kw = dict(full_well_e=2.0e4, e_per_adu=1.1, adu_max=65535.0)
        okw = dict(full_well=2.0e4, e_per_adu=1.1, adu_max=65535.0)
        for xt in (None, X):
            d_ex, keep = B.detector_ex_desc(det, d_pr, d_dk, xtalk=xt, **kw)
            out16 = torch.zeros((s.ny, s.nx), dtype=torch.uint16).pin_memory()
            B.e2e_render_frame_host_ex(r.fmt, r.psf, desc, out16.data_ptr(), ws, d_ex, adu16=True)
            want = oracle.detector_adu16(H, det, prnu=prnu, dark=dark, xtalk=xt, **okw)
            assert np.array_equal(out16.numpy(), want), "uint16 host path" + (" with cross-talk" if xt is not None else "")
            out64 = torch.zeros((s.ny, s.nx), dtype=torch.float64).pin_memory()
            B.e2e_render_frame_host_ex(r.fmt, r.psf, desc, out64.data_ptr(), ws, d_ex)
            assert np.array_equal(out64.numpy(), want.astype(np.float64))
        assert want.max() > 1.9e4 / 1.1 and want.min() >= 900
        # reproducible call to call, and refused without an ADC
        again = torch.zeros_like(out16)
        B.e2e_render_frame_host_ex(r.fmt, r.psf, desc, again.data_ptr(), ws, d_ex, adu16=True)
        assert np.array_equal(again.numpy(), out16.numpy())
        bad, _ = B.detector_ex_desc(det)
        with pytest.raises(B.E2EError):
            B.e2e_render_frame_host_ex(r.fmt, r.psf, desc, again.data_ptr(), ws, bad, adu16=True)
    finally:
        r.close()


def test_concurrent_renders_on_two_streams_from_two_threads(B):
    """include/e2e.h: handles are read-only during render, so concurrent renders on different streams into different
    frames are legal.  Two host threads render two different scenes repeatedly on their own streams (the library's fork /
    join stream and events are shared between the calls); every frame must equal the serial result bit for bit"""
    import threading
    import torch
    sa = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 3, 40, 41, 42, 84])
    sb = small_tiny(spp=40.0, lam=(5005.0, 5045.0))
    ra, rb = B.Renderer(sa), B.Renderer(sb)
    try:
        ref_a, ref_b = ra.render().clone(), rb.render().clone()
        torch.cuda.synchronize()
        errors = []

        def work(r, ref, n):
            try:
                st = torch.cuda.Stream()
                fr = torch.empty_like(ref)
                for _ in range(n):
                    with torch.cuda.stream(st):
                        B.e2e_render_frame(r.fmt, r.psf, r.spectra, fr, False, r.workspace, st)
                    st.synchronize()
                    if not torch.equal(fr, ref):
                        errors.append("frame differs from the serial render")
                        return
            except Exception as e:                                  # noqa: BLE001
                errors.append(repr(e))

        ta = threading.Thread(target=work, args=(ra, ref_a, 6))
        tb = threading.Thread(target=work, args=(rb, ref_b, 40))
        ta.start(); tb.start(); ta.join(); tb.join()
        assert not errors, errors
    finally:
        ra.close(); rb.close()


# ------------------------------------------------------------------------------------------ a6 detector
def test_detector_bit_exact(B):
    import torch
    rng = np.random.default_rng(5)
    nx, ny = 333, 77
    fr = np.concatenate([np.zeros(1000), rng.uniform(0, 5, 5000), rng.uniform(5, 64, 5000), rng.uniform(64, 200, 5000),
                         rng.uniform(3e4, 5e4, nx * ny - 16000)])
    fr[17] = -3.0
    fr = fr.reshape(ny, nx)
    det = W.Detector(gain=0.9, dark_e=0.4, ron_e=3.0, bias=100.0, seed=0x1234_5678_9ABC_DEF0)
    d_in = torch.from_numpy(fr).cuda()
    d_out = torch.empty_like(d_in)
    B.e2e_apply_detector(d_in, d_out, nx, ny, det)
    G = d_out.cpu().numpy()
    O = oracle.detector(fr, det)
    assert np.array_equal(G, O)
    # in place, and independent of launch geometry: same result when applied to the same buffer
    B.e2e_apply_detector(d_in, d_in, nx, ny, det)
    assert np.array_equal(d_in.cpu().numpy(), O)
    assert abs(G[-1].mean() / (0.9 * fr[-1].mean() + 0.4 + 100.0) - 1.0) < 0.01
    # buffers that are only 8-byte aligned (the kernel's one-load-per-pixel-pair form does not apply), odd pixel count
    src = torch.empty(nx * ny + 1, dtype=torch.float64, device="cuda")
    dst = torch.full((nx * ny + 2,), -1.0, dtype=torch.float64, device="cuda")
    src[1:] = torch.from_numpy(fr).cuda().reshape(-1)
    B.e2e_apply_detector(src[1:], dst[1:-1], nx, ny, det)
    assert np.array_equal(dst[1:-1].cpu().numpy().reshape(ny, nx), O)
    assert dst[0].item() == -1.0 and dst[-1].item() == -1.0


def test_detector_pairs_that_straddle_host_bands(B):
    """G12 round 3 keys the noise stream by pixel PAIR; on a frame of odd width the row bands of the host path start at odd
    pixel indices, so a pair's two pixels land in different launches.  Still bit-exact against the oracle's stage applied to
    the host path's own noise-free frame, fp64 and uint16"""
    import torch
    s = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    s.nx = 9215
    det = W.Detector(gain=1.0, dark_e=0.5, ron_e=3.0, bias=100.0, seed=31337)
    r = B.Renderer(s)
    try:
        pc = B.e2e_plan_check(r.fmt, r.psf)
        assert pc["n_host_bands"] >= 3
        host_tabs = [np.ascontiguousarray(sp.flux, dtype=np.float64) for sp in s.spectra]
        desc = B.spectra_array(s.spectra, [t.ctypes.data for t in host_tabs])
        ws = torch.empty(B.e2e_render_host_workspace_bytes(r.fmt, r.psf, desc), dtype=torch.uint8, device="cuda")
        clean = torch.empty((s.ny, s.nx), dtype=torch.float64).pin_memory()
        B.e2e_render_frame_host(r.fmt, r.psf, desc, clean.data_ptr(), ws)
        H = clean.numpy().copy()
        assert H.max() > 0
        noisy = torch.empty_like(clean)
        B.e2e_render_frame_host(r.fmt, r.psf, desc, noisy.data_ptr(), ws, det=det)
        assert np.array_equal(noisy.numpy(), oracle.detector(H, det))
        d_ex, keep = B.detector_ex_desc(det, e_per_adu=1.1, adu_max=65535.0)
        out16 = torch.zeros((s.ny, s.nx), dtype=torch.uint16).pin_memory()
        B.e2e_render_frame_host_ex(r.fmt, r.psf, desc, out16.data_ptr(), ws, d_ex, adu16=True)
        assert np.array_equal(out16.numpy(), oracle.detector_adu16(H, det, e_per_adu=1.1, adu_max=65535.0))
    finally:
        r.close()


def test_detector_ex_bit_exact(B):
    """full detector stage: PRNU / dark maps, full well, ADC -- every variant bit-exact vs the oracle"""
    import torch
    rng = np.random.default_rng(6)
    nx, ny = 419, 61
    n = nx * ny
    fr = np.concatenate([np.zeros(500), rng.uniform(0, 5, 4000), rng.uniform(5, 64, 4000), rng.uniform(64, 200, 4000),
                         rng.uniform(3e4, 9e4, n - 12500)])
    fr[3] = -7.0
    fr = fr.reshape(ny, nx)
    prnu = rng.normal(1.0, 0.02, (ny, nx))
    prnu[0, :7] = 0.0                                         # dead pixels
    dark = rng.uniform(0.0, 3.0, (ny, nx))
    dark[1, :5] = 500.0                                       # hot pixels
    det = W.Detector(gain=0.85, dark_e=0.4, ron_e=3.0, bias=200.0, seed=0x0BAD_CAFE_F00D_0001)
    d_in, d_pr, d_dk = (torch.from_numpy(a).cuda() for a in (fr, prnu, dark))
    d_out = torch.empty_like(d_in)
    variants = [dict(), dict(prnu=True), dict(dark=True), dict(prnu=True, dark=True, full_well_e=6.0e4),
                dict(prnu=True, dark=True, full_well_e=6.0e4, e_per_adu=1.3, adu_max=65535.0),
                dict(e_per_adu=0.7, adu_max=4095.0)]
    for v in variants:
        kw = {k: v[k] for k in ("full_well_e", "e_per_adu", "adu_max") if k in v}
        B.e2e_apply_detector_ex(d_in, d_out, nx, ny, det, d_prnu=d_pr if v.get("prnu") else None,
                                d_dark=d_dk if v.get("dark") else None, **kw)
        okw = {("full_well" if k == "full_well_e" else k): x for k, x in kw.items()}
        O = oracle.detector_ex(fr, det, prnu=prnu if v.get("prnu") else None, dark=dark if v.get("dark") else None, **okw)
        assert np.array_equal(d_out.cpu().numpy(), O), v
    # no maps / well / ADC = the basic stage; in place works
    B.e2e_apply_detector_ex(d_in, d_out, nx, ny, det)
    ref = torch.empty_like(d_in)
    B.e2e_apply_detector(d_in, ref, nx, ny, det)
    assert torch.equal(d_out, ref)
    B.e2e_apply_detector_ex(d_in, d_in, nx, ny, det, d_prnu=d_pr, d_dark=d_dk, full_well_e=6.0e4, e_per_adu=1.3)
    assert np.array_equal(d_in.cpu().numpy(), O if False else oracle.detector_ex(fr, det, prnu=prnu, dark=dark, full_well=6.0e4, e_per_adu=1.3))
    with pytest.raises(B.E2EError):
        B.e2e_apply_detector_ex(d_out, d_out, nx, ny, det, e_per_adu=-1.0)
    with pytest.raises(B.E2EError):
        B.e2e_apply_detector_ex(d_out, d_out, nx, ny, det, d_prnu=d_out)


def test_detector_crosstalk_and_adu16_bit_exact(B):
    """G20 cross-talk between read-out ports and the uint16 ADC output: every variant bit-exact vs the oracle,
    in place too; shapes that do not fit are refused"""
    import torch
    rng = np.random.default_rng(8)
    nx, ny = 16 * 37, 23                                      # 37 columns per port with 16 ports, 148 with 4
    fr = rng.uniform(0.0, 200.0, (ny, nx))
    fr[3, :40] = 0.0
    fr[4, :40] = rng.uniform(0.0, 3.0, 40)
    fr[:, 5] = 5.0e4                                          # a bright column: its ghost shows up in the other ports
    prnu = rng.normal(1.0, 0.02, (ny, nx))
    dark = rng.uniform(0.0, 3.0, (ny, nx))
    det = W.Detector(gain=0.9, dark_e=0.2, ron_e=2.5, bias=300.0, seed=0x5EED_0000_0000_0007)
    d_in, d_pr, d_dk = (torch.from_numpy(a).cuda() for a in (fr, prnu, dark))
    d_out = torch.empty_like(d_in)
    d_u16 = torch.empty((ny, nx), dtype=torch.uint16, device="cuda")
    for n_ports in (2, 4, 16):
        X = rng.uniform(-2e-4, 8e-4, (n_ports, n_ports))
        for kw in (dict(), dict(e_per_adu=1.1, adu_max=65535.0), dict(full_well_e=4.0e4, e_per_adu=0.8, adu_max=40000.0)):
            okw = {("full_well" if k == "full_well_e" else k): x for k, x in kw.items()}
            B.e2e_apply_detector_ex(d_in, d_out, nx, ny, det, d_prnu=d_pr, d_dark=d_dk, xtalk=X, **kw)
            O = oracle.detector_ex(fr, det, prnu=prnu, dark=dark, xtalk=X, **okw)
            assert np.array_equal(d_out.cpu().numpy(), O), (n_ports, kw)
            if kw:
                B.e2e_apply_detector_adu16(d_in, d_u16, nx, ny, det, d_prnu=d_pr, d_dark=d_dk, xtalk=X, **kw)
                G16 = d_u16.cpu().numpy()
                assert G16.dtype == np.uint16
                assert np.array_equal(G16, oracle.detector_adu16(fr, det, prnu=prnu, dark=dark, xtalk=X, **okw))
        # in place
        tmp = d_in.clone()
        B.e2e_apply_detector_ex(tmp, tmp, nx, ny, det, xtalk=X)
        assert np.array_equal(tmp.cpu().numpy(), oracle.detector_ex(fr, det, xtalk=X))
    # the ghost of the bright column is there: same in-port column of port 1, scaled by X[1][0]
    X = np.zeros((4, 4)); X[1, 0] = 1e-3
    B.e2e_apply_detector_ex(d_in, d_out, nx, ny, det, xtalk=X)
    plain = torch.empty_like(d_in)
    B.e2e_apply_detector_ex(d_in, plain, nx, ny, det)
    diff = (d_out - plain).cpu().numpy()
    assert np.all(np.abs(diff[:, 148 + 5] - 1e-3 * 0.9 * 5.0e4) < 3.0)
    assert np.abs(diff[:, :148]).max() < 1e-9            # port 0 receives nothing ((e + ron z1) + bias vs (e + bias) + ron z1: rounding only)
    # uint16 without cross-talk, and without maps
    B.e2e_apply_detector_adu16(d_in, d_u16, nx, ny, det, e_per_adu=1.3)
    assert np.array_equal(d_u16.cpu().numpy(), oracle.detector_adu16(fr, det, e_per_adu=1.3))
    with pytest.raises(B.E2EError):
        B.e2e_apply_detector_ex(d_in, d_out, nx, ny, det, xtalk=np.zeros((5, 5)))         # 592 % 5 != 0
    with pytest.raises(B.E2EError):
        B.e2e_apply_detector_ex(d_in, d_out, nx, ny, det, xtalk=np.zeros((32, 32)))
    with pytest.raises(B.E2EError):
        B.e2e_apply_detector_adu16(d_in, d_u16, nx, ny, det, e_per_adu=0.0)
    with pytest.raises(B.E2EError):
        B.e2e_apply_detector_adu16(d_in, d_u16, nx, ny, det, e_per_adu=1.0, adu_max=1.0e5)


def test_render_frames_batch_equals_single_renders(B):
    """batch render on fixed geometry.  The five Doppler-shifted frames of the RV sweep in one call are,
    frame by frame, the bits of five single renders, and every one of them matches the oracle's render of that velocity
    per pixel; the sparse-sampling scene takes the frame-after-frame route of the non-production kernels"""
    import torch
    for make in (lambda v: W.rv_sweep(v), lambda v: _sparse_rv(v)):
        scenes = [make(v) for v in (0.0, 0.01, 0.1, 1.0, 10.0)]
        r = B.Renderer(scenes[0])
        try:
            singles = []
            descs = []
            keep = []
            for sc in scenes:
                flux = [torch.from_numpy(np.ascontiguousarray(sp.flux, dtype=np.float64)).cuda() for sp in sc.spectra]
                keep.append(flux)
                d = B.spectra_array(sc.spectra, [t.data_ptr() for t in flux])
                descs.append(d)
                fr = torch.empty((sc.ny, sc.nx), dtype=torch.float64, device="cuda")
                B.e2e_render_frame(r.fmt, r.psf, d, fr, False, r.workspace)
                singles.append(fr.clone())
            nbytes = B.e2e_render_frames_workspace_bytes(r.fmt, r.psf, len(scenes))
            ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            frames = [torch.full((scenes[0].ny, scenes[0].nx), float("nan"), dtype=torch.float64, device="cuda") for _ in scenes]
            B.e2e_render_frames(r.fmt, r.psf, descs, frames, False, ws)
            torch.cuda.synchronize()
            for a, b in zip(frames, singles):
                assert torch.equal(a, b)
            for a, sc in zip(frames, scenes):                        # every frame of the batch against the oracle, per pixel
                O = oracle.render(sc)
                assert O.max() > 0
                assert_frame_parity(a.cpu().numpy(), O, f"batch frame {sc.name} v={sc.notes.get('v_mps')}")
            assert not torch.equal(frames[0], frames[4])            # the shift is there
            # accumulate = 1 adds on top
            B.e2e_render_frames(r.fmt, r.psf, descs, frames, True, ws)
            torch.cuda.synchronize()
            assert torch.allclose(frames[2], 2.0 * singles[2], rtol=1e-15, atol=0.0)
            with pytest.raises(B.E2EError):
                B.e2e_render_frames(r.fmt, r.psf, descs[:2], [frames[0], frames[0]], False, ws)
            with pytest.raises(B.E2EError):
                B.e2e_render_frames(r.fmt, r.psf, descs, frames, False, ws[:4096])
        finally:
            r.close()


def test_render_frames_batch_on_a_frame_that_fills_the_gpu(B):
    """the batch call on a multi-order, two-fiber frame (the single-warp flush kernel in its batch form, frames interleaved in
    one grid; the RV-sweep batches above take the wide kernel): three frames with different Doppler factors and illumination,
    each the bits of its single render, and windows of one of them against the oracle"""
    import torch
    base = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=list(range(0, 85, 4)))   # 44 strips, ~7500 work items
    scenes = []
    for dop, sc0, sc1 in ((1.0, 1.0, 1.0), (1.0 + 2e-4, 0.5, 2.0), (1.0 - 1e-4, 3.0, 0.0)):
        sc = copy.copy(base)
        sc.spectra = [Spectrum_like(base.spectra[0], doppler=dop, scale=base.spectra[0].scale * sc0),
                      Spectrum_like(base.spectra[1], doppler=dop, scale=base.spectra[1].scale * sc1)]
        scenes.append(sc)
    r = B.Renderer(base)
    try:
        name = B.e2e_render_kernel_info(r.fmt, r.psf)["name"]
        assert name.startswith("cell_flush_kernel<")                # not the wide (small-frame) kernel
        keep, descs, singles = [], [], []
        for sc in scenes:
            flux = [torch.from_numpy(np.ascontiguousarray(sp.flux, dtype=np.float64)).cuda() for sp in sc.spectra]
            keep.append(flux)
            d = B.spectra_array(sc.spectra, [t.data_ptr() for t in flux])
            descs.append(d)
            fr = torch.empty((sc.ny, sc.nx), dtype=torch.float64, device="cuda")
            B.e2e_render_frame(r.fmt, r.psf, d, fr, False, r.workspace)
            singles.append(fr)
        ws = torch.empty(B.e2e_render_frames_workspace_bytes(r.fmt, r.psf, len(scenes)), dtype=torch.uint8, device="cuda")
        ws.view(torch.float64).fill_(float("nan"))
        frames = [torch.full((base.ny, base.nx), float("nan"), dtype=torch.float64, device="cuda") for _ in scenes]
        B.e2e_render_frames(r.fmt, r.psf, descs, frames, False, ws)
        torch.cuda.synchronize()
        for a, b in zip(frames, singles):
            assert torch.equal(a, b)
        assert not torch.equal(frames[0], frames[1])
        G = frames[1].cpu().numpy()
        for o, frac in ((0, 0.3), (11, 0.7)):
            n = oracle.order_nsamples(scenes[1], o)
            k = int(frac * (n - 1))
            lam, x, y, w = oracle.samples(scenes[1], 0, o, k, k + 1)
            i0, j0 = max(0, int(x[0]) - 24), max(0, int(y[0]) - 20)
            O = oracle.render(scenes[1], window=(i0, j0, 48, 40))
            assert O.max() > 0
            assert_frame_parity(G[j0:j0 + 40, i0:i0 + 48], O, f"batch frame 1 window {i0},{j0}")
    finally:
        r.close()


def _sparse_rv(v):
    s = W.rv_sweep(v)
    s.samples_per_px = 3.0
    s.lam_max = np.array([s.lam_min[0] + 4.0])
    return s


def test_rv_sweep_photocenter_linear_in_velocity(B):
    """BASELINE.json configs[4]: 5 Doppler-shifted frames.  DESIGN.md G14 (the CPU-only pin of the same three checks is
    tests/test_oracle_render.py::test_g14_rv_sweep_photocenter_linear_in_velocity): (i) global photocenter == flux-weighted
    mean of the oracle's mapped samples at every velocity; (ii) residual against a least-squares line in v < 1e-6 px,
    globally and per line; (iii) shift == closed-form slope of the line list INCLUDING the blaze-slope term to 1e-7 px.
    GPU == oracle per pixel on the v = 10 m/s frame; detector stage bit-exact on the rendered frame"""
    import torch
    frames, xc = [], []
    for v in W.RV_SWEEP_V:
        s = W.rv_sweep(v)
        G = gpu_render(B, s)
        frames.append(G)
        xc.append(photocenter_x(G))
    s10 = W.rv_sweep(10.0)
    O = oracle.render(s10)
    assert_frame_parity(frames[-1], O, "rv 10 m/s")
    assert abs(photocenter_x(frames[-1]) - photocenter_x(O)) < 1e-9
    v = np.array(W.RV_SWEEP_V)
    # P5: the frame's global photocenter is the flux-weighted mean of the mapped sample positions, at every velocity
    xs = []
    for vv in W.RV_SWEEP_V:
        lam, x, y, w = oracle.samples(W.rv_sweep(vv), 0, 0)
        xs.append(float(np.sum(w * x) / np.sum(w)))
    assert np.max(np.abs(np.array(xc) - np.array(xs))) < 1e-9
    # and it moves linearly with velocity (least-squares line through the 5 velocities, G14), by ~3.5e-3 px at 10 m/s
    A = np.vstack([v, np.ones_like(v)]).T
    coef, *_ = np.linalg.lstsq(A, np.array(xc), rcond=None)
    assert np.max(np.abs(np.array(xc) - A @ coef)) < 1e-6
    assert 1e-3 < xc[-1] - xc[0] < 1e-2
    # (iii) closed-form slope (G14): d xbar / d beta = [sum W lam X' + sum E' lam (X - xbar)] / sum W over the 200 lines
    cen = W.rv_sweep(0.0).notes["line_centers"]
    Xf = lambda l: 1024 + 1000 * ((l - 5025) / 25) + ((l - 5025) / 25) ** 2
    Xp = lambda l: (1000 + 2 * ((l - 5025) / 25)) / 25

    def E(l):
        a = np.pi * 100 * (5025.0 / l - 1)
        return np.where(np.abs(a) < 1e-12, 1.0, (np.sin(a) / np.where(a == 0, 1.0, a)) ** 2)
    Wl, h = E(cen), 1e-4
    Ep = (E(cen + h) - E(cen - h)) / (2 * h)
    xbar = (Wl * Xf(cen)).sum() / Wl.sum()
    slope = ((Wl * cen * Xp(cen)).sum() + (Ep * cen * (Xf(cen) - xbar)).sum()) / Wl.sum()
    assert np.max(np.abs((np.array(xc) - xc[0]) - slope * v / W.C_LIGHT)) < 1e-7
    # per-line windows (Voronoi cells of integer columns between line positions)
    cen = W.rv_sweep(0.0).notes["line_centers"]
    xl = 1024 + 1000 * (cen - 5025) / 25 + ((cen - 5025) / 25) ** 2
    edges = np.round(0.5 * (xl[1:] + xl[:-1])).astype(int)
    worst = 0.0
    for ell in (3, 50, 100, 150, 196):
        c0, c1 = edges[ell - 1], edges[ell]
        pcs = np.array([photocenter_x(f[:, c0:c1], c0) for f in frames])
        A = np.vstack([v, np.ones_like(v)]).T
        coef, *_ = np.linalg.lstsq(A, pcs, rcond=None)
        worst = max(worst, float(np.max(np.abs(pcs - A @ coef))))
    assert worst < 1e-6
    det = s10.detector
    d_in = torch.from_numpy(frames[-1]).cuda()
    d_out = torch.empty_like(d_in)
    B.e2e_apply_detector(d_in, d_out, s10.nx, s10.ny, det)
    assert np.array_equal(d_out.cpu().numpy(), oracle.detector(frames[-1], det))
    assert 3e4 < frames[-1].max() < 6e4


# ------------------------------------------------------------------------------------------ schedule invariants
def _assert_plan_ok(B, scene, label):
    r = B.Renderer(scene)
    try:
        c = B.e2e_plan_check(r.fmt, r.psf)
    finally:
        r.close()
    assert c["claimed_px"] > 0 and c["n_items"] > 0, (label, c)
    for k in ("phase_conflicts", "queue_conflicts", "device_band_conflicts", "host_band_conflicts", "host_rows_not_final"):
        assert c[k] == 0, (label, k, c)
    return c


def test_schedule_invariants_small_scenes(B):
    """the frame is accumulated with L2 reductions, so its bits rest on the host schedule: no two items of a
    phase launch share a pixel, every pair of items that shares a pixel is ordered by a dependency edge of the persistent
    launch, row bands share no pixel.  e2e_plan_check stamps every footprint box into an owner frame on the device and
    counts violations: steep multi-fiber traces, overlapping orders, a reversed trace, sparse sampling, a tabulated PSF"""
    s = small_tiny(spp=8.0, lam=(5005.0, 5045.0))
    s.coef_y = np.array([128.0, 600.0, 0.0, 0.0])                    # steep: dy/dx = 0.6
    s.fiber_dx = np.array([0.0, 0.3, -0.2, 0.1]); s.fiber_dy = np.array([-7.0, -2.0, 3.0, 9.0])
    s.spectra = [s.spectra[0]] * 4
    c = _assert_plan_ok(B, s, "steep 4-fiber")
    assert c["n_dependencies"] > 0
    s = small_tiny(spp=40.0, lam=(5000.0, 5050.0))
    s.coef_x = np.array([1024.0, -1000.0, 1.0, 0.0])                 # x decreasing with lambda
    _assert_plan_ok(B, s, "reversed")
    _assert_plan_ok(B, small_tiny(spp=0.4, lam=(5005.0, 5045.0)), "sparse")
    _assert_plan_ok(B, W.tiny(), "tiny")
    _assert_plan_ok(B, small_field_scene(gx=3, gy=2), "tabulated")
    s = W.espresso_like(n_obj_lines=100, table_dlam=0.02).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    c = _assert_plan_ok(B, s, "espresso 7 orders")
    assert c["n_host_bands"] >= 2


@pytest.mark.parametrize("which", ["espresso_like", "hires_like", "field_psf"])
def test_schedule_invariants_full_size(B, which):
    """the same at BASELINE.json's full sizes (the plans bench.py's launches use), plus three renders that must agree bit for
    bit (the espresso_gpu fixture does that for espresso_like)"""
    if which == "espresso_like":
        s = W.espresso_like(n_obj_lines=100, table_dlam=0.02)
    elif which == "hires_like":
        s = W.hires_like(n_lines=200, table_dlam=0.02)
    else:
        s = W.field_psf(base=W.espresso_like(n_obj_lines=100, table_dlam=0.02))
    c = _assert_plan_ok(B, s, which)
    assert c["n_dependencies"] > c["n_items"] // 2
    if which != "espresso_like":
        r = B.Renderer(s)
        try:
            a = r.render().clone()
            for _ in range(2):
                assert r.torch.equal(r.render(), a)
        finally:
            r.close()


# ------------------------------------------------------------------------------------------ parametric spectrograph unit
def test_render_from_the_parametric_spectrograph_unit(B):
    """S8(f) 4: a frame rendered from a spectral format that e2e_spectrograph_format generated from geometrical
    parameters (R2 echelle, three orders, a tilted 3-fiber pseudo-slit).  The mapped sample positions follow the oracle's
    closed-form grating relations within the residual the generator reports, and the frame matches the oracle per pixel"""
    from oracle import spectrograph as OS
    kw = dict(groove_um=1000.0 / 52.6, blaze_deg=63.4, theta_deg=0.7, gamma_deg=0.9, xd_groove_um=1000.0 / 300.0, xd_lam_ref=5500.0,
              f_cam_mm=300.0, f_coll_mm=1200.0, pixel_um=15.0, fiber_core_um=200.0, m_lo=60, m_hi=62, x_c=1024.0, y_c=300.0,
              fiber_height_um=(-400.0, 0.0, 400.0))
    g = B.e2e_spectrograph_format(**kw)
    assert g["residual_x_px"] < 1e-4 and g["residual_y_px"] < 1e-4
    assert 0 < g["x_min"] and g["x_max"] < 2048 and 0 < g["y_min"] and g["y_max"] < 600
    rng = np.random.default_rng(61)
    lam_lo, lam_hi = float(g["lam_min"].min()) - 1.0, float(g["lam_max"].max()) + 1.0
    flux = 1.0 + 0.5 * rng.random(int((lam_hi - lam_lo) / 0.02) + 2)
    spectra = [W.Spectrum(flux=flux, lam0=lam_lo, dlam=0.02, scale=sc) for sc in (800.0, 1000.0, 700.0)]
    s = W.Scene(name="parametric_r2", nx=2048, ny=600, order_m=g["order_m"].copy(), lam_min=g["lam_min"].copy(), lam_max=g["lam_max"].copy(),
                fiber_dx=g["fiber_dx"].copy(), fiber_dy=g["fiber_dy"].copy(), deg_l=5, deg_m=5, coef_x=g["coef_x"].copy(),
                coef_y=g["coef_y"].copy(), lam0=g["lam0"], inv_dlam=g["inv_dlam"], m0=g["m0"], inv_dm=g["inv_dm"],
                blaze_lam_c=g["blaze_lam_c"].copy(), blaze_amp=g["blaze_amp"].copy(), samples_per_px=8.0,
                psf=W.Psf(kind=0, fiber_dx_px=g["fiber_dx_px"], fiber_dy_px=g["fiber_dy_px"], sigma_x=1.1, sigma_y=1.1), spectra=spectra)
    p = OS.Spectrograph(**kw)
    r = B.Renderer(s)
    try:
        for o in range(3):
            lam, x, y, w = r.samples(1, o)                                # the middle fiber sits on the base trace
            assert np.abs(x - OS.position_x(p, lam, int(g["order_m"][o]))).max() < 1.02 * g["residual_x_px"] + 1e-8
            assert np.abs(y - OS.position_y(p, lam)).max() < 1.02 * g["residual_y_px"] + 1e-8
            assert np.array_equal(x, oracle.samples(s, 1, o)[1])
        G = r.render().cpu().numpy()
    finally:
        r.close()
    O = oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, "parametric spectrograph unit")
    assert abs(G.sum() / oracle.total_weight(s) - 1.0) < 1e-12


# ------------------------------------------------------------------------------------------ degenerate inputs
def test_degenerate_inputs_and_limits(B):
    """edge cases of the boundary (include/e2e.h): orders wholly off the detector, an order of a single sample, 64 fibers (the
    limit) and 65 (refused), PSFs beyond the footprint / chord-order limits (refused), NaN parameters (refused), a misaligned
    workspace (refused), zero frames in a batch (refused) -- and the frames that ARE rendered match the oracle"""
    import torch
    # (1) one order on the detector, one wholly below it, one reduced to a single sample
    s = small_tiny(spp=4.0, lam=(5010.0, 5012.0))
    s.order_m = np.array([100, 101, 102], dtype=np.int32)
    s.lam_min = np.array([5010.0, 5010.0, 5011.0]); s.lam_max = np.array([5012.0, 5012.0, 5011.0 + 1e-5])
    s.blaze_lam_c = np.array([5025.0, 5025.0, 5025.0]); s.blaze_amp = np.ones(3)
    s.deg_m = 1
    s.coef_x = np.array([1024.0, 0.0, 1000.0, 0.0, 1.0, 0.0, 0.0, 0.0])
    s.coef_y = np.array([100.0, 900.0, 10.0, 0.0, 0.0, 0.0, 0.0, 0.0])        # m = 101 lands on row 1000 of a 256-row detector
    s.m0, s.inv_dm = 100.0, 1.0
    assert oracle.order_nsamples(s, 2) == 1
    G, O = gpu_render(B, s), oracle.render(s)
    assert O.max() > 0
    assert_frame_parity(G, O, "off-detector order + single-sample order")
    # (2) 64 fibers render, 65 are refused
    s = small_tiny(spp=2.0, lam=(5010.0, 5010.5))
    s.fiber_dx = np.linspace(-1.0, 1.0, 64); s.fiber_dy = np.linspace(-100.0, 100.0, 64)
    s.spectra = [s.spectra[0]] * 64
    assert_frame_parity(gpu_render(B, s), oracle.render(s), "64 fibers")
    s.fiber_dx = np.zeros(65); s.fiber_dy = np.zeros(65); s.spectra = [s.spectra[0]] * 65
    with pytest.raises(B.E2EError) as ei:
        B.Format(s)
    assert ei.value.code == -5
    # (3) PSF limits and bad parameters
    base = small_tiny(spp=2.0)
    for kw, code in ((dict(fiber_dx_px=3.0, fiber_dy_px=3.0, sigma_x=7.0, sigma_y=1.0), -5),          # footprint > 96 px
                     (dict(fiber_dx_px=3.0, fiber_dy_px=3.0, sigma_x=1.0, sigma_y=1.0, n_nodes=65), -5),
                     (dict(fiber_dx_px=3.0, fiber_dy_px=3.0, sigma_x=float("nan"), sigma_y=1.0), -1),
                     (dict(fiber_dx_px=-1.0, fiber_dy_px=3.0, sigma_x=1.0, sigma_y=1.0), -1),
                     (dict(fiber_dx_px=3.0, fiber_dy_px=3.0, sigma_x=0.0, sigma_y=1.0), -1)):
        with pytest.raises(B.E2EError) as ei:
            B.Psf(with_psf(base, **kw).psf, base.nx, base.ny)
        assert ei.value.code == code, kw
    bad = copy.copy(base); bad.coef_x = base.coef_x.copy(); bad.coef_x[1] = np.inf
    with pytest.raises(B.E2EError):
        B.Format(bad)
    # (4) workspace misaligned / batch of zero frames / spectrum descriptor with a non-positive step
    r = B.Renderer(base)
    try:
        fr = torch.empty((base.ny, base.nx), dtype=torch.float64, device="cuda")
        with pytest.raises(B.E2EError) as ei:
            B.e2e_render_frame(r.fmt, r.psf, r.spectra, fr, False, r.workspace[8:])
        assert ei.value.code == -6
        with pytest.raises(B.E2EError):
            B.e2e_render_frames_workspace_bytes(r.fmt, r.psf, 0)
        d = B.spectra_array(base.spectra, [t.data_ptr() for t in r.flux])
        d[0].dlam = 0.0
        with pytest.raises(B.E2EError) as ei:
            B.e2e_render_frame(r.fmt, r.psf, d, fr, False, r.workspace)
        assert ei.value.code == -1
        # the handle still renders after the refused calls
        assert_frame_parity(r.render().cpu().numpy(), oracle.render(base), "after refused calls")
    finally:
        r.close()
