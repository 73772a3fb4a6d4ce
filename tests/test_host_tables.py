"""Host logic of the CUDA path without a GPU: the pixel-phase polynomial tables (csrc/poly_tables.h, built by e2e_psf_create)
against closed forms -- NOT against the oracle: scipy's erf for the pure gaussian (pin P2's closed form), and, for the disk (x)
gaussian, the sum over chord terms against the mpmath polar quadrature fixture of pin P1."""
import ctypes as C
import subprocess
from pathlib import Path

import numpy as np
import pytest
from scipy.special import erf

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def shim(tmp_path_factory):
    out = tmp_path_factory.mktemp("shim") / "libtables_shim.so"
    subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-ffp-contract=off", str(ROOT / "tests/host/tables_shim.cpp"),
                    "-o", str(out)], check=True)
    L = C.CDLL(str(out))
    L.shim_build.restype = C.c_int
    L.shim_build.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int] + [C.POINTER(C.c_int)] * 6 + [C.POINTER(C.c_double)] * 3 + [C.POINTER(C.c_void_p)]
    for f in (L.shim_eval_x, L.shim_eval_y):
        f.restype = C.c_double
        f.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
    L.shim_eval_y_window.restype = C.c_double
    L.shim_eval_y_window.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double]
    L.shim_free.argtypes = [C.c_void_p]
    return L


def build(L, D, sigma, t=7.5, Q=12):
    ints = [C.c_int() for _ in range(6)]
    dbl = [C.c_double() for _ in range(3)]
    h = C.c_void_p()
    rc = L.shim_build(D, sigma, t, Q, *[C.byref(i) for i in ints], *[C.byref(d) for d in dbl], C.byref(h))
    assert rc == 0
    keys = ("P", "npt", "ncol", "nrow", "nyb", "T")
    info = {k: v.value for k, v in zip(keys, ints)}
    info.update(c0x=dbl[0].value, c0y=dbl[1].value, trunc_err=dbl[2].value, h=h)
    return info


def gauss_pix(u, sigma):
    """pixel-integrated unit gaussian at offset u (pixel centre - sample position): closed form"""
    return 0.5 * (erf((u + 0.5) / (sigma * np.sqrt(2.0))) - erf((u - 0.5) / (sigma * np.sqrt(2.0))))


@pytest.mark.parametrize("sigma", [0.8, 1.0, 1.2, 2.0])
def test_pure_gaussian_tables_match_the_erf_closed_form(shim, sigma):
    T = build(shim, 0.0, sigma)
    assert T["T"] == 1 and T["trunc_err"] <= 1e-17 and T["nyb"] in (16, 32, 64, 128, 256)
    rng = np.random.default_rng(5)
    worst = 0.0
    for _ in range(300):
        d = rng.uniform(-0.5, 0.5)
        i = int(rng.integers(0, T["ncol"]))
        want = gauss_pix((i - T["c0x"]) - d, sigma)            # column i sits at (i - c0x) - d from the sample
        worst = max(worst, abs(shim.shim_eval_x(T["h"], 0, i, d) - want), abs(shim.shim_eval_y(T["h"], 0, i, d) - want))
    assert worst < 2e-16                                        # fp64 Horner rounding on values <= ~0.4
    shim.shim_free(T["h"])


def test_y_window_is_accurate_over_its_whole_validity(shim):
    """a cell keeps its window while |delta| <= 1/nyb: the fit must hold there, not only inside +-1/(2 nyb)"""
    sigma = 1.2
    T = build(shim, 0.0, sigma)
    nyb = T["nyb"]
    worst = 0.0
    for b in (0, nyb // 3, nyb - 1):
        yc = (b + 0.5) / nyb - 0.5
        for dl in np.linspace(-1.0 / nyb, 1.0 / nyb, 9):
            for j in (0, 5, 11, 12, T["nrow"] - 1):
                want = gauss_pix((j - T["c0y"]) - (yc + dl), sigma)
                worst = max(worst, abs(shim.shim_eval_y_window(T["h"], 0, j, b, float(dl)) - want))
    assert worst < 2e-16
    shim.shim_free(T["h"])


def test_disk_gaussian_tables_sum_to_the_polar_quadrature_fixture(shim):
    """sum_t FX_t(i, dx) GY_t(j, dy) against pin P1's values (tests/golden/p1_polar_quadrature.txt: 40-digit 2-D polar
    quadrature of the disk-averaged pixel-integrated gaussian, x_k = 10.3173, y_k = 7.8641)"""
    rows = []
    for line in (ROOT / "tests/golden/p1_polar_quadrature.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            rows.append(line.split())
    assert rows
    checked = 0
    for r in rows:
        Dx, Dy, sx, sy, xk, yk = (float(v) for v in r[:6])
        i, j, val = int(r[6]), int(r[7]), float(r[8])
        if Dx != Dy or sx != sy:
            continue                                            # the shim builds circular PSFs
        T = build(shim, Dx, sx)
        hb = 0.5 * Dx + 7.5 * sx + 0.5
        ilo, jlo = int(np.ceil(xk - hb)), int(np.ceil(yk - hb))
        dx, dy = (xk - ilo) - T["c0x"], (yk - jlo) - T["c0y"]
        got = sum(shim.shim_eval_x(T["h"], t, i - ilo, dx) * shim.shim_eval_y(T["h"], t, j - jlo, dy) for t in range(T["T"]))
        assert got == pytest.approx(val, rel=2e-11, abs=2e-14)      # chord quadrature Q = 12: converged to ~1e-12 of the peak
        checked += 1
        shim.shim_free(T["h"])
    assert checked >= 4
