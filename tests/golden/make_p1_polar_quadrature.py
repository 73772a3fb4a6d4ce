"""Pin P1: brute-force 2-D polar quadrature, in 30-digit mpmath arithmetic, of the DEFINITION of
the pixel-integrated instrument PSF ("surface integral of the convolution between the spatial
profile of the fiber and the PSF"):

    P(u, v) = 1/(pi a b)  integral over the ellipse (s/a)^2 + (t/b)^2 <= 1 of  Gx(u - s) Gy(v - t) ds dt
    G(d)    = Phi((d + 1/2)/sigma) - Phi((d - 1/2)/sigma)        (gaussian integrated over a unit pixel)

with s = a r cos(th), t = b r sin(th).  No chord trick, no oracle code: this script imports only mpmath.
Writes tests/golden/p1_polar_quadrature.txt.   Usage: python tests/golden/make_p1_polar_quadrature.py
"""
from pathlib import Path
import mpmath as mp

mp.mp.dps = 30


def Phi(z):
    return mp.erfc(-z / mp.sqrt(2)) / 2


def G(d, sigma):
    return Phi((d + mp.mpf(1) / 2) / sigma) - Phi((d - mp.mpf(1) / 2) / sigma)


def P(u, v, Dx, Dy, sx, sy):
    a, b = mp.mpf(Dx) / 2, mp.mpf(Dy) / 2
    f = lambda r, th: G(u - a * r * mp.cos(th), sx) * G(v - b * r * mp.sin(th), sy) * r
    val = mp.quad(f, [0, mp.mpf(1) / 2, 1], [0, mp.pi / 2, mp.pi, 3 * mp.pi / 2, 2 * mp.pi])
    return val / mp.pi


CASES = [
    # Dx, Dy, sx, sy, xk, yk, list of pixels (i, j)
    (3.0, 3.0, 1.0, 1.0, "10.3173", "7.8641", [(10, 8), (12, 6), (15, 8), (10, 1)]),
    (4.0, 4.0, 1.2, 1.2, "10.3173", "7.8641", [(10, 8), (12, 6), (15, 8), (3, 8)]),
    (5.0, 2.0, 0.9, 1.4, "20.75", "15.125", [(20, 15), (23, 15), (20, 18), (17, 13)]),   # asymmetric: catches x/y swaps
]

if __name__ == "__main__":
    out = ["# Dx Dy sigma_x sigma_y x_k y_k i j P   (mpmath %s, dps=%d, 2-D polar quadrature of the definition)" % (mp.__version__, mp.mp.dps)]
    for Dx, Dy, sx, sy, xk, yk, pix in CASES:
        for (i, j) in pix:
            u = mp.mpf(i) - mp.mpf(xk)
            v = mp.mpf(j) - mp.mpf(yk)
            val = P(u, v, Dx, Dy, mp.mpf(sx), mp.mpf(sy))
            out.append("%r %r %r %r %s %s %d %d %s" % (Dx, Dy, sx, sy, xk, yk, i, j, mp.nstr(val, 22)))
            print(out[-1], flush=True)
    Path(__file__).with_name("p1_polar_quadrature.txt").write_text("\n".join(out) + "\n")
