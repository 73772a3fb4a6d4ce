// spectrograph.cu -- the parametric Spectrograph Unit (host code only; no kernel, no device call).
//
// "the Parametric Version works without the need of the optical design files and requires only geometrical
// parameters (such as dispersing elements working angle, optical elements working F-Number) to recover the expected spectral
// format required for rendering the image"; "analytical calculation of the echelle grating blaze profile for each
// order"; "orders curvature, lines tilt", "tilted pseudoslit projection".  The paper gives no equations; the model
// is reading G22 of DESIGN.md -- the textbook relations of a cross-dispersed echelle spectrograph:
//
//   echelle        m lam = d cos(gamma) (sin alpha + sin beta),      alpha = theta_B + theta,  beta_c = theta_B - theta (blaze peak)
//                  K = d cos(gamma) (sin alpha + sin beta_c) = 2 d cos(gamma) sin(theta_B) cos(theta)      ->  lam_c(m) = K / m
//                  one free spectral range per order: lam in [K / (m + 1/2), K / (m - 1/2)]
//   camera         x = x_c + F tan(beta - beta_c),   F = f_cam / pixel                       (main dispersion)
//   cross-disperser (first-order grating, Littrow at lam_ref):  sin beta_x = lam / d_x - sin alpha_x,  sin alpha_x = lam_ref / (2 d_x)
//                  y = y_c + F tan(beta_x(lam) - alpha_x)                                     (cross dispersion)
//   fiber image    Dy = core f_cam / (f_coll pixel),  Dx = Dy cos(alpha) / cos(beta_c)        (anamorphic magnification)
//   pseudo-slit    fiber f at height h_f along the slit: dy_f = h_f f_cam / (f_coll pixel); line tilt from the off-plane angle,
//                  tan(chi) = tan(gamma) (sin alpha + sin beta_c) / cos(beta_c)  ->  dx_f = tan(chi) dy_f
//   blaze peak     amp = min(1, cos(alpha) / cos(beta_c))  (groove shadowing for alpha > beta; "shadowing")
//
// The render path takes the spectral format as tensor polynomials of degree (5, 5) in the normalised (L, M) (e2e.h).  x depends
// on (lam, m) only through t = m lam / K - 1, |t| <= 1 / (2 m_lo - 1), which is bilinear in (L, M): g(t) is replaced by its
// degree-5 Chebyshev interpolant on that range and expanded exactly into the tensor basis.  y depends on lam only: degree-5
// Chebyshev interpolant in L.  Both residuals against the closed forms are measured on a dense grid and returned.
#include "common.cuh"

#include <cmath>
#include <vector>

namespace {

constexpr long double kPi = 3.14159265358979323846264338327950288L;

// monomial coefficients (in u, |u| <= 1) of the degree-P Chebyshev interpolant of f on [-1, 1]
template <class F>
void cheb_mono(F f, int P, long double* mono)
{
    const int N = P + 1;
    std::vector<long double> fv(N), c(N);
    for (int j = 0; j < N; ++j) fv[j] = f(cosl(kPi * ((long double)j + 0.5L) / (long double)N));
    for (int i = 0; i < N; ++i) {
        long double acc = 0.0L;
        for (int j = 0; j < N; ++j) acc += fv[j] * cosl(kPi * (long double)i * ((long double)j + 0.5L) / (long double)N);
        c[i] = acc * 2.0L / (long double)N;
    }
    c[0] *= 0.5L;
    std::vector<long double> t0(N, 0.0L), t1(N, 0.0L), t2(N, 0.0L);
    for (int k = 0; k < N; ++k) mono[k] = 0.0L;
    t0[0] = 1.0L;
    mono[0] += c[0];
    if (N > 1) { t1[1] = 1.0L; mono[1] += c[1]; }
    for (int i = 2; i < N; ++i) {
        for (int k = 0; k < N; ++k) t2[k] = (k > 0 ? 2.0L * t1[k - 1] : 0.0L) - t0[k];
        for (int k = 0; k < N; ++k) mono[k] += c[i] * t2[k];
        t0.swap(t1);
        t1.swap(t2);
    }
}

}  // namespace

extern "C" int e2e_spectrograph_format(const e2e_spectrograph_t* sp, e2e_spectrograph_format_t* out)
{
    using namespace e2e;
    if (!sp || !out) return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: NULL argument");
    if (!out->order_m || !out->lam_min || !out->lam_max || !out->blaze_lam_c || !out->blaze_amp || !out->coef_x || !out->coef_y)
        return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: NULL output array");
    if (sp->n_fibers > 0 && (!sp->fiber_height_um || !out->fiber_dx || !out->fiber_dy))
        return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: NULL fiber array");
    const double vals[] = {sp->groove_um, sp->blaze_deg, sp->theta_deg, sp->gamma_deg, sp->xd_groove_um, sp->xd_lam_ref, sp->f_cam_mm,
                           sp->f_coll_mm, sp->pixel_um, sp->fiber_core_um, sp->x_c, sp->y_c};
    for (double v : vals)
        if (!std::isfinite(v)) return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: non-finite parameter");
    if (!(sp->groove_um > 0.0) || !(sp->xd_groove_um > 0.0) || !(sp->xd_lam_ref > 0.0) || !(sp->f_cam_mm > 0.0) || !(sp->f_coll_mm > 0.0) ||
        !(sp->pixel_um > 0.0) || !(sp->fiber_core_um >= 0.0))
        return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: lengths must be > 0");
    if (sp->m_lo < 2 || sp->m_hi < sp->m_lo || sp->m_hi - sp->m_lo + 1 > 4096) return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: need 2 <= m_lo <= m_hi");
    if (out->capacity_orders < sp->m_hi - sp->m_lo + 1) return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: order arrays too short");
    const long double rad = kPi / 180.0L;
    const long double thB = sp->blaze_deg * rad, th = sp->theta_deg * rad, gam = sp->gamma_deg * rad;
    if (!(thB > 0.0L && thB < 0.5L * kPi) || !(fabsl(th) < 0.25L * kPi) || !(fabsl(gam) < 0.25L * kPi))
        return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: angles out of range");
    const long double alpha = thB + th, beta_c = thB - th;
    if (!(alpha < 0.5L * kPi) || !(beta_c > 0.0L)) return fail(E2E_ERR_INVALID_ARG, "spectrograph_format: |theta| too large for this blaze angle");
    const long double d = (long double)sp->groove_um * 1.0e4L;            // Angstrom
    const long double s0 = sinl(alpha) + sinl(beta_c);                   // = 2 sin(theta_B) cos(theta)
    const long double K = d * cosl(gam) * s0;                            // m lam at the blaze peak
    const long double F = (long double)sp->f_cam_mm * 1.0e3L / (long double)sp->pixel_um;   // pixels per radian (tangent plane)
    const int no = sp->m_hi - sp->m_lo + 1;
    // ---- orders, ranges, blaze
    long double lam_lo = 1.0e300L, lam_hi = 0.0L;
    const long double amp = fminl(1.0L, cosl(alpha) / cosl(beta_c));
    for (int o = 0; o < no; ++o) {
        const int m = sp->m_lo + o;
        out->order_m[o] = m;
        out->blaze_lam_c[o] = (double)(K / (long double)m);
        out->blaze_amp[o] = (double)amp;
        out->lam_min[o] = (double)(K / ((long double)m + 0.5L));
        out->lam_max[o] = (double)(K / ((long double)m - 0.5L));
        lam_lo = fminl(lam_lo, (long double)out->lam_min[o]);
        lam_hi = fmaxl(lam_hi, (long double)out->lam_max[o]);
    }
    out->n_orders = no;
    out->deg_l = 5; out->deg_m = 5;
    const long double lam0 = 0.5L * (lam_lo + lam_hi), inv_dlam = 2.0L / (lam_hi - lam_lo);
    const long double m0 = 0.5L * (long double)(sp->m_lo + sp->m_hi), inv_dm = no > 1 ? 2.0L / (long double)(sp->m_hi - sp->m_lo) : 1.0L;
    out->lam0 = (double)lam0; out->inv_dlam = (double)inv_dlam; out->m0 = (double)m0; out->inv_dm = (double)inv_dm;
    // the doubles the render path will really use (L and M are computed from these)
    const long double lam0d = out->lam0, idl = out->inv_dlam, m0d = out->m0, idm = out->inv_dm;
    // ---- x: g(t) = x_c + F tan(beta(t) - beta_c), sin beta = (1 + t) s0 - sin alpha, on |t| <= tmax (2 % margin)
    const long double tmax = 1.02L / (2.0L * (long double)sp->m_lo - 1.0L);
    if (!((1.0L + tmax) * s0 - sinl(alpha) < 0.999L)) return fail(E2E_ERR_UNSUPPORTED, "spectrograph_format: diffraction angle reaches 90 degrees");
    auto g_exact = [&](long double t) { return (long double)sp->x_c + F * tanl(asinl((1.0L + t) * s0 - sinl(alpha)) - beta_c); };
    long double a[6];
    cheb_mono([&](long double u) { return g_exact(u * tmax); }, 5, a);
    { long double sc = 1.0L; for (int j = 0; j < 6; ++j) { a[j] *= sc; sc /= tmax; } }       // monomials in t
    // t = m lam / K - 1 with lam = lam0 + L / inv_dlam, m = m0 + M / inv_dm: bilinear in (L, M); T[p][q] multiplies L^p M^q
    long double T[2][2] = {{m0d * lam0d / K - 1.0L, lam0d / (K * idm)}, {m0d / (K * idl), 1.0L / (K * idl * idm)}};
    long double cx[6][6] = {}, pw[6][6] = {}, nxt[6][6];
    pw[0][0] = 1.0L;                                                     // t^0
    for (int j = 0; j < 6; ++j) {
        for (int p = 0; p < 6; ++p)
            for (int q = 0; q < 6; ++q) cx[p][q] += a[j] * pw[p][q];
        for (int p = 0; p < 6; ++p)
            for (int q = 0; q < 6; ++q) nxt[p][q] = 0.0L;
        for (int p = 0; p < 6; ++p)
            for (int q = 0; q < 6; ++q)
                if (pw[p][q] != 0.0L)
                    for (int dp = 0; dp < 2; ++dp)
                        for (int dq = 0; dq < 2; ++dq)
                            if (p + dp < 6 && q + dq < 6) nxt[p + dp][q + dq] += pw[p][q] * T[dp][dq];
        for (int p = 0; p < 6; ++p)
            for (int q = 0; q < 6; ++q) pw[p][q] = nxt[p][q];
    }
    // ---- y: h(lam) = y_c + F tan(beta_x(lam) - alpha_x), degree-5 Chebyshev interpolant in L on [-1, 1]
    const long double dx_ = (long double)sp->xd_groove_um * 1.0e4L;
    const long double sax = (long double)sp->xd_lam_ref / (2.0L * dx_);
    if (!(sax < 0.999L) || !(lam_hi / dx_ - sax < 0.999L) || !(lam_lo / dx_ - sax > -0.999L))
        return fail(E2E_ERR_UNSUPPORTED, "spectrograph_format: cross-disperser angle out of range");
    const long double alpha_x = asinl(sax);
    auto h_exact = [&](long double lam) { return (long double)sp->y_c + F * tanl(asinl(lam / dx_ - sax) - alpha_x); };
    long double b[6];
    cheb_mono([&](long double L) { return h_exact(lam0d + L / idl); }, 5, b);
    for (int p = 0; p < 6; ++p)
        for (int q = 0; q < 6; ++q) {
            out->coef_x[p * 6 + q] = (double)cx[p][q];
            out->coef_y[p * 6 + q] = q == 0 ? (double)b[p] : 0.0;
        }
    // ---- residuals of the polynomials (as stored, in double) against the closed forms over every order's range
    auto poly = [&](const double* c, long double L, long double M) {
        long double acc = 0.0L;
        for (int p = 5; p >= 0; --p) {
            long double in = 0.0L;
            for (int q = 5; q >= 0; --q) in = in * M + (long double)c[p * 6 + q];
            acc = acc * L + in;
        }
        return acc;
    };
    long double rx = 0.0L, ry = 0.0L, xlo = 1.0e300L, xhi = -1.0e300L, ylo = 1.0e300L, yhi = -1.0e300L;
    for (int o = 0; o < no; ++o) {
        const long double m = (long double)out->order_m[o], M = (m - m0d) * idm;
        for (int i = 0; i <= 256; ++i) {
            const long double lam = (long double)out->lam_min[o] + ((long double)out->lam_max[o] - (long double)out->lam_min[o]) * (long double)i / 256.0L;
            const long double L = (lam - lam0d) * idl;
            const long double xe = g_exact(m * lam / K - 1.0L), ye = h_exact(lam);
            rx = fmaxl(rx, fabsl(poly(out->coef_x, L, M) - xe));
            ry = fmaxl(ry, fabsl(poly(out->coef_y, L, M) - ye));
            xlo = fminl(xlo, xe); xhi = fmaxl(xhi, xe); ylo = fminl(ylo, ye); yhi = fmaxl(yhi, ye);
        }
    }
    out->residual_x_px = (double)rx; out->residual_y_px = (double)ry;
    out->x_min = (double)xlo; out->x_max = (double)xhi; out->y_min = (double)ylo; out->y_max = (double)yhi;
    // ---- fiber images
    const long double mag = (long double)sp->f_cam_mm / (long double)sp->f_coll_mm / (long double)sp->pixel_um;   // px per micron at the slit
    out->fiber_dy_px = (double)((long double)sp->fiber_core_um * mag);
    out->fiber_dx_px = (double)((long double)sp->fiber_core_um * mag * cosl(alpha) / cosl(beta_c));
    const long double tan_chi = tanl(gam) * s0 / cosl(beta_c);
    out->tilt_tan = (double)tan_chi;
    for (int f = 0; f < sp->n_fibers; ++f) {
        const long double dy = (long double)sp->fiber_height_um[f] * mag;
        out->fiber_dy[f] = (double)dy;
        out->fiber_dx[f] = (double)(tan_chi * dy);
    }
    out->K = (double)K;
    out->px_per_radian = (double)F;
    return E2E_OK;
}
