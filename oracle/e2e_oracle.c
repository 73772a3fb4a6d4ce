/*
 * e2e_oracle.c -- CPU oracle for the echellogram-rendering hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct C written from the paper
 * (Genoni, Landoni et al., arXiv 2008.05858; /root/reference/PAPER.md, cited as P:line) under
 * the readings of SURVEY.md section 8(c) (cited as O1..O7, G1..G18, T1..T3; listed again in
 * DESIGN.md).  It shares no code with the CUDA path (paper_2008_05858_b200/csrc) and is never
 * called by the product: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * What it computes: the frame is the superposition, over fibers, echelle orders and
 * wavelength samples, of the pixel-integrated image of the fiber (geometric fiber profile
 * convolved with the optical PSF), each weighted by the photons in its wavelength bin.
 *
 *   frame[j][i] = sum_f sum_m sum_k  w_{f,m,k} * P(i - x_{f,m,k}, j - y_{f,m,k})
 *
 * restricted per sample to the footprint box of G9 and to the detector (G11).
 *
 * Precision: wavelengths and positions are IEEE double with an exactly specified operation
 * sequence (O1, O2, G8) because the footprint boxes depend on them; the special functions are
 * libm double (erf, erfc, exp; < 1 ulp) used in cancellation-free arrangements; every sum and
 * product after that is long double.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):  P1 mpmath 2-D polar quadrature of the
 * definition, P2 pure-gaussian closed form, P3 flux conservation, P4/P5 photocenter, P6 second
 * moment, P7 symmetries, P8 linearity, P9 integer translation, P10 tabulated == analytic limit and
 * == summed-area form, P11 the paper's own 0.1-px sub-pixel scheme, blaze closed forms,
 * Philox known-answer vectors and noise moments (P12); G21 PSF map: reduction to the constant PSF, mixture of the pinned
 * constant-sigma pixels with independently computed bilinear weights, mixture second moments, box from the largest node
 * sigma, clamping.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_SQRT2   1.41421356237309504880168872420969808
#define ORC_SQRT2PI 2.50662827463100050241576528481104525
#define ORC_PI      3.14159265358979323846264338327950288

typedef struct {
    int32_t nx, ny;
    int32_t n_orders, n_fibers;
    int32_t deg_l, deg_m;
    const int32_t *order_m;
    const double *lam_min, *lam_max;
    const double *fiber_dx, *fiber_dy;
    const double *coef_x, *coef_y;           /* c[p*(deg_m+1)+q] multiplies L^p M^q */
    double lam0, inv_dlam, m0, inv_dm;
    const double *blaze_lam_c, *blaze_amp;   /* amp may be NULL (=1) */
    const double *eff_table; int64_t eff_n; double eff_lam0, eff_dlam;   /* NULL = 1 */
    double samples_per_px;
} orc_format_t;

typedef struct {
    int32_t kind;                            /* 0 analytic, 1 tabulated */
    double fiber_dx_px, fiber_dy_px;         /* full widths Dx, Dy of the fiber image */
    double sigma_x, sigma_y;                 /* optical PSF */
    double support_nsigma;                   /* t of G9 */
    int32_t n_nodes;                         /* Q of O4 (oracle: 32) */
    int32_t tab_npix, tab_os, tab_gx, tab_gy;
    const double *tab;                       /* [gy][gx][npix*os][npix*os] */
    /* G21 ("PSF ... for each wavelength"): analytic PSF MAP.  an_gx * an_gy > 0: the optical PSF was evaluated at the
     * nodes of an an_gx x an_gy grid over the detector (node positions as T3) and sigma_x, sigma_y above are ignored */
    int32_t an_gx, an_gy;
    const double *an_sigma_x, *an_sigma_y;   /* [an_gy][an_gx] */
} orc_psf_t;

typedef struct {
    const double *flux; int64_t n; double lam0, dlam, scale, doppler;
} orc_spectrum_t;

/* ------------------------------------------------------------------------------------------
 * O2 / G8: spectral-format polynomial, fma-Horner in the fixed order
 *   inner: over q = deg_m..0 in M,  outer: over p = deg_l..0 in L,  each step acc = fma(acc, var, coef)
 * ("centroid coordinates" of each spectral fiber image; polynomials per BASELINE.json)
 * ------------------------------------------------------------------------------------------ */
static double poly2(const double *c, int deg_l, int deg_m, double L, double M)
{
    double acc = 0.0;
    for (int p = deg_l; p >= 0; --p) {
        double inner = 0.0;
        for (int q = deg_m; q >= 0; --q)
            inner = fma(inner, M, c[p * (deg_m + 1) + q]);
        acc = fma(acc, L, inner);
    }
    return acc;
}

static void map_lambda(const orc_format_t *f, int o, double lam, double *X, double *Y)
{
    double L = (lam - f->lam0) * f->inv_dlam;
    double M = ((double)f->order_m[o] - f->m0) * f->inv_dm;
    *X = poly2(f->coef_x, f->deg_l, f->deg_m, L, M);
    *Y = poly2(f->coef_y, f->deg_l, f->deg_m, L, M);
}

/* a1 ("sampled on a proper wavelength grid"): N_m = ceil(spp * |x(lmax) - x(lmin)|) */
int64_t orc_order_nsamples(const orc_format_t *f, int32_t o)
{
    double xa, ya, xb, yb;
    map_lambda(f, o, f->lam_min[o], &xa, &ya);
    map_lambda(f, o, f->lam_max[o], &xb, &yb);
    double n = ceil(f->samples_per_px * fabs(xb - xa));
    if (!(n >= 0.0)) return 0;
    return (int64_t)n;
}

/* O3: spectrum by linear interpolation in a uniform table, 0 outside */
static double spectrum_at(const orc_spectrum_t *s, double lam)
{
    double t = (lam / s->doppler - s->lam0) / s->dlam;       /* G13: S'(lam) = S(lam / (1+v/c)) */
    double fl = floor(t);
    if (!(fl >= 0.0) || !(fl <= (double)(s->n - 2))) return 0.0;
    int64_t idx = (int64_t)fl;
    double frac = t - fl;
    return s->flux[idx] + frac * (s->flux[idx + 1] - s->flux[idx]);
}

/* G7 (BASELINE.json "sinc^2 blaze"): E = A * sinc^2(pi * m * (lc/lam - 1)), sinc(0) = 1 */
static double blaze_at(const orc_format_t *f, int o, double lam)
{
    double A = f->blaze_amp ? f->blaze_amp[o] : 1.0;
    double t = (double)f->order_m[o] * (f->blaze_lam_c[o] / lam - 1.0);
    if (fabs(t) < 1e-8) return A;
    double a = ORC_PI * t;
    double sc = sin(a) / a;
    return A * sc * sc;
}

/* optional common throughput T(lam) (P:165 glass transmission), linear interpolation, 1 if absent */
static double eff_at(const orc_format_t *f, double lam)
{
    if (!f->eff_table) return 1.0;
    double t = (lam - f->eff_lam0) / f->eff_dlam;
    double fl = floor(t);
    if (!(fl >= 0.0) || !(fl <= (double)(f->eff_n - 2))) return 0.0;
    int64_t idx = (int64_t)fl;
    double frac = t - fl;
    return f->eff_table[idx] + frac * (f->eff_table[idx + 1] - f->eff_table[idx]);
}

/* a1-a3 for one (fiber, order): lam_k, x_k, y_k, w_k  (O1, O2, O3; G6 midpoint photons per bin) */
void orc_samples(const orc_format_t *f, const orc_spectrum_t *spec, int32_t fiber, int32_t o,
                 int64_t k0, int64_t k1, double *lam, double *x, double *y, double *w)
{
    int64_t N = orc_order_nsamples(f, o);
    if (N <= 0) return;
    double dl = (f->lam_max[o] - f->lam_min[o]) / (double)N;
    for (int64_t k = k0; k < k1; ++k) {
        double l = fma((double)k + 0.5, dl, f->lam_min[o]);                   /* O1 */
        double X, Y;
        map_lambda(f, o, l, &X, &Y);                                         /* O2 */
        lam[k - k0] = l;
        x[k - k0] = X + f->fiber_dx[fiber];
        y[k - k0] = Y + f->fiber_dy[fiber];
        w[k - k0] = spec->scale * spectrum_at(spec, l) * blaze_at(f, o, l) * eff_at(f, l) * dl;   /* O3 */
    }
}

/* ------------------------------------------------------------------------------------------
 * O4: pixel-integrated (uniform ellipse (x) gaussian) PSF
 * ------------------------------------------------------------------------------------------ */
/* Phi(b) - Phi(a) for the standard normal CDF, a <= b, with erfc of same-sign arguments so both
 * tails keep relative accuracy (Phi(z) = erfc(-z/sqrt2)/2) */
static long double dPhi(long double a, long double b)
{
    double ad = (double)(a / ORC_SQRT2), bd = (double)(b / ORC_SQRT2);
    if (ad >= 0.0) return 0.5L * ((long double)erfc(ad) - (long double)erfc(bd));
    if (bd <= 0.0) return 0.5L * ((long double)erfc(-bd) - (long double)erfc(-ad));
    return 0.5L * ((long double)erf(bd) + (long double)erf(-ad));
}

/* Psi(z) = int_{-inf}^{z} Phi = z Phi(z) + phi(z)  split as  relu(z) + Psi(-|z|)  so that the linear part
 * can be differenced exactly; psi_m(t) = Psi(-t) = phi(t) - t * erfc(t/sqrt2)/2,  t >= 0 */
static long double psi_m(long double t)
{
    double td = (double)t;
    return (long double)exp(-0.5 * td * td) / ORC_SQRT2PI - t * 0.5L * (long double)erfc(td / ORC_SQRT2);
}
static long double relu(long double z) { return z > 0.0L ? z : 0.0L; }

/* x-factor of O4 at chord abscissa s: integral over the pixel [u-1/2, u+1/2] of the gaussian centred at s */
static long double ax_factor(long double u, long double s, long double sigma)
{
    return dPhi((u - 0.5L - s) / sigma, (u + 0.5L - s) / sigma);
}

/* y-factor of O4 for a chord of half-length c: (1/2c) int_{-c}^{c} dt int_{v-1/2}^{v+1/2} gauss(y - t) dy
 *   = (sigma / 2c) { [Psi(z+ + c/s) - Psi(z+ - c/s)] - [Psi(z- + c/s) - Psi(z- - c/s)] },  z+- = (v +- 1/2)/sigma */
static long double by_factor(long double v, long double c, long double sigma)
{
    long double zp = (v + 0.5L) / sigma, zm = (v - 0.5L) / sigma, cs = c / sigma;
    long double lin = (relu(zp + cs) - relu(zp - cs)) - (relu(zm + cs) - relu(zm - cs));
    long double smooth = (psi_m(fabsl(zp + cs)) - psi_m(fabsl(zp - cs))) - (psi_m(fabsl(zm + cs)) - psi_m(fabsl(zm - cs)));
    return (sigma / (2.0L * c)) * (lin + smooth);
}

/* P(u, v) of O4: Gauss-Chebyshev (2nd kind) quadrature over the chords of the ellipse,
 *   P = sum_{q=1..Q} (2/(Q+1)) sin^2(th_q) * Ax_q(u) * By_q(v),  th_q = q pi/(Q+1), s_q = a cos th_q, c_q = b sin th_q.
 * Dx = 0 or Dy = 0 degenerate to the plain gaussian factor in that axis (P2). */
long double orc_psf_pixel_l(const orc_psf_t *p, long double u, long double v)
{
    long double a = 0.5L * p->fiber_dx_px, b = 0.5L * p->fiber_dy_px;
    long double sx = p->sigma_x, sy = p->sigma_y;
    int Q = p->n_nodes > 0 ? p->n_nodes : 32;
    if (a <= 0.0L && b <= 0.0L)
        return ax_factor(u, 0.0L, sx) * ax_factor(v, 0.0L, sy);
    long double sum = 0.0L;
    for (int q = 1; q <= Q; ++q) {
        long double th = (long double)q * ORC_PI / (long double)(Q + 1);
        long double sn = sinl(th), cn = cosl(th);
        long double Ax = ax_factor(u, a * cn, sx);
        long double By = (b > 0.0L) ? by_factor(v, b * sn, sy) : ax_factor(v, 0.0L, sy);
        sum += (2.0L / (long double)(Q + 1)) * sn * sn * Ax * By;
    }
    return sum;
}
double orc_psf_pixel(const orc_psf_t *p, double u, double v) { return (double)orc_psf_pixel_l(p, u, v); }

/* G9: footprint box.  Half-widths H = a + t*sigma (analytic) or npix/2 (tabulated); hb = H + 1/2;
 * columns ceil(x - hb) .. floor(x + hb)  (all pixels that touch [x-H, x+H]); same for rows. */
static int psf_is_map(const orc_psf_t *p) { return p->kind == 0 && p->an_gx > 0 && p->an_gy > 0 && p->an_sigma_x && p->an_sigma_y; }

void orc_support(const orc_psf_t *p, double *hbx, double *hby)
{
    if (p->kind == 1) {
        *hbx = 0.5 * (double)p->tab_npix + 0.5;
        *hby = *hbx;
    } else {
        double sx = p->sigma_x, sy = p->sigma_y;
        if (psf_is_map(p)) {                 /* G21: ONE box for the whole frame, from the largest node sigma per axis */
            sx = p->an_sigma_x[0]; sy = p->an_sigma_y[0];
            for (int c = 1; c < p->an_gx * p->an_gy; ++c) {
                if (p->an_sigma_x[c] > sx) sx = p->an_sigma_x[c];
                if (p->an_sigma_y[c] > sy) sy = p->an_sigma_y[c];
            }
        }
        double Hx = 0.5 * p->fiber_dx_px + p->support_nsigma * sx;
        double Hy = 0.5 * p->fiber_dy_px + p->support_nsigma * sy;
        *hbx = Hx + 0.5;
        *hby = Hy + 0.5;
    }
}
void orc_footprint(const orc_psf_t *p, double xk, double yk, int32_t *ilo, int32_t *ihi, int32_t *jlo, int32_t *jhi)
{
    double hbx, hby;
    orc_support(p, &hbx, &hby);
    *ilo = (int32_t)ceil(xk - hbx);  *ihi = (int32_t)floor(xk + hbx);
    *jlo = (int32_t)ceil(yk - hby);  *jhi = (int32_t)floor(yk + hby);
}

/* ------------------------------------------------------------------------------------------
 * O5 / T1-T3: tabulated, field-dependent PSF
 * ------------------------------------------------------------------------------------------ */
/* T3: bilinear blend weights of the 4 surrounding node kernels at detector position (xk, yk);
 * nodes at X_g = g (nx-1)/(gx-1), Y_h = h (ny-1)/(gy-1); weights clamped outside the grid */
static void grid_weights(int gx, int gy, int nx, int ny, double xk, double yk,
                         int *g0, int *h0, long double *fx, long double *fy)
{
    long double tx = 0.0L, ty = 0.0L;
    *g0 = 0; *h0 = 0;
    if (gx > 1) {
        tx = (long double)xk * (long double)(gx - 1) / (long double)(nx - 1);
        if (tx < 0.0L) tx = 0.0L;
        if (tx > (long double)(gx - 1)) tx = (long double)(gx - 1);
        *g0 = (int)floorl(tx); if (*g0 > gx - 2) *g0 = gx - 2;
        tx -= (long double)*g0;
    }
    if (gy > 1) {
        ty = (long double)yk * (long double)(gy - 1) / (long double)(ny - 1);
        if (ty < 0.0L) ty = 0.0L;
        if (ty > (long double)(gy - 1)) ty = (long double)(gy - 1);
        *h0 = (int)floorl(ty); if (*h0 > gy - 2) *h0 = gy - 2;
        ty -= (long double)*h0;
    }
    *fx = tx; *fy = ty;
}
static void field_weights(const orc_psf_t *p, int nx, int ny, double xk, double yk,
                          int *g0, int *h0, long double *fx, long double *fy)
{
    grid_weights(p->tab_gx, p->tab_gy, nx, ny, xk, yk, g0, h0, fx, fy);
}

/* G21: the 4 nodes of the analytic PSF map around (xk, yk) and their bilinear weights (same node positions and clamping
 * as T3); node[c] indexes an_sigma_x / an_sigma_y, c = 2 (row) + (column) */
static void map_nodes(const orc_psf_t *p, int nx, int ny, double xk, double yk, int node[4], long double beta[4])
{
    int g0, h0; long double fx, fy;
    grid_weights(p->an_gx, p->an_gy, nx, ny, xk, yk, &g0, &h0, &fx, &fy);
    int g1 = p->an_gx > 1 ? g0 + 1 : g0, h1 = p->an_gy > 1 ? h0 + 1 : h0;
    node[0] = h0 * p->an_gx + g0; node[1] = h0 * p->an_gx + g1; node[2] = h1 * p->an_gx + g0; node[3] = h1 * p->an_gx + g1;
    beta[0] = (1.0L - fy) * (1.0L - fx); beta[1] = (1.0L - fy) * fx; beta[2] = fy * (1.0L - fx); beta[3] = fy * fx;
}

/* G21: pixel integral of the blended PSF of a sample at (xk, yk): sum over the 4 surrounding nodes of
 * beta_c * P(u, v; sigma_x[c], sigma_y[c]) -- the PSF itself is interpolated between the field points where it was evaluated */
long double orc_psf_map_pixel_l(const orc_psf_t *p, int nx, int ny, double xk, double yk, int i, int j)
{
    int node[4]; long double beta[4];
    map_nodes(p, nx, ny, xk, yk, node, beta);
    long double sum = 0.0L;
    for (int c = 0; c < 4; ++c) {
        if (beta[c] == 0.0L) continue;
        orc_psf_t q = *p;
        q.an_gx = q.an_gy = 0;
        q.sigma_x = p->an_sigma_x[node[c]]; q.sigma_y = p->an_sigma_y[node[c]];
        sum += beta[c] * orc_psf_pixel_l(&q, (long double)i - (long double)xk, (long double)j - (long double)yk);
    }
    return sum;
}
double orc_psf_map_pixel(const orc_psf_t *p, int32_t nx, int32_t ny, double xk, double yk, int32_t i, int32_t j)
{ return (double)orc_psf_map_pixel_l(p, nx, ny, xk, yk, i, j); }

static long double overlap(long double a0, long double a1, long double b0, long double b1)
{
    long double lo = a0 > b0 ? a0 : b0, hi = a1 < b1 ? a1 : b1;
    return hi > lo ? hi - lo : 0.0L;
}

/* T1/T2: the blended kernel is a piecewise-constant density on 1/os-px cells centred on the sample;
 * pixel integral = sum over cells of cell value * (overlap_x * os) * (overlap_y * os) */
long double orc_psf_tab_pixel_l(const orc_psf_t *p, int nx, int ny, double xk, double yk, int i, int j)
{
    int n = p->tab_npix * p->tab_os;
    long double os = (long double)p->tab_os, H = 0.5L * (long double)p->tab_npix;
    int g0, h0; long double fx, fy;
    field_weights(p, nx, ny, xk, yk, &g0, &h0, &fx, &fy);
    int g1 = p->tab_gx > 1 ? g0 + 1 : g0, h1 = p->tab_gy > 1 ? h0 + 1 : h0;
    const double *T00 = p->tab + ((size_t)(h0 * p->tab_gx + g0)) * n * n;
    const double *T01 = p->tab + ((size_t)(h0 * p->tab_gx + g1)) * n * n;
    const double *T10 = p->tab + ((size_t)(h1 * p->tab_gx + g0)) * n * n;
    const double *T11 = p->tab + ((size_t)(h1 * p->tab_gx + g1)) * n * n;
    long double px0 = (long double)i - 0.5L - (long double)xk, px1 = px0 + 1.0L;   /* pixel in kernel coords */
    long double py0 = (long double)j - 0.5L - (long double)yk, py1 = py0 + 1.0L;
    long double sum = 0.0L;
    for (int b = 0; b < n; ++b) {
        long double cy0 = -H + (long double)b / os, cy1 = -H + (long double)(b + 1) / os;
        long double oy = overlap(cy0, cy1, py0, py1);
        if (oy <= 0.0L) continue;
        for (int a = 0; a < n; ++a) {
            long double cx0 = -H + (long double)a / os, cx1 = -H + (long double)(a + 1) / os;
            long double ox = overlap(cx0, cx1, px0, px1);
            if (ox <= 0.0L) continue;
            long double T = (1.0L - fy) * ((1.0L - fx) * T00[b * n + a] + fx * T01[b * n + a])
                          + fy * ((1.0L - fx) * T10[b * n + a] + fx * T11[b * n + a]);
            sum += T * (ox * os) * (oy * os);
        }
    }
    return sum;
}
double orc_psf_tab_pixel(const orc_psf_t *p, int32_t nx, int32_t ny, double xk, double yk, int32_t i, int32_t j)
{ return (double)orc_psf_tab_pixel_l(p, nx, ny, xk, yk, i, j); }

/* ------------------------------------------------------------------------------------------
 * a4 + a5: scatter one sample into a long-double box (O4/O5, O6)
 * box covers columns [bi0, bi0+bw) x rows [bj0, bj0+bh); pixels outside the box or outside the
 * detector are dropped (G11)
 * ------------------------------------------------------------------------------------------ */
#define ORC_MAXFP 160

static void scatter_sample(const orc_format_t *f, const orc_psf_t *p, double xk, double yk, double wk,
                           long double *box, int bi0, int bj0, int bw, int bh)
{
    int32_t ilo, ihi, jlo, jhi;
    orc_footprint(p, xk, yk, &ilo, &ihi, &jlo, &jhi);
    int ncol = ihi - ilo + 1, nrow = jhi - jlo + 1;
    if (ncol <= 0 || nrow <= 0 || ncol > ORC_MAXFP || nrow > ORC_MAXFP) return;
    if (p->kind == 1) {
        for (int j = jlo; j <= jhi; ++j) {
            if (j < 0 || j >= f->ny || j < bj0 || j >= bj0 + bh) continue;
            for (int i = ilo; i <= ihi; ++i) {
                if (i < 0 || i >= f->nx || i < bi0 || i >= bi0 + bw) continue;
                box[(size_t)(j - bj0) * bw + (i - bi0)] += (long double)wk * orc_psf_tab_pixel_l(p, f->nx, f->ny, xk, yk, i, j);
            }
        }
        return;
    }
    if (psf_is_map(p)) {                     /* G21: blend of the 4 surrounding node PSFs, the box is the common one */
        for (int j = jlo; j <= jhi; ++j) {
            if (j < 0 || j >= f->ny || j < bj0 || j >= bj0 + bh) continue;
            for (int i = ilo; i <= ihi; ++i) {
                if (i < 0 || i >= f->nx || i < bi0 || i >= bi0 + bw) continue;
                box[(size_t)(j - bj0) * bw + (i - bi0)] += (long double)wk * orc_psf_map_pixel_l(p, f->nx, f->ny, xk, yk, i, j);
            }
        }
        return;
    }
    long double a = 0.5L * p->fiber_dx_px, b = 0.5L * p->fiber_dy_px;
    long double sx = p->sigma_x, sy = p->sigma_y;
    int Q = p->n_nodes > 0 ? p->n_nodes : 32;
    if (a <= 0.0L && b <= 0.0L) Q = 1;
    long double Ax[ORC_MAXFP], By[ORC_MAXFP];
    for (int q = 1; q <= Q; ++q) {
        long double wq, sq, cq;
        if (a <= 0.0L && b <= 0.0L) { wq = 1.0L; sq = 0.0L; cq = 0.0L; }
        else {
            long double th = (long double)q * ORC_PI / (long double)(Q + 1);
            long double sn = sinl(th), cn = cosl(th);
            wq = (2.0L / (long double)(Q + 1)) * sn * sn;  sq = a * cn;  cq = b * sn;
        }
        for (int i = ilo; i <= ihi; ++i)
            Ax[i - ilo] = ax_factor((long double)i - (long double)xk, sq, sx);
        for (int j = jlo; j <= jhi; ++j)
            By[j - jlo] = (cq > 0.0L) ? by_factor((long double)j - (long double)yk, cq, sy)
                                      : ax_factor((long double)j - (long double)yk, 0.0L, sy);
        for (int j = jlo; j <= jhi; ++j) {
            if (j < 0 || j >= f->ny || j < bj0 || j >= bj0 + bh) continue;
            for (int i = ilo; i <= ihi; ++i) {
                if (i < 0 || i >= f->nx || i < bi0 || i >= bi0 + bw) continue;
                box[(size_t)(j - bj0) * bw + (i - bi0)] += (long double)wk * wq * Ax[i - ilo] * By[j - jlo];
            }
        }
    }
}

/* a1-a5: render the window [i0, i0+wnx) x [j0, j0+wny) of the detector frame (the whole frame when
 * the window is the detector).  out is row-major double [wny][wnx].  Samples are processed in chunks
 * of consecutive k; each chunk accumulates in a private long-double box, boxes are added into a
 * long-double window in chunk order (deterministic).  Returns the number of samples that touched the window. */
#define ORC_CHUNK 128
int64_t orc_render(const orc_format_t *f, const orc_psf_t *p, const orc_spectrum_t *spectra,
                   int32_t i0, int32_t j0, int32_t wnx, int32_t wny, double *out, int32_t nthreads)
{
    size_t npx = (size_t)wnx * (size_t)wny;
    long double *win = (long double *)calloc(npx, sizeof(long double));
    if (!win) return -1;
    double hbx, hby;
    orc_support(p, &hbx, &hby);
    int64_t touched = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    for (int fb = 0; fb < f->n_fibers; ++fb) {
        for (int o = 0; o < f->n_orders; ++o) {
            int64_t N = orc_order_nsamples(f, o);
            int64_t nchunk = (N + ORC_CHUNK - 1) / ORC_CHUNK;
#pragma omp parallel for ordered schedule(dynamic, 1) reduction(+ : touched)
            for (int64_t c = 0; c < nchunk; ++c) {
                int64_t k0 = c * ORC_CHUNK, k1 = k0 + ORC_CHUNK < N ? k0 + ORC_CHUNK : N;
                double lam[ORC_CHUNK], x[ORC_CHUNK], y[ORC_CHUNK], w[ORC_CHUNK];
                orc_samples(f, &spectra[fb], fb, o, k0, k1, lam, x, y, w);
                /* bounding box of the chunk's footprints, clipped to the window */
                int bi0 = INT32_MAX, bi1 = INT32_MIN, bj0 = INT32_MAX, bj1 = INT32_MIN;
                int64_t nt = 0;
                for (int64_t k = 0; k < k1 - k0; ++k) {
                    int32_t ilo, ihi, jlo, jhi;
                    orc_footprint(p, x[k], y[k], &ilo, &ihi, &jlo, &jhi);
                    if (ihi < i0 || ilo >= i0 + wnx || jhi < j0 || jlo >= j0 + wny) { w[k] = NAN; continue; }
                    ++nt;
                    if (ilo < bi0) bi0 = ilo;  if (ihi > bi1) bi1 = ihi;
                    if (jlo < bj0) bj0 = jlo;  if (jhi > bj1) bj1 = jhi;
                }
                long double *box = NULL; int bw = 0, bh = 0;
                if (nt > 0) {
                    if (bi0 < i0) bi0 = i0;  if (bi1 > i0 + wnx - 1) bi1 = i0 + wnx - 1;
                    if (bj0 < j0) bj0 = j0;  if (bj1 > j0 + wny - 1) bj1 = j0 + wny - 1;
                    bw = bi1 - bi0 + 1; bh = bj1 - bj0 + 1;
                    box = (long double *)calloc((size_t)bw * bh, sizeof(long double));
                    for (int64_t k = 0; k < k1 - k0; ++k)
                        if (w[k] == w[k]) scatter_sample(f, p, x[k], y[k], w[k], box, bi0, bj0, bw, bh);
                    touched += nt;
                }
#pragma omp ordered
                {
                    if (box) {
                        for (int jj = 0; jj < bh; ++jj)
                            for (int ii = 0; ii < bw; ++ii)
                                win[(size_t)(bj0 - j0 + jj) * wnx + (bi0 - i0 + ii)] += box[(size_t)jj * bw + ii];
                    }
                }
                free(box);
            }
        }
    }
    for (size_t q = 0; q < npx; ++q) out[q] = (double)win[q];
    free(win);
    return touched;
}

/* sum of all sample weights (injected photons), long-double accumulate: the right-hand side of P3 */
double orc_total_weight(const orc_format_t *f, const orc_spectrum_t *spectra)
{
    long double tot = 0.0L;
    for (int fb = 0; fb < f->n_fibers; ++fb)
        for (int o = 0; o < f->n_orders; ++o) {
            int64_t N = orc_order_nsamples(f, o);
            for (int64_t k0 = 0; k0 < N; k0 += ORC_CHUNK) {
                int64_t k1 = k0 + ORC_CHUNK < N ? k0 + ORC_CHUNK : N;
                double lam[ORC_CHUNK], x[ORC_CHUNK], y[ORC_CHUNK], w[ORC_CHUNK];
                orc_samples(f, &spectra[fb], fb, o, k0, k1, lam, x, y, w);
                for (int64_t k = 0; k < k1 - k0; ++k) tot += w[k];
            }
        }
    return (double)tot;
}
