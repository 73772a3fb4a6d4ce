// poly_tables.h -- host side of the pixel-phase polynomial tables of the analytic PSF.
//
// For a sample at x in [X, X+1) the pixel-integrated x-factor of chord term t at column X + n is a smooth function
// of the sub-pixel phase d = x - (X + 1/2) in [-1/2, 1/2):
//
//     FX_t,n(d) = wq_t * [ G_x(n - 1/2 - d - s_t) + G_x(n - 1/2 - d + s_t) ],   G_x(u) = Phi((u+1/2)/sx) - Phi((u-1/2)/sx)
//     GY_t,n(d) = g_t * [ E_t((n - d)/sy) - E_t((n - 1 - d)/sy) ],               E_t(z) = Psi(z + c_t/sy) - Psi(z - c_t/sy)
//
// ("surface integral of the convolution between the spatial profile of the fiber and the PSF"; O4 of DESIGN.md).
// Each is replaced by its degree-P Chebyshev interpolant on [-1/2, 1/2], stored in the monomial basis of d and
// evaluated by fma-Horner on the device.  P is the smallest degree of kPolyDegrees whose truncation error, measured
// here in long double against the closed forms on a dense set of phases, is below kPolyTol (far below the fp64
// rounding of the Horner evaluation itself, ~1e-16 of the PSF peak).
#pragma once
#include <cmath>
#include <vector>

namespace e2e {

constexpr int kPolyDegrees[] = {10, 12, 14, 16, 20, 24};
constexpr int kNumPolyDegrees = 6;
constexpr long double kPolyTol = 1.0e-17L;
constexpr long double kLSqrt2 = 1.41421356237309504880168872420969808L;
constexpr long double kLSqrt2Pi = 2.50662827463100050241576528481104525L;
constexpr long double kLPi = 3.14159265358979323846264338327950288L;

// Phi(b) - Phi(a), a <= b, from the tail that keeps both terms small
inline long double cdf_span(long double a, long double b)
{
    if (a >= 0.0L) return 0.5L * (erfcl(a / kLSqrt2) - erfcl(b / kLSqrt2));
    if (b <= 0.0L) return 0.5L * (erfcl(-b / kLSqrt2) - erfcl(-a / kLSqrt2));
    return 0.5L * (erfl(b / kLSqrt2) - erfl(a / kLSqrt2));
}
// Psi(z) = z Phi(z) + phi(z) = max(z, 0) + tail(|z|),  tail(t) = phi(t) - t Phi(-t)
inline long double psi_tail(long double t)
{
    return expl(-0.5L * t * t) / kLSqrt2Pi - t * 0.5L * erfcl(t / kLSqrt2);
}
inline long double psi_diff(long double z, long double cs)   // Psi(z + cs) - Psi(z - cs)
{
    const long double a = z + cs, b = z - cs;
    const long double lin = (a > 0.0L ? a : 0.0L) - (b > 0.0L ? b : 0.0L);
    return lin + (psi_tail(fabsl(a)) - psi_tail(fabsl(b)));
}

struct ChordTerm {          // one (paired) node of the Gauss-Chebyshev chord rule
    long double s;          // chord abscissa >= 0 (px)
    long double cs;         // chord half-length / sigma_y
    long double wq;         // quadrature weight
    long double g;          // sigma_y / (2 c)   (1 when the y-factor is a plain gaussian)
    bool paired;            // stands for the two nodes +-s
};

struct PsfShape {
    long double sx, sy;
    bool by_gauss;          // Dy = 0: y-factor is the pixel-integrated gaussian
    std::vector<ChordTerm> terms;
};

inline long double fx_exact(const PsfShape& S, const ChordTerm& t, long double u)
{
    auto G = [&](long double c) { return cdf_span((c - 0.5L) / S.sx, (c + 0.5L) / S.sx); };
    long double v = G(u - t.s);
    if (t.paired) v += G(u + t.s);
    return t.wq * v;
}
inline long double gy_exact(const PsfShape& S, const ChordTerm& t, long double v)
{
    const long double zm = (v - 0.5L) / S.sy, zp = (v + 0.5L) / S.sy;
    if (S.by_gauss) return cdf_span(zm, zp);
    return t.g * (psi_diff(zp, t.cs) - psi_diff(zm, t.cs));
}

// monomial coefficients (in d, |d| <= hw) of the degree-P Chebyshev interpolant of f on [-hw, hw]
template <class F>
inline void cheb_fit(F f, int P, long double* mono /* [P+1] */, long double hw = 0.5L)
{
    const int N = P + 1;
    std::vector<long double> fv(N), c(N);
    for (int j = 0; j < N; ++j) fv[j] = f(hw * cosl(kLPi * ((long double)j + 0.5L) / (long double)N));
    for (int i = 0; i < N; ++i) {
        long double acc = 0.0L;
        for (int j = 0; j < N; ++j) acc += fv[j] * cosl(kLPi * (long double)i * ((long double)j + 0.5L) / (long double)N);
        c[i] = acc * 2.0L / (long double)N;
    }
    c[0] *= 0.5L;
    // sum_i c_i T_i(tau), tau = d / hw  ->  monomials in tau, then in d
    std::vector<long double> t0(N, 0.0L), t1(N, 0.0L), t2(N, 0.0L), m(N, 0.0L);
    t0[0] = 1.0L;
    m[0] += c[0];
    if (N > 1) { t1[1] = 1.0L; m[1] += c[1]; }
    for (int i = 2; i < N; ++i) {
        for (int k = 0; k < N; ++k) t2[k] = (k > 0 ? 2.0L * t1[k - 1] : 0.0L) - t0[k];
        for (int k = 0; k < N; ++k) m[k] += c[i] * t2[k];
        t0.swap(t1);
        t1.swap(t2);
    }
    long double sc = 1.0L;
    for (int k = 0; k < N; ++k) { mono[k] = m[k] * sc; sc /= hw; }
}

inline long double horner_l(const long double* a, int P, long double d)
{
    long double p = a[P];
    for (int k = P - 1; k >= 0; --k) p = p * d + a[k];
    return p;
}

struct PolyTables {
    int P = 0;                       // degree in use
    int nlo_x = 0, ncol = 0;         // window columns X + nlo_x .. X + nlo_x + ncol - 1
    int nlo_y = 0, nrow = 0;
    int T = 0;                       // chord terms
    std::vector<double> tx;          // [T][P+1][ncol_pad]   (column fastest; pad = multiple of 8, zero polynomials)
    std::vector<double> ty;          // [T][P+1][nrow_pad]
    int ncol_pad = 0, nrow_pad = 0;
    long double trunc_err = 0.0L;    // measured truncation error of the degree chosen
};

// hbx, hby: footprint half-width + 1/2 per axis (G9).  Returns false when no degree of kPolyDegrees reaches kPolyTol.
inline bool build_poly_tables(const PsfShape& S, double hbx, double hby, PolyTables& out)
{
    const double eps = 1e-6;
    out.nlo_x = (int)std::ceil(-hbx - eps);
    out.ncol = (int)std::floor(1.0 + hbx + eps) - out.nlo_x + 1;
    out.nlo_y = (int)std::ceil(-hby - eps);
    out.nrow = (int)std::floor(1.0 + hby + eps) - out.nlo_y + 1;
    out.ncol_pad = (out.ncol + 7) / 8 * 8;
    out.nrow_pad = (out.nrow + 7) / 8 * 8;
    out.T = (int)S.terms.size();
    const int ntest = 24;
    for (int di = 0; di < kNumPolyDegrees; ++di) {
        const int P = kPolyDegrees[di];
        std::vector<long double> mono(P + 1);
        std::vector<double> tx((size_t)out.T * (P + 1) * out.ncol_pad, 0.0), ty((size_t)out.T * (P + 1) * out.nrow_pad, 0.0);
        long double worst = 0.0L;
        for (int t = 0; t < out.T; ++t) {
            const ChordTerm& ct = S.terms[t];
            for (int axis = 0; axis < 2; ++axis) {
                const int cnt = axis == 0 ? out.ncol : out.nrow, pad = axis == 0 ? out.ncol_pad : out.nrow_pad;
                const int nlo = axis == 0 ? out.nlo_x : out.nlo_y;
                std::vector<double>& tab = axis == 0 ? tx : ty;
                for (int c = 0; c < cnt; ++c) {
                    const long double base = (long double)(nlo + c) - 0.5L;      // pixel centre offset from X + 1/2
                    auto f = [&](long double d) { return axis == 0 ? fx_exact(S, ct, base - d) : gy_exact(S, ct, base - d); };
                    cheb_fit(f, P, mono.data());
                    for (int k = 0; k <= P; ++k) tab[((size_t)t * (P + 1) + k) * pad + c] = (double)mono[k];
                    for (int i = 0; i <= ntest; ++i) {
                        const long double d = -0.5L + (long double)i / (long double)ntest;
                        const long double e = fabsl(horner_l(mono.data(), P, d) - f(d));
                        if (e > worst) worst = e;
                    }
                }
            }
        }
        if (worst <= kPolyTol || di == kNumPolyDegrees - 1) {
            out.P = P;
            out.tx.swap(tx);
            out.ty.swap(ty);
            out.trunc_err = worst;
            return worst <= kPolyTol;
        }
    }
    return false;
}

// ------------------------------------------------------------------------------------------------
// Moment tables (render_moment.cuh).  Same polynomials, but
//  * the cell is the set of samples that share one footprint box (G9): first column ilo = ceil(x - hbx), and the
//    phase is d = (x - ilo) - c0x with c0x = hbx - 1/2 (as a double), d in (-1/2, 1/2]; column n = i - ilo >= 0 sits
//    at offset (n - c0x) - d from the sample, so no per-sample mask is left inside a cell;
//  * the coefficients are stored in mma.m8n8k4 fragment order, two k-slots per lane:
//        fy[((b*T + t)*njt + jt)*32 + lane][e]    = cy_{b,t}[p = 2 (lane%4) + e][j = 8 jt + lane/4]   (y-phase window b)
//        fx[((t*nit + it)*npt + qt)*32 + lane][e] = cx_t[q = 8 qt + 2 (lane%4) + e][i = 8 it + lane/4]
//    (zero beyond the degree and beyond the window).
// ------------------------------------------------------------------------------------------------
struct MomentTables {
    int P = 0, npt = 0;              // x: degree, power tiles (8 npt >= P + 1)
    int ncol = 0, nrow = 0;          // largest footprint in columns / rows
    int nit = 0, njt = 0;            // 8-wide tiles per axis
    int T = 0;
    double c0x = 0.0, c0y = 0.0;
    int nyb = 0;                     // y: phase bins, centres -1/2 + (b + 1/2)/nyb, degree-7 fits valid for |dy - centre| <= 1/nyb
    std::vector<double> fx, fy;      // fy[((b*T + t)*njt + jt)*32 + lane][e] = cy_{b,t}[p = 2 (lane%4) + e][j = 8 jt + lane/4]
    long double trunc_err = 0.0L;
};

constexpr int kMomYDegree = 7;       // one 8-deep power tile in y
constexpr int kMomYBins[] = {16, 32, 64, 128, 256};

// The y-phase of the samples of one cell moves by (trace slope) x (1 px) only, so the y-factors do not need a polynomial
// that is good on the whole (-1/2, 1/2]: the range is cut into nyb overlapping windows (centres 1/nyb apart, each fit
// valid for +-1/nyb around its centre) and each window gets its own degree-7 Chebyshev fit -- 8 coefficients = one DMMA
// power tile instead of two or three.  A cell takes the window whose centre is nearest to its first sample (|delta| <=
// 1/(2 nyb)) and keeps it while |delta| <= 1/nyb (render_moment.cuh).  nyb = the coarsest of kMomYBins that reaches kPolyTol.
// force_P / force_nyb > 0: use exactly that x degree / that number of y windows (a PSF map needs one layout for all its nodes)
inline bool build_moment_tables(const PsfShape& S, double hbx, double hby, MomentTables& out, int force_P = 0, int force_nyb = 0)
{
    out.c0x = hbx - 0.5;
    out.c0y = hby - 0.5;
    out.ncol = (int)std::floor(2.0 * hbx) + 1;
    out.nrow = (int)std::floor(2.0 * hby) + 1;
    out.nit = (out.ncol + 7) / 8;
    out.njt = (out.nrow + 7) / 8;
    out.T = (int)S.terms.size();
    const int ntest = 24;
    // ---- x: one polynomial per (term, column) on the whole phase range
    bool okx = false;
    long double worst_x = 0.0L;
    for (int di = 0; di < kNumPolyDegrees && !okx; ++di) {
        const int P = kPolyDegrees[di];
        if (force_P > 0 && P != force_P) continue;
        const int npt = (P + 1 + 7) / 8;
        std::vector<long double> mono(P + 1);
        std::vector<double> fx((size_t)out.T * out.nit * npt * 64, 0.0);
        long double worst = 0.0L;
        for (int t = 0; t < out.T; ++t) {
            const ChordTerm& ct = S.terms[t];
            for (int c = 0; c < out.ncol; ++c) {
                const long double base = (long double)c - (long double)out.c0x;   // pixel centre - sample position at d = 0
                auto f = [&](long double d) { return fx_exact(S, ct, base - d); };
                cheb_fit(f, P, mono.data());
                for (int k = 0; k <= P; ++k) {
                    const int tile = c >> 3, lane = ((c & 7) << 2) | ((k & 7) >> 1), e = k & 1, kt = k >> 3;
                    fx[((((size_t)t * out.nit + tile) * npt + kt) * 32 + lane) * 2 + e] = (double)mono[k];
                }
                for (int i = 0; i <= ntest; ++i) {
                    const long double d = -0.5L + (long double)i / (long double)ntest;
                    const long double e = fabsl(horner_l(mono.data(), P, d) - f(d));
                    if (e > worst) worst = e;
                }
            }
        }
        if (worst <= kPolyTol || di == kNumPolyDegrees - 1 || force_P > 0) {
            out.P = P;
            out.npt = npt;
            out.fx.swap(fx);
            worst_x = worst;
            okx = worst <= kPolyTol;
            break;
        }
    }
    if (!okx) return false;
    // ---- y: windows
    for (int nyb : kMomYBins) {
        if (force_nyb > 0 && nyb != force_nyb) continue;
        const long double hw = 1.0L / (long double)nyb;
        std::vector<long double> mono(kMomYDegree + 1);
        std::vector<double> fy((size_t)nyb * out.T * out.njt * 64, 0.0);
        long double worst = 0.0L;
        for (int b = 0; b < nyb; ++b) {
            const long double yc = -0.5L + ((long double)b + 0.5L) * hw;
            for (int t = 0; t < out.T; ++t) {
                const ChordTerm& ct = S.terms[t];
                for (int c = 0; c < out.nrow; ++c) {
                    const long double base = (long double)c - (long double)out.c0y - yc;
                    auto f = [&](long double d) { return gy_exact(S, ct, base - d); };
                    cheb_fit(f, kMomYDegree, mono.data(), hw);
                    for (int k = 0; k <= kMomYDegree; ++k) {
                        const int tile = c >> 3, lane = ((c & 7) << 2) | (k >> 1), e = k & 1;
                        fy[((((size_t)b * out.T + t) * out.njt + tile) * 32 + lane) * 2 + e] = (double)mono[k];
                    }
                    for (int i = 0; i <= 8; ++i) {
                        const long double d = hw * (-1.0L + (long double)i / 4.0L);
                        const long double e = fabsl(horner_l(mono.data(), kMomYDegree, d) - f(d));
                        if (e > worst) worst = e;
                    }
                }
            }
        }
        if (worst <= kPolyTol) {
            out.nyb = nyb;
            out.fy.swap(fy);
            out.trunc_err = worst > worst_x ? worst : worst_x;
            return true;
        }
    }
    return false;
}

}  // namespace e2e
