// Host-only shim around paper_2008_05858_b200/csrc/poly_tables.h (header-only, no CUDA) for tests/test_host_tables.py:
// builds the moment tables of an analytic PSF exactly as e2e_psf_create does and evaluates the fitted polynomials, so that
// the table builder can be checked against closed forms on a machine without a GPU.
#include "../../paper_2008_05858_b200/csrc/poly_tables.h"
#include <cstring>

using namespace e2e;

extern "C" {

// pure gaussian (D = 0) or disk (x) gaussian with Q chord nodes; returns 0 on success and fills the table description
int shim_build(double D, double sigma, double t_support, int Q, int* P, int* npt, int* ncol, int* nrow, int* nyb, int* T,
               double* c0x, double* c0y, double* trunc_err, void** handle)
{
    PsfShape S;
    S.sx = sigma; S.sy = sigma; S.by_gauss = !(D > 0.0);
    const long double a = 0.5L * D;
    if (!(D > 0.0)) {
        ChordTerm ct; ct.s = 0; ct.cs = 0; ct.wq = 1; ct.g = 1; ct.paired = false;
        S.terms.push_back(ct);
    } else {
        for (int q = 1; 2 * q <= Q + 1; ++q) {
            const long double th = (long double)q * kLPi / (long double)(Q + 1), sn = sinl(th), cn = cosl(th);
            ChordTerm ct;
            ct.s = a * cn; const long double c = a * sn;
            ct.cs = c / (long double)sigma; ct.wq = (2.0L / (long double)(Q + 1)) * sn * sn; ct.g = (long double)sigma / (2.0L * c);
            ct.paired = 2 * q != Q + 1;
            if (!ct.paired) ct.s = 0;
            S.terms.push_back(ct);
        }
    }
    const double hb = 0.5 * D + t_support * sigma + 0.5;
    MomentTables* M = new MomentTables;
    if (!build_moment_tables(S, hb, hb, *M)) { delete M; return 1; }
    *P = M->P; *npt = M->npt; *ncol = M->ncol; *nrow = M->nrow; *nyb = M->nyb; *T = M->T;
    *c0x = M->c0x; *c0y = M->c0y; *trunc_err = (double)M->trunc_err;
    *handle = M;
    return 0;
}

// x-factor of term t at window column i for phase dx (fma-Horner over the stored fragment-ordered coefficients)
double shim_eval_x(void* handle, int t, int i, double dx)
{
    const MomentTables& M = *(const MomentTables*)handle;
    double acc = 0.0;
    for (int q = 8 * M.npt - 1; q >= 0; --q) {
        const int tile = i >> 3, lane = ((i & 7) << 2) | ((q & 7) >> 1), e = q & 1, kt = q >> 3;
        acc = fma(acc, dx, M.fx[((((size_t)t * M.nit + tile) * M.npt + kt) * 32 + lane) * 2 + e]);
    }
    return acc;
}

// y-factor of term t at window row j for y-phase dy, through the window the kernel would choose (nearest centre)
double shim_eval_y(void* handle, int t, int j, double dy)
{
    const MomentTables& M = *(const MomentTables*)handle;
    int b = (int)floor((dy + 0.5) * M.nyb);
    if (b < 0) b = 0;
    if (b > M.nyb - 1) b = M.nyb - 1;
    const double yc = ((double)b + 0.5) / (double)M.nyb - 0.5, dl = dy - yc;
    double acc = 0.0;
    for (int p = 7; p >= 0; --p) {
        const int tile = j >> 3, lane = ((j & 7) << 2) | (p >> 1), e = p & 1;
        acc = fma(acc, dl, M.fy[((((size_t)b * M.T + t) * M.njt + tile) * 32 + lane) * 2 + e]);
    }
    return acc;
}

// the same fit evaluated at the far edge of the NEXT window's validity (the kernel keeps a window while |delta| <= 1/nyb)
double shim_eval_y_window(void* handle, int t, int j, int b, double dl)
{
    const MomentTables& M = *(const MomentTables*)handle;
    double acc = 0.0;
    for (int p = 7; p >= 0; --p) {
        const int tile = j >> 3, lane = ((j & 7) << 2) | (p >> 1), e = p & 1;
        acc = fma(acc, dl, M.fy[((((size_t)b * M.T + t) * M.njt + tile) * 32 + lane) * 2 + e]);
    }
    return acc;
}

void shim_free(void* handle) { delete (MomentTables*)handle; }

}  // extern "C"
