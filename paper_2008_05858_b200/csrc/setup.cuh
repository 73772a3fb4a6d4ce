// setup.cuh -- steps a1-a3: wavelength grid, photon weight, detector position of every sample.
// ("sampled on a proper wavelength grid"; P:45/P:75 photons per wavelength bin; P:165 blaze; P:63 positions)
#pragma once
#include "common.cuh"

namespace e2e {

// order-preserving map double -> uint64 so that atomicMin/atomicMax on the integers order the doubles
__device__ __forceinline__ unsigned long long enc_double(double v)
{
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ULL);
}
inline double dec_double(unsigned long long u)
{
    unsigned long long b = (u >> 63) ? (u & 0x7fffffffffffffffULL) : ~u;
    double v;
    memcpy(&v, &b, 8);
    return v;
}

// a1 + a3 (base trace, no fiber offset) for sample k of order o
__device__ __forceinline__ void sample_position(const FormatView& f, int o, long long k, double& lam, double& X, double& Y)
{
    lam = fma((double)k + 0.5, f.dl[o], f.lam_min[o]);                    // O1
    double L = __dmul_rn(__dsub_rn(lam, f.lam0), f.inv_dlam);              // O2
    double M = __dmul_rn(__dsub_rn((double)f.order_m[o], f.m0), f.inv_dm);
    X = poly2(f.coef_x, f.deg_l, f.deg_m, L, M);
    Y = poly2(f.coef_y, f.deg_l, f.deg_m, L, M);
}

// the same positions from the per-order inner sums (format_create): outer Horner in L only.  The padded leading
// steps compute fma(0, L, 0) = 0 and fma(0, L, c) = c exactly, so the result has the bits of sample_position.
__device__ __forceinline__ void sample_position_fast(const FormatView& f, int o, long long k, double& lam, double& X, double& Y)
{
    lam = fma((double)k + 0.5, __ldg(f.dl + o), __ldg(f.lam_min + o));     // O1
    const double L = __dmul_rn(__dsub_rn(lam, f.lam0), f.inv_dlam);        // O2
    const double* cx = f.inner_x + (size_t)o * (kMaxDeg + 1);
    const double* cy = f.inner_y + (size_t)o * (kMaxDeg + 1);
    double ax = 0.0, ay = 0.0;
#pragma unroll
    for (int p = kMaxDeg; p >= 0; --p) {
        ax = fma(ax, L, __ldg(cx + p));
        ay = fma(ay, L, __ldg(cy + p));
    }
    X = ax;
    Y = ay;
}

// e2e_format_create: one pass over every sample of every order.
//   spacing[o] = (min, max) over k of x_{k+1} - x_k   (monotone  <=>  min > 0 or max < 0)
//   bins[o][b] = (min, max) of y over the samples with floor((x + pad) / 64) == b
__global__ void scan_format_kernel(FormatView f, int n_bins, unsigned long long* spacing_min,
                                   unsigned long long* spacing_max, unsigned long long* bin_ymin,
                                   unsigned long long* bin_ymax)
{
    int o = blockIdx.y;
    long long N = f.nsamp[o];
    long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double dmin = INFINITY, dmax = -INFINITY;
    if (k < N) {
        double lam, X, Y;
        sample_position(f, o, k, lam, X, Y);
        if (k + 1 < N) {
            double l1, X1, Y1;
            sample_position(f, o, k + 1, l1, X1, Y1);
            dmin = dmax = X1 - X;
        }
        double bx = floor((X + (double)kBinPad) * (1.0 / (double)(1 << kBinShift)));
        if (bx >= 0.0 && bx < (double)n_bins && Y == Y) {
            int b = (int)bx;
            atomicMin(&bin_ymin[(size_t)o * n_bins + b], enc_double(Y));
            atomicMax(&bin_ymax[(size_t)o * n_bins + b], enc_double(Y));
        }
        if (!(X == X) || !(Y == Y)) { dmin = -INFINITY; dmax = INFINITY; }   // NaN position: flag as non-monotone
    }
    for (int s = 16; s > 0; s >>= 1) {
        dmin = fmin(dmin, __shfl_xor_sync(0xffffffffu, dmin, s));
        dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, s));
    }
    if ((threadIdx.x & 31) == 0) {
        if (dmin != INFINITY) atomicMin(&spacing_min[o], enc_double(dmin));
        if (dmax != -INFINITY) atomicMax(&spacing_max[o], enc_double(dmax));
    }
}

// a2: spectrum table, linear interpolation, 0 outside (O3; G13 doppler on the wavelength axis)
__device__ __forceinline__ double spectrum_at(const e2e_spectrum_t& s, double lam)
{
    double t = __ddiv_rn(__dsub_rn(__ddiv_rn(lam, s.doppler), s.lam0), s.dlam);
    double fl = floor(t);
    if (!(fl >= 0.0) || !(fl <= (double)(s.n - 2))) return 0.0;
    long long idx = (long long)fl;
    double frac = __dsub_rn(t, fl);
    double f0 = __ldg(s.d_flux + idx), f1 = __ldg(s.d_flux + idx + 1);
    return __dadd_rn(f0, __dmul_rn(frac, __dsub_rn(f1, f0)));
}

// G7: E = A sinc^2(pi m (lam_c / lam - 1)), sinc(0) = 1
__device__ __forceinline__ double blaze_at(const FormatView& f, int o, double lam)
{
    double A = f.blaze_amp ? f.blaze_amp[o] : 1.0;
    double t = __dmul_rn((double)f.order_m[o], __dsub_rn(__ddiv_rn(f.blaze_lam_c[o], lam), 1.0));
    if (fabs(t) < 1e-8) return A;
    double a = __dmul_rn(3.14159265358979323846, t);
    double sc = __ddiv_rn(sin(a), a);
    return __dmul_rn(__dmul_rn(A, sc), sc);
}

// optional common throughput T(lam) (P:165 glass transmission)
__device__ __forceinline__ double eff_at(const FormatView& f, double lam)
{
    if (!f.eff_table) return 1.0;
    double t = __ddiv_rn(__dsub_rn(lam, f.eff_lam0), f.eff_dlam);
    double fl = floor(t);
    if (!(fl >= 0.0) || !(fl <= (double)(f.eff_n - 2))) return 0.0;
    long long idx = (long long)fl;
    double frac = __dsub_rn(t, fl);
    double f0 = __ldg(f.eff_table + idx), f1 = __ldg(f.eff_table + idx + 1);
    return __dadd_rn(f0, __dmul_rn(frac, __dsub_rn(f1, f0)));
}

// a1-a3 for every strip (fiber, order) of a render: blockIdx.y = strip = fiber * n_orders + order.
// Coalesced: thread <-> sample, structure-of-arrays output.
// strip_ids (optional): the strips of this launch (the host path sets up one row band at a time); strips is then the
// whole strip table.
__global__ void setup_samples_kernel(FormatView f, SpectraParam sp, const Strip* __restrict__ strips,
                                     int strip0, double* __restrict__ out_lam, double* __restrict__ out_x,
                                     double* __restrict__ out_y, double* __restrict__ out_w,
                                     const int* __restrict__ strip_ids = nullptr, Strip single = Strip{0, -1})
{
    int sidx = strip_ids ? strip_ids[blockIdx.y] : strip0 + blockIdx.y;
    int fiber = sidx / f.n_orders, o = sidx - fiber * f.n_orders;
    // single.n >= 0: a one-strip launch whose strip travels as a kernel parameter (e2e_setup_samples: no device table)
    Strip st = single.n >= 0 ? single : strips[strip_ids ? sidx : blockIdx.y];
    long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= st.n) return;
    double lam, X, Y;
    sample_position_fast(f, o, k, lam, X, Y);
    const e2e_spectrum_t& s = sp.s[fiber];
    double w = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(s.scale, spectrum_at(s, lam)), blaze_at(f, o, lam)), eff_at(f, lam)),
                         f.dl[o]);
    long long q = st.off + k;
    if (out_lam) out_lam[q] = lam;
    if (out_x) out_x[q] = __dadd_rn(X, f.fiber_dx[fiber]);
    if (out_y) out_y[q] = __dadd_rn(Y, f.fiber_dy[fiber]);
    if (out_w) out_w[q] = w;
}

}  // namespace e2e
