// detector.cu -- step a6: the detector stage on the rendered frame.
//
// P:79 "photon noise and all other specific detector noises (e.g. dark current, RON, pixels non-uniform response and
// cross-talk) are added on the final synthetic echellogram".  The paper names the noises only; the algorithm is reading
// G12 of DESIGN.md as re-specified in rounds 2 and 3 (a FIXED number of Philox blocks, shared by the two pixels of a pair: one for
// the Box-Muller pair, at most one more for the Poisson counts; no rejection loop), G19 (PRNU / dark maps, full well, ADC) and G20 (cross-talk
// between read-out ports).  Everything is made of IEEE-exact operations (+ - * / sqrt fma, integer ops; log, exp and
// sin 2 pi y are spelled out below) and this file is compiled with --fmad=false, so the result is reproducible bit for bit
// and independent of the launch geometry: pixel pair q = p >> 1 owns the Philox4x32-10 stream (key = seed, counter = (q, block)).
#include "common.cuh"

#include <algorithm>
#include <cstring>

namespace e2e {

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11): block `block` of pixel `pixel`
// ------------------------------------------------------------------------------------------------
// rk = the 10 round keys (k0 + r 0x9E3779B9, k1 + r 0xBB67AE85), computed once on the host (integer arithmetic: exact)
struct PhiloxKeys { uint32_t a[10], b[10]; };

__device__ __forceinline__ void philox_block(const PhiloxKeys& rk, uint32_t p_lo, uint32_t p_hi, uint32_t block,
                                             uint32_t& w0, uint32_t& w1, uint32_t& w2, uint32_t& w3)
{
    uint32_t x0 = p_lo, x1 = p_hi, x2 = block, x3 = 0u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long m0 = (unsigned long long)0xD2511F53u * x0;      // one IMAD.WIDE each: high and low word
        const unsigned long long m1 = (unsigned long long)0xCD9E8D57u * x2;
        x0 = (uint32_t)(m1 >> 32) ^ x1 ^ rk.a[r]; x1 = (uint32_t)m1;
        x2 = (uint32_t)(m0 >> 32) ^ x3 ^ rk.b[r]; x3 = (uint32_t)m0;
    }
    w0 = x0; w1 = x1; w2 = x2; w3 = x3;
}

// U(hi, lo) = ((hi >> 5) 2^26 + (lo >> 6) + 1/2) 2^-53  in (0, 1)
__device__ __forceinline__ double uniform53(uint32_t hi, uint32_t lo)
{
    const double a = (double)(hi >> 5), b = (double)(lo >> 6);
    return (a * 67108864.0 + b + 0.5) * (1.0 / 9007199254740992.0);
}

// ------------------------------------------------------------------------------------------------
// tables of the stage, rebuilt by every CTA in shared memory (4 KB; ~100 fp64 operations per thread, once)
//   invc[i] = 1 / c_i, logc[i] = -series_log(invc[i]) for the 128 intervals of the mantissa range [0.7071, 1.4142)
//   rcp[n]  = 1 / n (IEEE division), n = 1 .. 255, for the Poisson inversion's p <- (p mu) (1/n)
// ------------------------------------------------------------------------------------------------
// polynomial coefficients in the constant bank: fp64 instructions take them as c[][] operands (an immediate would cost two
// moves per coefficient).  kLog1p: -1/2 .. 1/7;  kSin: Taylor series of sin(2 pi y) in y^2, y^1 .. y^23
__constant__ double kLog1p[6] = {-0.5, 1.0 / 3.0, -1.0 / 4.0, 1.0 / 5.0, -1.0 / 6.0, 1.0 / 7.0};
__constant__ double kSin[12] = {6.283185307179586476925287, -41.34170224039976023396842, 81.60524927607505420339768,
                                -76.70585975306138584163064, 42.05869394489765314498681, -15.09464257682299039182662,
                                3.819952584848282127733792, -0.7181223017785005122317403, 0.1042291622081398411727104,
                                -0.01203158594212062723320257, 0.001130923748251796187770218, -0.00008823533599243005134484484};
__constant__ double kExpC[14] = {1.0, 1.0, 1.0 / 2.0, (1.0 / 2.0) / 3.0, ((1.0 / 2.0) / 3.0) / 4.0, (((1.0 / 2.0) / 3.0) / 4.0) / 5.0,
                                 ((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0, (((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0,
                                 ((((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0) / 8.0,
                                 (((((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0) / 8.0) / 9.0,
                                 ((((((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0) / 8.0) / 9.0) / 10.0,
                                 (((((((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0) / 8.0) / 9.0) / 10.0) / 11.0,
                                 ((((((((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0) / 8.0) / 9.0) / 10.0) / 11.0) / 12.0,
                                 (((((((((((1.0 / 2.0) / 3.0) / 4.0) / 5.0) / 6.0) / 7.0) / 8.0) / 9.0) / 10.0) / 11.0) / 12.0) / 13.0};   // c[i] = c[i-1] / i (IEEE)

struct DetTables {
    double invc[128], logc[128], rcp[256];
};
constexpr unsigned long long kLogOff = 0x3fe6a09e00000000ULL;       // just below sqrt(1/2)

// series log of a normal x > 0 (the generator of the table): x = m 2^e, m in [sqrt(1/2), sqrt(2)); r = (m-1)/(m+1);
// log x = e ln2 + 2 r (1 + r^2/3 + ... + r^22/23), fma-Horner
__device__ double series_log(double x)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(x);
    int e = (int)((b >> 52) & 0x7ff) - 1022;
    b = (b & 0x000fffffffffffffULL) | 0x3fe0000000000000ULL;
    double m = __longlong_as_double((long long)b);
    if (m < 0.70710678118654752440) { m = m * 2.0; e -= 1; }
    const double r = (m - 1.0) / (m + 1.0);
    const double r2 = r * r;
    double P = 1.0 / 23.0;
#pragma unroll
    for (int i = 10; i >= 0; --i) P = fma(P, r2, 1.0 / (double)(2 * i + 1));
    return fma((double)e, 0.693147180559945309417232, (2.0 * r) * P);
}

__device__ __forceinline__ void build_tables(DetTables& T)
{
    for (int i = threadIdx.x; i < 256; i += blockDim.x) {
        if (i < 128) {
            const unsigned long long lo = kLogOff + ((unsigned long long)i << 45), hi = lo + (1ULL << 45);
            const double c = 0.5 * __longlong_as_double((long long)lo) + 0.5 * __longlong_as_double((long long)hi);   // exact
            const double ic = 1.0 / c;
            T.invc[i] = ic;
            T.logc[i] = -series_log(ic);
        }
        T.rcp[i] = i > 0 ? 1.0 / (double)i : 0.0;
    }
    __syncthreads();
}

// table log: t = bits(x) - OFF; k = t >> 52 (arithmetic); i = (t >> 45) & 127; z = bits^-1(bits(x) - (k << 52));
// r = fma(z, invc[i], -1), log1p(r) = r + r^2 (-1/2 + r/3 - r^2/4 + r^3/5 - r^4/6 + r^5/7); log x = fma(k, ln2, logc[i] + log1p(r))
__device__ __forceinline__ double table_log(const DetTables& T, double x)
{
    const unsigned long long ix = (unsigned long long)__double_as_longlong(x);
    const unsigned long long t = ix - kLogOff;
    const long long k = (long long)t >> 52;
    const int i = (int)((t >> 45) & 127);
    const double z = __longlong_as_double((long long)(ix - ((unsigned long long)k << 52)));
    const double r = fma(z, T.invc[i], -1.0);
    double P = kLog1p[5];
#pragma unroll
    for (int i = 4; i >= 0; --i) P = fma(P, r, kLog1p[i]);
    const double y = fma(r * r, P, r);
    return fma((double)k, 0.693147180559945309417232, T.logc[i] + y);
}

// exp(y), |y| < 700: k = rint(y / ln2), r = y - k ln2 (two constants), Taylor to degree 13, times 2^k
__device__ __forceinline__ double spec_exp(double y)
{
    const double k = rint(y * 1.44269504088896340736);
    double r = fma(-k, 6.93147180369123816490e-01, y);
    r = fma(-k, 1.90821492927058770002e-10, r);
    double P = kExpC[13];
#pragma unroll
    for (int i = 12; i >= 0; --i) P = fma(P, r, kExpC[i]);
    const unsigned long long b = (unsigned long long)((long long)k + 1023) << 52;
    return P * __longlong_as_double((long long)b);
}

// sin(2 pi y), y in [0, 1.25]: y -= rint(y); fold to |y| <= 1/4; Taylor series to y^23, fma-Horner in y^2
__device__ __forceinline__ double sin2pi(double y)
{
    y = y - rint(y);
    if (y > 0.25) y = 0.5 - y;
    if (y < -0.25) y = -0.5 - y;
    const double g = y * y;
    double P = kSin[11];
#pragma unroll
    for (int i = 10; i >= 0; --i) P = fma(P, g, kSin[i]);
    return y * P;
}

// the draws of the two pixels 2q, 2q + 1 of pair q (G12 rounds 2 + 3): z1 for the read noise, cnt = Poisson(mu).  The pixels of a
// pair share the Philox blocks of the pair's stream (counter = (q, block)): block 0 -> one Box-Muller pair, its cos half for
// pixel 2q and its sin half for pixel 2q + 1; block 1 -> the two uniforms of the Poisson inversions; block 2 -> the normals of
// the Cornish-Fisher branch.  want: bit i set = pixel i is asked for (the other one must come with mu = 0).
__device__ __forceinline__ void pair_draws(const DetTables& T, const PhiloxKeys& rk, unsigned long long q, const double (&mu)[2],
                                           unsigned want, double (&z1_out)[2], double (&cnt_out)[2])
{
    uint32_t w0, w1, w2, w3;
    philox_block(rk, (uint32_t)q, (uint32_t)(q >> 32), 0u, w0, w1, w2, w3);
    {
        const double u1 = uniform53(w0, w1), u2 = uniform53(w2, w3);
        const double rho = sqrt(-2.0 * table_log(T, u1));
        z1_out[0] = (want & 1u) ? rho * sin2pi(u2 + 0.25) : 0.0;      // cos(2 pi u2)
        z1_out[1] = (want & 2u) ? rho * sin2pi(u2) : 0.0;
    }
    const bool lit0 = mu[0] > 0.0, lit1 = mu[1] > 0.0;
    const bool small = (lit0 && mu[0] < 64.0) || (lit1 && mu[1] < 64.0);
    const bool large = (lit0 && !(mu[0] < 64.0)) || (lit1 && !(mu[1] < 64.0));
    double v[2] = {0.0, 0.0}, z2[2] = {0.0, 0.0};
    if (small) {                                          // inversion by sequential search, one uniform per pixel
        philox_block(rk, (uint32_t)q, (uint32_t)(q >> 32), 1u, w0, w1, w2, w3);
        v[0] = uniform53(w0, w1);
        v[1] = uniform53(w2, w3);
    }
    if (large) {                                          // normal + first Cornish-Fisher term
        philox_block(rk, (uint32_t)q, (uint32_t)(q >> 32), 2u, w0, w1, w2, w3);
        const double u1 = uniform53(w0, w1), u2 = uniform53(w2, w3);
        const double rho = sqrt(-2.0 * table_log(T, u1));
        z2[0] = rho * sin2pi(u2 + 0.25);
        z2[1] = rho * sin2pi(u2);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        double cnt;
        if (!(mu[i] > 0.0)) {
            cnt = 0.0;
        } else if (mu[i] < 64.0) {
            int n = 0;
            // Exact shortcut for the PSF wings (mu << 1, about half of an echellogram's illuminated pixels): the search
            // returns n = 0 iff v <= F0 = spec_exp(-mu), and F0 >= (1 - mu)(1 - 6e-16) (e^-mu >= 1 - mu; spec_exp is within
            // 5e-16 relative of e^y, pinned by the oracle's tests), so v < (1 - mu) - 1e-15 implies v <= F0: same n, no exp.
            if (!(mu[i] < 0.5 && v[i] < (1.0 - mu[i]) - 1.0e-15)) {
                double pr = spec_exp(-mu[i]), F = pr;
                while (v[i] > F && n < 255) {
                    n += 1;
                    pr = (pr * mu[i]) * T.rcp[n];
                    F = F + pr;
                }
            }
            cnt = (double)n;
        } else {
            const double a = sqrt(mu[i]) * z2[i];
            const double b = (z2[i] * z2[i] - 1.0) * (1.0 / 6.0);
            cnt = floor(((mu[i] + a) + b) + 0.5);
            if (cnt < 0.0) cnt = 0.0;
        }
        cnt_out[i] = cnt;
    }
}

// one pixel alone (the cross-talk kernel walks the ports, not the pairs): the draws of its pair, its own half
__device__ __forceinline__ void pixel_draws(const DetTables& T, const PhiloxKeys& rk, unsigned long long gp, double mu, double& z1,
                                            double& cnt)
{
    const bool odd = (gp & 1ull) != 0;
    const double mu2[2] = {odd ? 0.0 : mu, odd ? mu : 0.0};
    double z[2], c[2];
    pair_draws(T, rk, gp >> 1, mu2, odd ? 2u : 1u, z, c);
    z1 = odd ? z[1] : z[0];
    cnt = odd ? c[1] : c[0];
}

// parameters of one launch (by value)
struct DetParams {
    e2e_detector_t base;
    PhiloxKeys rk;
    const double* prnu;            // whole-frame maps (indexed by the pixel's index in the frame) or nullptr
    const double* dark;
    double full_well, e_per_adu, adu_max;
    int n_ports, port_w;           // cross-talk: ports and columns per port (0 = none)
    int nx;
    double xtalk[16 * 16];         // X[a][b]
};

__device__ __forceinline__ double adc(const DetParams& D, double v)
{
    double a = floor((v / D.e_per_adu + D.base.bias) + 0.5);
    if (a < 0.0) a = 0.0;
    if (a > D.adu_max) a = D.adu_max;
    return a;
}

template <typename OutT>
__device__ __forceinline__ void store_out(OutT* out, long long p, double v);
template <>
__device__ __forceinline__ void store_out<double>(double* out, long long p, double v) { out[p] = v; }
template <>
__device__ __forceinline__ void store_out<uint16_t>(uint16_t* out, long long p, double v) { out[p] = (uint16_t)(unsigned)v; }   // whole number in [0, 65535]

// in / out point at pixel p0 of the frame (the host path applies the stage band by band); the stream is keyed by the
// pixel's index in the whole frame, so the result does not depend on how the frame is split into launches.  in may
// alias out (each pixel is read before it is written, by the same thread): no __restrict__ on the two.
// GENERAL = false: the basic stage (no maps, no well, no ADC) without the tests for them.  Thread <-> pixel pair (G12 round 3):
// pair j of the launch = global pair (p0 >> 1) + j = local pixels 2 j - (p0 & 1) + {0, 1}; a launch that starts or ends inside
// a pair computes that pair's draws for the one pixel it owns.  VEC: p0 is even and both pointers allow 16-byte (in, fp64 out)
// and 4-byte (uint16 out) accesses: one load and one store per pair.
template <typename OutT>
struct OutPair;
template <>
struct OutPair<double> { typedef double2 type; static __device__ __forceinline__ double2 make(double a, double b) { return make_double2(a, b); } };
template <>
struct OutPair<uint16_t> {
    typedef ushort2 type;
    static __device__ __forceinline__ ushort2 make(double a, double b) { return make_ushort2((unsigned short)(unsigned)a, (unsigned short)(unsigned)b); }
};

template <typename OutT, bool GENERAL, bool VEC>
__global__ void __launch_bounds__(256) detector_kernel(const double* in, OutT* out, long long n, long long p0, DetParams D)
{
    __shared__ DetTables T;
    build_tables(T);
    const long long stride = (long long)gridDim.x * 256;
    const bool use_adc = GENERAL && D.e_per_adu > 0.0;
    const long long shift = p0 & 1;                              // local index of the first pair's even pixel is -shift
    const long long npairs = (n + shift + 1) >> 1;
    const unsigned long long q0 = (unsigned long long)p0 >> 1;
    for (long long j = (long long)blockIdx.x * 256 + threadIdx.x; j < npairs; j += stride) {
        const long long pl = 2 * j - shift;                      // local index of the pair's even pixel
        const bool ok0 = pl >= 0, ok1 = pl + 1 < n;
        double f[2];
        if (VEC && ok1) {
            const double2 v = *reinterpret_cast<const double2*>(in + pl);
            f[0] = v.x; f[1] = v.y;
        } else {
            f[0] = ok0 ? in[pl] : 0.0;
            f[1] = ok1 ? in[pl + 1] : 0.0;
        }
        double mu[2], z1[2], e[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const bool ok = i ? ok1 : ok0;
            double g = D.base.gain, dk = D.base.dark_e;
            if (GENERAL) {
                const unsigned long long gp = (unsigned long long)(p0 + pl + i);
                if (D.prnu && ok) g = g * __ldg(D.prnu + gp);
                if (D.dark && ok) dk = __ldg(D.dark + gp);
            }
            double m = g * f[i] + dk;
            if (!(m > 0.0) || !ok) m = 0.0;
            mu[i] = m;
        }
        pair_draws(T, D.rk, q0 + (unsigned long long)j, mu, 3u, z1, e);
        double r[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            if (GENERAL && D.full_well > 0.0 && e[i] > D.full_well) e[i] = D.full_well;
            if (!use_adc) r[i] = (e[i] + D.base.bias) + D.base.ron_e * z1[i];
            else r[i] = adc(D, e[i] + D.base.ron_e * z1[i]);
        }
        if (VEC && ok1) {
            *reinterpret_cast<typename OutPair<OutT>::type*>(out + pl) = OutPair<OutT>::make(r[0], r[1]);
        } else {
            if (ok0) store_out<OutT>(out, pl, r[0]);
            if (ok1) store_out<OutT>(out, pl + 1, r[1]);
        }
    }
}

// cross-talk (G20): thread <-> (row, in-port column c); it draws the video signal v_b = e + ron z1 of that column in every
// port b, then writes s_a = v_a + sum_{b != a, ascending} X[a][b] v_b (+ bias, or through the ADC) for every port a.
// Reads of one thread precede its writes and no other thread touches those pixels: in may alias out.
template <typename OutT>
__global__ void __launch_bounds__(128) detector_xtalk_kernel(const double* in, OutT* out, long long n_rows, long long p0, DetParams D)
{
    __shared__ DetTables T;
    __shared__ double V[16][128];
    build_tables(T);
    const int W = D.port_w, np = D.n_ports;
    const long long per_row = (W + 127) / 128;                  // CTAs per row
    const bool use_adc = D.e_per_adu > 0.0;
    for (long long blk = blockIdx.x; blk < n_rows * per_row; blk += gridDim.x) {
        const long long row = blk / per_row;
        const int c = (int)(blk - row * per_row) * 128 + threadIdx.x;
        if (c < W) {
            for (int b = 0; b < np; ++b) {
                const long long p = row * D.nx + (long long)b * W + c;
                const unsigned long long gp[1] = {(unsigned long long)(p0 + p)};
                double g = D.base.gain;
                if (D.prnu) g = g * __ldg(D.prnu + gp[0]);
                double mu[1] = {g * in[p] + (D.dark ? __ldg(D.dark + gp[0]) : D.base.dark_e)};
                if (!(mu[0] > 0.0)) mu[0] = 0.0;
                double z1[1], e[1];
                pixel_draws(T, D.rk, gp[0], mu[0], z1[0], e[0]);
                if (D.full_well > 0.0 && e[0] > D.full_well) e[0] = D.full_well;
                V[b][threadIdx.x] = e[0] + D.base.ron_e * z1[0];
            }
            for (int a = 0; a < np; ++a) {
                double s = V[a][threadIdx.x];
                for (int b = 0; b < np; ++b)
                    if (b != a) s = s + D.xtalk[a * np + b] * V[b][threadIdx.x];
                const double r = use_adc ? adc(D, s) : s + D.base.bias;
                store_out<OutT>(out, row * D.nx + (long long)a * W + c, r);
            }
        }
    }
}

static int resident_ctas(int threads)
{
    static int sms[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148 * 8;
    if (!sms[dev]) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        sms[dev] = n;
    }
    return sms[dev] * (2048 / threads);
}

template <typename OutT>
static int launch_detector_any(const double* d_in, OutT* d_out, long long n, int nx, const DetParams& D, cudaStream_t stream, long long p0)
{
    if (n <= 0) return E2E_OK;
    if (D.n_ports > 1) {
        const long long rows = n / nx, per_row = (D.port_w + 127) / 128;
        const long long blocks = std::min<long long>(rows * per_row, resident_ctas(128));
        detector_xtalk_kernel<OutT><<<(unsigned)blocks, 128, 0, stream>>>(d_in, d_out, rows, p0, D);
    } else {
        const long long per = 256 * 2;                               // one pixel pair per thread and iteration
        const long long blocks = std::min<long long>((n + 1 + per - 1) / per, resident_ctas(256));
        const bool general = D.prnu || D.dark || D.full_well > 0.0 || D.e_per_adu > 0.0;
        const bool vec = (p0 & 1) == 0 && ((uintptr_t)d_in & 15) == 0 && ((uintptr_t)d_out & (2 * sizeof(OutT) - 1)) == 0;
        if (general && vec) detector_kernel<OutT, true, true><<<(unsigned)blocks, 256, 0, stream>>>(d_in, d_out, n, p0, D);
        else if (general) detector_kernel<OutT, true, false><<<(unsigned)blocks, 256, 0, stream>>>(d_in, d_out, n, p0, D);
        else if (vec) detector_kernel<OutT, false, true><<<(unsigned)blocks, 256, 0, stream>>>(d_in, d_out, n, p0, D);
        else detector_kernel<OutT, false, false><<<(unsigned)blocks, 256, 0, stream>>>(d_in, d_out, n, p0, D);
    }
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "detector kernel launch");
    return E2E_OK;
}

static DetParams basic_params(const e2e_detector_t& det)
{
    DetParams D;
    memset(&D, 0, sizeof(D));
    D.base = det;
    for (int r = 0; r < 10; ++r) {
        D.rk.a[r] = (uint32_t)det.seed + (uint32_t)r * 0x9E3779B9u;
        D.rk.b[r] = (uint32_t)(det.seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    return D;
}

int launch_detector(const double* d_in, double* d_out, long long n, const e2e_detector_t& det, cudaStream_t stream, long long p0)
{
    return launch_detector_any<double>(d_in, d_out, n, 1, basic_params(det), stream, p0);
}

// full stage.  d_in / d_out point at pixel p0 (a whole number of rows from the frame start when cross-talk is on);
// the maps are whole-frame pointers.  out16 selects the uint16 ADC output.
int launch_detector_ex(const double* d_in, void* d_out, bool out16, long long n, int nx, const e2e_detector_ex_t& det,
                       cudaStream_t stream, long long p0)
{
    DetParams D = basic_params(det.base);
    D.prnu = det.d_prnu; D.dark = det.d_dark;
    D.full_well = det.full_well_e; D.e_per_adu = det.e_per_adu; D.adu_max = det.adu_max;
    D.nx = nx;
    if (det.xtalk && det.n_ports > 1) {
        D.n_ports = det.n_ports; D.port_w = nx / det.n_ports;
        for (int i = 0; i < det.n_ports * det.n_ports; ++i) D.xtalk[i] = det.xtalk[i];
    }
    if (out16) return launch_detector_any<uint16_t>(d_in, (uint16_t*)d_out, n, nx, D, stream, p0);
    return launch_detector_any<double>(d_in, (double*)d_out, n, nx, D, stream, p0);
}

}  // namespace e2e
