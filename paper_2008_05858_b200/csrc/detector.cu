// detector.cu -- step a6: Poisson photon noise + gaussian read noise on the rendered frame.
//
// P:79 "photon noise and all other specific detector noises (e.g. dark current, RON ...) are added on the
// final synthetic echellogram".  The paper names the noises only; the algorithm is reading G12 of DESIGN.md.
// It is made of IEEE-exact operations only (+ - * / sqrt fma and integer ops; the log and exp are spelled
// out below), and this file is compiled with --fmad=false, so the result is reproducible bit for bit and
// independent of the launch geometry: pixel p owns the Philox4x32-10 stream (key = seed, counter = (p, block)).
#include "common.cuh"

namespace e2e {

// Philox4x32-10 stream of one pixel, consumed a whole counter block (4 words = 2 uniforms) at a time so that the
// words stay in registers; the word order is the stream's: block 0 words 0..3, block 1 words 0..3, ...
struct Philox {
    uint32_t k0, k1;      // key
    uint32_t c0, c1;      // pixel index (low, high)
    uint32_t block;       // next counter block

    __device__ __forceinline__ void init(uint64_t seed, uint64_t pixel)
    {
        k0 = (uint32_t)seed; k1 = (uint32_t)(seed >> 32);
        c0 = (uint32_t)pixel; c1 = (uint32_t)(pixel >> 32);
        block = 0;
    }
    __device__ __forceinline__ void next_block(uint32_t& w0, uint32_t& w1, uint32_t& w2, uint32_t& w3)
    {
        uint32_t x0 = c0, x1 = c1, x2 = block, x3 = 0, ka = k0, kb = k1;
#pragma unroll
        for (int r = 0; r < 10; ++r) {
            uint32_t h0 = __umulhi(0xD2511F53u, x0), l0 = 0xD2511F53u * x0;
            uint32_t h1 = __umulhi(0xCD9E8D57u, x2), l1 = 0xCD9E8D57u * x2;
            uint32_t y0 = h1 ^ x1 ^ ka, y2 = h0 ^ x3 ^ kb;
            x0 = y0; x1 = l1; x2 = y2; x3 = l0;
            ka += 0x9E3779B9u; kb += 0xBB67AE85u;
        }
        w0 = x0; w1 = x1; w2 = x2; w3 = x3;
        block += 1;
    }
    // u = ((hi >> 5) * 2^26 + (lo >> 6) + 1/2) * 2^-53  in (0, 1)
    static __device__ __forceinline__ double uniform(uint32_t hi, uint32_t lo)
    {
        double a = (double)(hi >> 5), b = (double)(lo >> 6);
        return (a * 67108864.0 + b + 0.5) * (1.0 / 9007199254740992.0);
    }
};

// natural log of a normal x > 0: x = m 2^e, m in [sqrt(1/2), sqrt(2)); r = (m-1)/(m+1);
// log x = e ln2 + 2 r (1 + r^2/3 + ... + r^22/23), fma-Horner
__device__ __forceinline__ double spec_log(double x)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(x);
    int e = (int)((b >> 52) & 0x7ff) - 1022;
    b = (b & 0x000fffffffffffffULL) | 0x3fe0000000000000ULL;
    double m = __longlong_as_double((long long)b);
    if (m < 0.70710678118654752440) { m = m * 2.0; e -= 1; }
    double r = (m - 1.0) / (m + 1.0);
    double r2 = r * r;
    double P = 1.0 / 23.0;
#pragma unroll
    for (int i = 10; i >= 0; --i) P = fma(P, r2, 1.0 / (double)(2 * i + 1));
    return fma((double)e, 0.693147180559945309417232, (2.0 * r) * P);
}

// exp(y), |y| < 700: k = rint(y / ln2), r = y - k ln2 (two constants), Taylor to degree 13, times 2^k
__device__ __forceinline__ double spec_exp(double y)
{
    double k = rint(y * 1.44269504088896340736);
    double r = fma(-k, 6.93147180369123816490e-01, y);
    r = fma(-k, 1.90821492927058770002e-10, r);
    double c[14];
    c[0] = 1.0;
#pragma unroll
    for (int i = 1; i <= 13; ++i) c[i] = c[i - 1] / (double)i;
    double P = c[13];
#pragma unroll
    for (int i = 12; i >= 0; --i) P = fma(P, r, c[i]);
    unsigned long long b = (unsigned long long)((long long)k + 1023) << 52;
    return P * __longlong_as_double((long long)b);
}

// the draws of one pixel (G12): z1 for the read noise, cnt = Poisson(mu)
__device__ __forceinline__ void detector_draws(uint64_t seed, long long p, double mu, double& z1_out, double& cnt_out)
{
    Philox g;
    g.init(seed, (uint64_t)p);
    // Marsaglia polar pair: the rejection loop only draws (v1, v2, q); the log / sqrt run once after it, converged
    double v1, v2, q;
    uint32_t w0, w1, w2, w3;
    do {
        g.next_block(w0, w1, w2, w3);
        v1 = 2.0 * Philox::uniform(w0, w1) - 1.0;
        v2 = 2.0 * Philox::uniform(w2, w3) - 1.0;
        q = fma(v1, v1, v2 * v2);
    } while (!(q < 1.0 && q > 0.0));
    const double fz = sqrt(-2.0 * spec_log(q) / q);
    const double z1 = v1 * fz, z2 = v2 * fz;
    double cnt;
    if (!(mu > 0.0)) {
        cnt = 0.0;
    } else if (mu < 64.0) {                        // Knuth multiplication method
        bool second = false;                       // the uniforms after the gaussian pair start on a block boundary
        auto next_u = [&]() {
            second = !second;
            if (second) { g.next_block(w0, w1, w2, w3); return Philox::uniform(w0, w1); }
            return Philox::uniform(w2, w3);
        };
        double L = spec_exp(-mu), prod = next_u();
        cnt = 0.0;
        while (prod > L) { cnt += 1.0; prod = prod * next_u(); }
    } else {                                       // normal + first Cornish-Fisher term
        double a = sqrt(mu) * z2;
        double b = (z2 * z2 - 1.0) / 6.0;
        cnt = floor(((mu + a) + b) + 0.5);
        if (cnt < 0.0) cnt = 0.0;
    }
    z1_out = z1; cnt_out = cnt;
}

// in / out point at pixel p0 of the frame (the host path applies the stage band by band); the stream is keyed by the
// pixel's index in the whole frame, so the result does not depend on how the frame is split into launches
__global__ void __launch_bounds__(256, 6) detector_kernel(const double* __restrict__ in, double* __restrict__ out, long long n, long long p0, e2e_detector_t det)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    double mu = det.gain * in[p] + det.dark_e;
    if (!(mu > 0.0)) mu = 0.0;
    double z1, cnt;
    detector_draws(det.seed, p0 + p, mu, z1, cnt);
    out[p] = (cnt + det.bias) + det.ron_e * z1;
}

// full detector stage (e2e.h e2e_apply_detector_ex; G19): PRNU / dark maps, full well, ADC
__global__ void detector_ex_kernel(const double* __restrict__ in, double* __restrict__ out, long long n, e2e_detector_ex_t det)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    double g = det.base.gain;
    if (det.d_prnu) g = g * __ldg(det.d_prnu + p);
    double mu = g * in[p] + (det.d_dark ? __ldg(det.d_dark + p) : det.base.dark_e);
    if (!(mu > 0.0)) mu = 0.0;
    double z1, e;
    detector_draws(det.base.seed, p, mu, z1, e);
    if (det.full_well_e > 0.0 && e > det.full_well_e) e = det.full_well_e;
    if (!(det.e_per_adu > 0.0)) {
        out[p] = (e + det.base.bias) + det.base.ron_e * z1;
    } else {
        const double v = e + det.base.ron_e * z1;
        double a = floor((v / det.e_per_adu + det.base.bias) + 0.5);
        if (a < 0.0) a = 0.0;
        if (a > det.adu_max) a = det.adu_max;
        out[p] = a;
    }
}

int launch_detector(const double* d_in, double* d_out, long long n, const e2e_detector_t& det, cudaStream_t stream, long long p0)
{
    if (n <= 0) return E2E_OK;
    const int threads = 256;
    long long blocks = (n + threads - 1) / threads;
    detector_kernel<<<(unsigned)blocks, threads, 0, stream>>>(d_in, d_out, n, p0, det);
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "detector_kernel launch");
    return E2E_OK;
}

int launch_detector_ex(const double* d_in, double* d_out, long long n, const e2e_detector_ex_t& det, cudaStream_t stream)
{
    if (n <= 0) return E2E_OK;
    const int threads = 256;
    long long blocks = (n + threads - 1) / threads;
    detector_ex_kernel<<<(unsigned)blocks, threads, 0, stream>>>(d_in, d_out, n, det);
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "detector_ex_kernel launch");
    return E2E_OK;
}

}  // namespace e2e
