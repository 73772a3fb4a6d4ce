/*
 * detector_oracle.c -- CPU oracle for step a6, the detector stage.
 *
 * TEST INFRASTRUCTURE ONLY (see e2e_oracle.c).  P:79: "photon noise and all other specific detector noises
 * (e.g. dark current, RON, pixels non-uniform response and cross-talk) are added on the final synthetic echellogram".
 * The paper names the noises only; the algorithm below is reading G12 of DESIGN.md as re-specified in round 2
 * (G12: a fixed number of Philox blocks and no rejection loop; pixel pairs share the blocks), made of
 * IEEE-exact operations (+ - * / sqrt fma, integer ops) only, so that a second implementation can match it bit for bit:
 *
 *   mu       = max(0, gain * frame[p] + dark_e)
 *   Pixels are keyed in PAIRS (G12 round 3): pixel p belongs to pair q = p >> 1 with parity s = p & 1, and the two pixels of a
 *   pair share each Philox block of the pair's stream -- every block yields two independent variates, one per pixel:
 *   z1       = read-noise normal from block 0 of the pair:  u1 = U(w0, w1), u2 = U(w2, w3),  rho = sqrt(-2 log u1),
 *                z1 = rho cos(2 pi u2) for s = 0,  rho sin(2 pi u2) for s = 1      (the two halves of one Box-Muller pair)
 *   n        = Poisson(mu):  0 if mu == 0;
 *              mu < 64:  inversion by sequential search with ONE uniform of block 1 of the pair, v = U(w0, w1) for s = 0,
 *                        U(w2, w3) for s = 1:
 *                        p = exp(-mu), F = p, n = 0;  while (v > F and n < 255) { n += 1; p = (p mu) (1/n); F += p; }
 *              else      max(0, floor(mu + sqrt(mu) z2 + (z2^2 - 1)/6 + 1/2)) with z2 from block 2 of the pair, formed like z1 from
 *                        block 0 (cos half for s = 0, sin half for s = 1)           (normal + first Cornish-Fisher term:
 *                        mean mu, skewness 1/sqrt(mu) as Poisson, variance mu + 5/36 -- an approximation, 0.2 % high at mu = 64)
 *   out[p]   = (n + bias) + ron_e * z1
 *
 * Random stream of pair q: Philox4x32-10 (Salmon et al., SC'11), key = (seed_lo, seed_hi),
 * counter = (q_lo, q_hi, block, 0); a uniform takes two 32-bit words: U(hi, lo) = ((hi >> 5) * 2^26 + (lo >> 6) + 1/2) * 2^-53
 * in (0, 1).  log, exp, sin and cos are spelled out below (no libm call), every a*b+c that is meant fused is written fma().
 *
 * Pins (tests/test_oracle_detector.py): Philox known-answer vectors of the Random123 distribution; orc_log / orc_exp /
 * orc_sin2pi against libm; which words of which block feed which pixel (libm / scipy restatement); Box-Muller pair: moments,
 * independence of the two pixels of a pair, tail; Poisson pmf (chi-square) at several mu and the mean / variance / third cumulant
 * across both branches; the two pixels of a pair: counts uncorrelated with each other and with the read noise, in both branches;
 * independence of how the frame is split into calls (pixel_offset, even and odd: a pair may straddle two calls);
 * full stage: reductions, (prnu, dark) grid, ADC moments, saturation; cross-talk: matrix form, charge bookkeeping.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { double gain, dark_e, ron_e, bias; uint64_t seed; } orc_detector_t;

void orc_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4])
{
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* block `block` of pixel pair `pair`: 4 words */
static void pair_block(uint64_t seed, uint64_t pair, uint32_t block, uint32_t w[4])
{
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {(uint32_t)pair, (uint32_t)(pair >> 32), block, 0u};
    orc_philox4x32_10(ctr, key, w);
}
static double uniform53(uint32_t hi, uint32_t lo)
{
    double a = (double)(hi >> 5), b = (double)(lo >> 6);
    return (a * 67108864.0 + b + 0.5) * (1.0 / 9007199254740992.0);
}

/* series log for normal x > 0 (round 1's log; now the generator of the table below): x = m 2^e with
 * m in [sqrt(1/2), sqrt(2)), r = (m-1)/(m+1), log x = e ln2 + 2 r (1 + r^2/3 + ... + r^22/23) by fma-Horner */
double orc_log_series(double x)
{
    uint64_t b; memcpy(&b, &x, 8);
    int e = (int)((b >> 52) & 0x7ff) - 1022;
    b = (b & 0x000fffffffffffffULL) | 0x3fe0000000000000ULL;        /* m in [0.5, 1) */
    double m; memcpy(&m, &b, 8);
    if (m < 0.70710678118654752440) { m = m * 2.0; e -= 1; }
    double r = (m - 1.0) / (m + 1.0);
    double r2 = r * r;
    double P = 1.0 / 23.0;
    for (int i = 10; i >= 0; --i) P = fma(P, r2, 1.0 / (double)(2 * i + 1));
    return fma((double)e, 0.693147180559945309417232, (2.0 * r) * P);
}

/* table log (G12 round 2), division-free per call.  With OFF = bits(0x3fe6a09e00000000) (just below sqrt(1/2)):
 *   t = bits(x) - OFF;  k = t >> 52 (arithmetic);  i = (t >> 45) & 127;  z = bits^-1(bits(x) - (k << 52))   in [0.7071, 1.4142)
 * interval i of that range (128 equal steps of the bit pattern) has the midpoint c_i;
 *   INVC[i] = 1 / c_i (IEEE division),  LOGC[i] = -orc_log_series(INVC[i]);
 *   r = fma(z, INVC[i], -1)   (|r| < 2^-8),   log1p(r) = r + r^2 (-1/2 + r/3 - r^2/4 + r^3/5 - r^4/6 + r^5/7)
 *   log x = fma(k, ln2, LOGC[i] + log1p(r)) */
#define LOG_OFF 0x3fe6a09e00000000ULL
static double LOG_INVC[128], LOG_LOGC[128];
static int log_ready = 0;
static void log_init(void)
{
    for (int i = 0; i < 128; ++i) {
        uint64_t lo = LOG_OFF + ((uint64_t)i << 45), hi = lo + ((uint64_t)1 << 45);
        double a, b; memcpy(&a, &lo, 8); memcpy(&b, &hi, 8);
        double c = 0.5 * a + 0.5 * b;                     /* exact: both have at most 20 significant bits here */
        LOG_INVC[i] = 1.0 / c;
        LOG_LOGC[i] = -orc_log_series(LOG_INVC[i]);
    }
    log_ready = 1;
}
double orc_log(double x)
{
    if (!log_ready) log_init();
    uint64_t ix; memcpy(&ix, &x, 8);
    uint64_t t = ix - LOG_OFF;
    int64_t k = (int64_t)t >> 52;
    int i = (int)((t >> 45) & 127);
    uint64_t iz = ix - ((uint64_t)k << 52);
    double z; memcpy(&z, &iz, 8);
    double r = fma(z, LOG_INVC[i], -1.0);
    double P = 1.0 / 7.0;
    P = fma(P, r, -1.0 / 6.0);
    P = fma(P, r, 1.0 / 5.0);
    P = fma(P, r, -1.0 / 4.0);
    P = fma(P, r, 1.0 / 3.0);
    P = fma(P, r, -0.5);
    double y = fma(r * r, P, r);
    return fma((double)k, 0.693147180559945309417232, LOG_LOGC[i] + y);
}

/* self-specified exp for |y| < 700: k = rint(y / ln2), r = y - k ln2 (two-constant), Taylor degree 13, scale by 2^k */
double orc_exp(double y)
{
    double k = rint(y * 1.44269504088896340736);
    double r = fma(-k, 6.93147180369123816490e-01, y);
    r = fma(-k, 1.90821492927058770002e-10, r);
    double c[14];
    c[0] = 1.0;
    for (int i = 1; i <= 13; ++i) c[i] = c[i - 1] / (double)i;
    double P = c[13];
    for (int i = 12; i >= 0; --i) P = fma(P, r, c[i]);
    uint64_t b = (uint64_t)((int64_t)k + 1023) << 52;
    double s; memcpy(&s, &b, 8);
    return P * s;
}

/* sin(2 pi y) for any y in [0, 1.25]: y -= rint(y) -> [-1/2, 1/2]; fold to |y| <= 1/4 (sin(pi - a) = sin a);
 * then the Taylor series of sin(2 pi y) to y^23, coefficients (-1)^n (2 pi)^(2n+1) / (2n+1)!, fma-Horner in y^2 */
double orc_sin2pi(double y)
{
    static const double S[12] = {
        6.283185307179586476925287, -41.34170224039976023396842, 81.60524927607505420339768,
        -76.70585975306138584163064, 42.05869394489765314498681, -15.09464257682299039182662,
        3.819952584848282127733792, -0.7181223017785005122317403, 0.1042291622081398411727104,
        -0.01203158594212062723320257, 0.001130923748251796187770218, -0.00008823533599243005134484484};
    y = y - rint(y);
    if (y > 0.25) y = 0.5 - y;
    if (y < -0.25) y = -0.5 - y;
    double g = y * y;
    double P = S[11];
    for (int i = 10; i >= 0; --i) P = fma(P, g, S[i]);
    return y * P;
}

/* the standard normal of pixel `pixel` from block `block` of its pair: one half of the block's Box-Muller pair */
static double pair_normal(uint64_t seed, uint64_t pixel, uint32_t block)
{
    uint32_t w[4];
    pair_block(seed, pixel >> 1, block, w);
    double u1 = uniform53(w[0], w[1]), u2 = uniform53(w[2], w[3]);
    double rho = sqrt(-2.0 * orc_log(u1));
    return (pixel & 1u) ? rho * orc_sin2pi(u2) : rho * orc_sin2pi(u2 + 0.25);      /* sin half : cos half */
}

/* the draws for one pixel: z1 (read noise), n (Poisson count) */
void orc_detector_draws(const orc_detector_t *d, uint64_t pixel, double mu, double *z1_out, double *n_out)
{
    double z1 = pair_normal(d->seed, pixel, 0u);
    double n;
    if (!(mu > 0.0)) n = 0.0;
    else if (mu < 64.0) {
        uint32_t w[4];
        pair_block(d->seed, pixel >> 1, 1u, w);
        double v = (pixel & 1u) ? uniform53(w[2], w[3]) : uniform53(w[0], w[1]);
        double p = orc_exp(-mu), F = p;
        n = 0.0;
        while (v > F && n < 255.0) {
            n += 1.0;
            p = (p * mu) * (1.0 / n);
            F = F + p;
        }
    } else {
        double z2 = pair_normal(d->seed, pixel, 2u);
        double a = sqrt(mu) * z2;
        double b = (z2 * z2 - 1.0) * (1.0 / 6.0);
        n = floor(((mu + a) + b) + 0.5);
        if (n < 0.0) n = 0.0;
    }
    *z1_out = z1; *n_out = n;
}

/* the read-noise normals of the two pixels of pair `pair` (pins: moments, independence) */
void orc_gaussian_pair(uint64_t seed, uint64_t pair, double *z1, double *z2)
{
    *z1 = pair_normal(seed, 2 * pair, 0u);
    *z2 = pair_normal(seed, 2 * pair + 1, 0u);
}

/* a6 over n pixels; pixel p of this call has global index pixel_offset + p (so results do not depend on
 * how a frame is split into calls).  in may equal out. */
void orc_detector(const double *in, double *out, int64_t n, int64_t pixel_offset, const orc_detector_t *d)
{
    if (!log_ready) log_init();
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        double mu = d->gain * in[p] + d->dark_e;
        if (!(mu > 0.0)) mu = 0.0;
        double z1, cnt;
        orc_detector_draws(d, (uint64_t)(pixel_offset + p), mu, &z1, &cnt);
        out[p] = (cnt + d->bias) + d->ron_e * z1;
    }
}

/*
 * Full detector stage.  The paper names the effects only; the reading (G19, and
 * G20 for the cross-talk) is, per pixel p = j nx + i of an nx x ny frame:
 *
 *   mu   = max(0, gain * prnu[p] * frame[p] + dark[p])        prnu = pixel response non-uniformity map (NULL = 1),
 *                                                              dark = dark-current map in e- (NULL = dark_e)
 *   (z1, n) = the same draws as the basic stage (orc_detector_draws)
 *   e    = min(n, full_well)            if full_well > 0       (the well saturates before read-out)
 *   no cross-talk (xtalk == NULL):
 *     e_per_adu <= 0:  out = (e + bias) + ron_e * z1                             (electrons, no quantisation)
 *     e_per_adu  > 0:  out = clamp(floor(((e + ron_e * z1) / e_per_adu + bias) + 1/2), 0, adu_max)   (ADC)
 *   cross-talk (G20): the detector is read through n_ports ports, port a = columns [a W, (a+1) W), W = nx / n_ports,
 *     all ports clocked together; pixel (j, a W + c) is read at the same instant as pixel (j, b W + c) of every other
 *     port b, and a fraction X[a][b] of port b's video signal v = e + ron_e z1 appears in port a:
 *       s = v_a;  for b = 0 .. n_ports-1, b != a:  s = s + X[a][b] * v_b      (in this order, multiply then add)
 *     e_per_adu <= 0:  out = s + bias;       e_per_adu > 0:  out = clamp(floor((s / e_per_adu + bias) + 1/2), 0, adu_max)
 *
 * With prnu = dark = xtalk = NULL, full_well = 0, e_per_adu = 0 it IS the basic stage, operation for operation (pinned).
 */
typedef struct {
    orc_detector_t base;
    const double *prnu, *dark;       /* [n] maps or NULL */
    double full_well, e_per_adu, adu_max;
    int32_t nx;                      /* row length (cross-talk only) */
    int32_t n_ports;                 /* read-out ports (cross-talk only), nx % n_ports == 0 */
    const double *xtalk;             /* [n_ports][n_ports] or NULL */
} orc_detector_ex_t;

static double ex_signal(const orc_detector_ex_t *d, const double *in, int64_t p, int64_t pixel_offset, double *z1_out)
{
    double g = d->base.gain;
    if (d->prnu) g = g * d->prnu[p];
    double mu = g * in[p] + (d->dark ? d->dark[p] : d->base.dark_e);
    if (!(mu > 0.0)) mu = 0.0;
    double z1, e;
    orc_detector_draws(&d->base, (uint64_t)(pixel_offset + p), mu, &z1, &e);
    if (d->full_well > 0.0 && e > d->full_well) e = d->full_well;
    *z1_out = z1;
    return e;
}

static double ex_adc(const orc_detector_ex_t *d, double v)
{
    double a = floor((v / d->e_per_adu + d->base.bias) + 0.5);
    if (a < 0.0) a = 0.0;
    if (a > d->adu_max) a = d->adu_max;
    return a;
}

/* returns 0, or -1 when cross-talk is asked for with a shape that does not fit (n not whole rows, nx % n_ports != 0,
 * pixel_offset not at a row start) */
int orc_detector_ex(const double *in, double *out, int64_t n, int64_t pixel_offset, const orc_detector_ex_t *d)
{
    if (!log_ready) log_init();
    if (!d->xtalk) {
#pragma omp parallel for schedule(static)
        for (int64_t p = 0; p < n; ++p) {
            double z1;
            double e = ex_signal(d, in, p, pixel_offset, &z1);
            if (!(d->e_per_adu > 0.0)) out[p] = (e + d->base.bias) + d->base.ron_e * z1;
            else out[p] = ex_adc(d, e + d->base.ron_e * z1);
        }
        return 0;
    }
    const int np = d->n_ports;
    if (np < 1 || d->nx < 1 || d->nx % np != 0 || n % d->nx != 0 || pixel_offset % d->nx != 0) return -1;
    const int W = d->nx / np;
    double *v = (double *)malloc((size_t)n * sizeof(double));     /* video signal of every pixel first (in may equal out) */
    if (!v) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        double z1;
        double e = ex_signal(d, in, p, pixel_offset, &z1);
        v[p] = e + d->base.ron_e * z1;
    }
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        int64_t row = p / d->nx;
        int col = (int)(p - row * d->nx), a = col / W, c = col - a * W;
        double s = v[p];
        for (int b = 0; b < np; ++b)
            if (b != a) s = s + d->xtalk[a * np + b] * v[row * d->nx + (int64_t)b * W + c];
        out[p] = (d->e_per_adu > 0.0) ? ex_adc(d, s) : s + d->base.bias;
    }
    free(v);
    return 0;
}
