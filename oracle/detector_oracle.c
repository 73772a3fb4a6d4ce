/*
 * detector_oracle.c -- CPU oracle for step a6, the detector-noise stage.
 *
 * TEST INFRASTRUCTURE ONLY (see e2e_oracle.c).  P:79: "photon noise and all other specific detector noises
 * (e.g. dark current, RON ...) are added on the final synthetic echellogram".  The paper names the noises
 * only; the algorithm below is the reading SURVEY 8(c) G12 fixes (listed in DESIGN.md), made of IEEE-exact
 * operations (+ - * / sqrt fma, integer ops) only, so that a second implementation can match it bit for bit:
 *
 *   mu   = max(0, gain * frame[p] + dark_e)
 *   (z1, z2) = one Marsaglia-polar pair from the pixel's Philox stream
 *   n    = Poisson(mu):  0 if mu == 0;  Knuth multiplication method if mu < 64 (threshold exp(-mu) from the
 *          self-specified exp below);  else max(0, floor(mu + sqrt(mu) z2 + (z2^2 - 1)/6 + 1/2))
 *   out[p] = (n + bias) + ron_e * z1
 *
 * Random stream of pixel p: Philox4x32-10 (Salmon et al., SC'11), key = (seed_lo, seed_hi),
 * counter = (p_lo, p_hi, block, 0), block = 0, 1, 2, ...; 32-bit words are consumed in order, two per
 * uniform: u = ((hi >> 5) * 2^26 + (lo >> 6) + 1/2) * 2^-53  in (0, 1).
 *
 * Pins (tests/test_oracle_detector.py): Philox known-answer vectors of the Random123 distribution;
 * orc_log / orc_exp against libm to 1e-15; sample mean / variance / skewness of the output at several mu;
 * independence of how the frame is split into calls (pixel_offset).
 */
#include <math.h>
#include <stdint.h>
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

typedef struct { uint32_t key[2]; uint32_t ctr[4]; uint32_t buf[4]; int have; } stream_t;

static void stream_init(stream_t *s, uint64_t seed, uint64_t pixel)
{
    s->key[0] = (uint32_t)seed; s->key[1] = (uint32_t)(seed >> 32);
    s->ctr[0] = (uint32_t)pixel; s->ctr[1] = (uint32_t)(pixel >> 32); s->ctr[2] = 0; s->ctr[3] = 0;
    s->have = 0;
}
static uint32_t stream_word(stream_t *s)
{
    if (s->have == 0) { orc_philox4x32_10(s->ctr, s->key, s->buf); s->ctr[2] += 1; s->have = 4; }
    uint32_t w = s->buf[4 - s->have];
    s->have -= 1;
    return w;
}
static double stream_uniform(stream_t *s)
{
    uint32_t hi = stream_word(s), lo = stream_word(s);
    double a = (double)(hi >> 5), b = (double)(lo >> 6);
    return (a * 67108864.0 + b + 0.5) * (1.0 / 9007199254740992.0);
}

/* self-specified natural log for normal x > 0: x = m 2^e with m in [sqrt(1/2), sqrt(2)),
 * r = (m-1)/(m+1), log x = e ln2 + 2 r (1 + r^2/3 + ... + r^22/23) by fma-Horner */
double orc_log(double x)
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

/* the draws for one pixel: z1 (read noise), n (Poisson count) */
void orc_detector_draws(const orc_detector_t *d, uint64_t pixel, double mu, double *z1_out, double *n_out)
{
    stream_t s;
    stream_init(&s, d->seed, pixel);
    double z1, z2;
    for (;;) {                                                   /* Marsaglia polar */
        double v1 = 2.0 * stream_uniform(&s) - 1.0;
        double v2 = 2.0 * stream_uniform(&s) - 1.0;
        double q = fma(v1, v1, v2 * v2);
        if (q < 1.0 && q > 0.0) {
            double f = sqrt(-2.0 * orc_log(q) / q);
            z1 = v1 * f; z2 = v2 * f;
            break;
        }
    }
    double n;
    if (!(mu > 0.0)) n = 0.0;
    else if (mu < 64.0) {
        double L = orc_exp(-mu), p = stream_uniform(&s);
        n = 0.0;
        while (p > L) { n += 1.0; p = p * stream_uniform(&s); }
    } else {
        double a = sqrt(mu) * z2;
        double b = (z2 * z2 - 1.0) / 6.0;
        n = floor(((mu + a) + b) + 0.5);
        if (n < 0.0) n = 0.0;
    }
    *z1_out = z1; *n_out = n;
}

/* a6 over n pixels; pixel p of this call has global index pixel_offset + p (so results do not depend on
 * how a frame is split into calls).  in may equal out. */
void orc_detector(const double *in, double *out, int64_t n, int64_t pixel_offset, const orc_detector_t *d)
{
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
 * Full detector stage ("photon noise and all other specific detector noises (e.g. dark
 * current, RON ...)").  The paper names the effects only; the reading (G19) is, per pixel p:
 *
 *   mu   = max(0, gain * prnu[p] * frame[p] + dark[p])        prnu = pixel response non-uniformity map (NULL = 1),
 *                                                              dark = dark-current map in e- (NULL = dark_e)
 *   (z1, n) = the same draws as the basic stage (orc_detector_draws: one Philox stream per pixel)
 *   e    = min(n, full_well)            if full_well > 0       (the well saturates before read-out)
 *   e_per_adu <= 0:  out = (e + bias) + ron_e * z1                             (electrons, no quantisation)
 *   e_per_adu  > 0:  out = clamp(floor(((e + ron_e * z1) / e_per_adu + bias) + 1/2), 0, adu_max)   (ADC)
 *
 * With prnu = dark = NULL, full_well = 0, e_per_adu = 0 it IS the basic stage, operation for operation (pinned).
 * Cross-talk between read-out ports couples pixels and is not part of this stage (not built).
 */
typedef struct {
    orc_detector_t base;
    const double *prnu, *dark;       /* [n] maps or NULL */
    double full_well, e_per_adu, adu_max;
} orc_detector_ex_t;

void orc_detector_ex(const double *in, double *out, int64_t n, int64_t pixel_offset, const orc_detector_ex_t *d)
{
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        double g = d->base.gain;
        if (d->prnu) g = g * d->prnu[p];
        double mu = g * in[p] + (d->dark ? d->dark[p] : d->base.dark_e);
        if (!(mu > 0.0)) mu = 0.0;
        double z1, e;
        orc_detector_draws(&d->base, (uint64_t)(pixel_offset + p), mu, &z1, &e);
        if (d->full_well > 0.0 && e > d->full_well) e = d->full_well;
        if (!(d->e_per_adu > 0.0)) {
            out[p] = (e + d->base.bias) + d->base.ron_e * z1;
        } else {
            double v = e + d->base.ron_e * z1;
            double a = floor((v / d->e_per_adu + d->base.bias) + 0.5);
            if (a < 0.0) a = 0.0;
            if (a > d->adu_max) a = d->adu_max;
            out[p] = a;
        }
    }
}
