"""Pins for the oracle's detector-noise stage (step a6, pin P12)."""
import math

import numpy as np
import pytest

import oracle
from paper_2008_05858_b200.workloads import Detector


def test_philox_known_answer_vectors():
    """Philox4x32-10 known-answer vectors published with Random123 (Salmon et al., SC'11 reference distribution)"""
    kat = [
        ((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
        ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
        ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0), (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)),
    ]
    for ctr, key, out in kat:
        assert tuple(int(v) for v in oracle.philox4x32_10(ctr, key)) == out


def test_philox_bijection_and_key_sensitivity():
    a = oracle.philox4x32_10((1, 2, 3, 4), (5, 6))
    assert not np.array_equal(a, oracle.philox4x32_10((1, 2, 3, 5), (5, 6)))
    assert not np.array_equal(a, oracle.philox4x32_10((1, 2, 3, 4), (5, 7)))


def test_self_specified_log_exp_sin_match_libm():
    """G12 (round 2): the table log, its generator (the series log), the exp and sin(2 pi y) are spelled out in IEEE
    operations; each must agree with libm to a few ulp over its whole domain of use"""
    rng = np.random.default_rng(1)
    xs = np.concatenate([rng.uniform(1e-30, 1.0, 400), rng.uniform(0.5, 2.0, 400), 1.0 - 2.0 ** -rng.uniform(1, 53, 200),
                         [2.0 ** -54, 2.0 ** -104, 1.0 - 2.0 ** -53, 0.7071067811865475, 0.7071067811865476, 1.0, 0.70710, 1.41421]])
    for x in xs:
        # the table constants come from the series log (4e-16 relative) and add one rounding of their own
        assert oracle.olog(float(x)) == pytest.approx(math.log(x), rel=1e-15, abs=1e-18)
        assert oracle.olog_series(float(x)) == pytest.approx(math.log(x), rel=4e-16, abs=2e-16)
    for y in np.concatenate([-rng.uniform(0.0, 64.0, 400), rng.uniform(-1.0, 1.0, 100), [0.0, -63.999999]]):
        assert oracle.oexp(float(y)) == pytest.approx(math.exp(y), rel=5e-16)
    ys = np.concatenate([rng.uniform(0.0, 1.25, 2000), [0.0, 0.25, 0.5, 0.75, 1.0, 1.25, 2.0 ** -54, 0.125, 0.375]])
    for y in ys:
        want = float(mp_sin2pi(y))
        assert oracle.osin2pi(float(y)) == pytest.approx(want, rel=0.0, abs=3e-16)
    assert oracle.osin2pi(0.5) == 0.0 and oracle.osin2pi(1.0) == 0.0 and oracle.osin2pi(0.0) == 0.0
    assert abs(oracle.osin2pi(0.25) - 1.0) < 2.3e-16 and abs(oracle.osin2pi(0.75) + 1.0) < 2.3e-16


def mp_sin2pi(y):
    import mpmath as mp
    mp.mp.dps = 30
    return mp.sin(2 * mp.pi * mp.mpf(float(y)))


def _uniform53(hi, lo):
    return ((int(hi) >> 5) * 67108864.0 + (int(lo) >> 6) + 0.5) / 9007199254740992.0


def test_draws_follow_the_stated_word_order():
    """which Philox words feed which pixel (G12 rounds 2 + 3), checked with libm in place of the self-specified functions.
    Pixel p = pair q = p >> 1, parity s = p & 1; counter = (q, block).  Block 0 -> u1 = U(w0, w1), u2 = U(w2, w3),
    z1 = sqrt(-2 ln u1) cos(2 pi u2) for s = 0, sin for s = 1; block 1 -> v = U(w0, w1) (s = 0) or U(w2, w3) (s = 1) for the
    Poisson inversion (scipy's Poisson ppf of the same v); mu >= 64 -> z2 from block 2, formed like z1, in the Cornish-Fisher
    formula"""
    from scipy.stats import poisson
    seed = 0x0123_4567_89AB_CDEF
    key = (seed & 0xffffffff, seed >> 32)

    def normal(q, s, block):
        w = oracle.philox4x32_10((q & 0xffffffff, q >> 32, block, 0), key)
        u1, u2 = _uniform53(w[0], w[1]), _uniform53(w[2], w[3])
        rho = math.sqrt(-2.0 * math.log(u1))
        return rho * (math.sin(2 * math.pi * u2) if s else math.cos(2 * math.pi * u2))

    for pixel, mu in [(0, 0.0), (1, 3.3), (77, 20.5), (76, 20.5), (2 ** 33 + 5, 63.5), (2 ** 33 + 4, 63.5), (123456789, 64.0),
                      (123456788, 64.0), (31337, 4.1e4), (5, 0.01), (4, 0.01)]:
        q, par = pixel >> 1, pixel & 1
        det = Detector(gain=1.0, dark_e=0.0, ron_e=1.0, bias=0.0, seed=seed)
        z1 = float(oracle.detector(np.array([0.0]), det, pixel_offset=pixel)[0])        # mu = 0: out = ron z1
        cnt = float(oracle.detector(np.array([mu]), Detector(gain=1.0, ron_e=0.0, seed=seed), pixel_offset=pixel)[0])
        assert z1 == pytest.approx(normal(q, par, 0), abs=1e-14)
        assert float(oracle.detector(np.array([mu]), det, pixel_offset=pixel)[0]) == cnt + z1
        if mu == 0.0:
            assert cnt == 0.0
        elif mu < 64.0:
            w1 = oracle.philox4x32_10((q & 0xffffffff, q >> 32, 1, 0), key)
            v = _uniform53(w1[2], w1[3]) if par else _uniform53(w1[0], w1[1])
            assert cnt == poisson.ppf(v, mu)
        else:
            z2 = normal(q, par, 2)
            assert cnt == max(0.0, math.floor(mu + math.sqrt(mu) * z2 + (z2 * z2 - 1.0) / 6.0 + 0.5))


@pytest.mark.parametrize("mu", [0.4, 12.0, 64.0, 900.0])
def test_the_two_pixels_of_a_pair_are_independent(mu):
    """G12 round 3: the pixels 2q and 2q + 1 share their Philox blocks; each block yields two independent variates, so their
    counts, their read-noise normals and count x partner's read noise must be uncorrelated (4-sigma), in both Poisson
    branches, and each parity alone must have the Poisson mean and variance"""
    n = 400_000
    cnt = oracle.detector(np.full(n, mu), Detector(ron_e=0.0, seed=99))
    z = oracle.detector(np.zeros(n), Detector(ron_e=1.0, seed=99))
    ce, co, ze, zo = cnt[0::2], cnt[1::2], z[0::2], z[1::2]
    se = 4.0 / math.sqrt(n / 2)
    assert abs(np.corrcoef(ce, co)[0, 1]) < se
    assert abs(np.corrcoef(ze, zo)[0, 1]) < se
    assert abs(np.corrcoef(ce, zo)[0, 1]) < se and abs(np.corrcoef(co, ze)[0, 1]) < se
    assert abs(np.corrcoef(ce, ze)[0, 1]) < se and abs(np.corrcoef(co, zo)[0, 1]) < se
    assert abs(np.corrcoef((ce - mu) ** 2, (co - mu) ** 2)[0, 1]) < se                # not just uncorrelated
    var = mu + (5.0 / 36.0 if mu >= 64.0 else 0.0)
    for c in (ce, co):
        assert abs(c.mean() - mu) < 4.0 * math.sqrt(var / (n / 2))
        assert abs(c.var() - var) < 4.0 * var * math.sqrt((2.0 + 1.0 / mu) / (n / 2))


def test_box_muller_pair_is_standard_normal_and_independent():
    # (z1, z2) = the read-noise normals of the two pixels of a pair (the cos and the sin half of one Box-Muller pair)
    n = 200_000
    z1, z2 = oracle.gaussian_pairs(424242, n)
    se = 1.0 / math.sqrt(n)
    for z in (z1, z2):
        assert abs(z.mean()) < 4 * se
        assert abs(z.var() - 1.0) < 4 * math.sqrt(2.0) * se
        assert abs(np.mean(z ** 3)) < 4 * math.sqrt(15.0) * se
        assert abs(np.mean(z ** 4) - 3.0) < 4 * math.sqrt(96.0) * se
        # empirical CDF against Phi (Kolmogorov distance, 4-sigma-like bound 1.95 / sqrt(n) is the 0.1 % point)
        zs = np.sort(z)
        Phi = 0.5 * (1.0 + np.array([math.erf(v / math.sqrt(2.0)) for v in zs[::50]]))
        assert np.max(np.abs(Phi - (np.arange(n)[::50] + 0.5) / n)) < 1.95 * se + 50.0 / n
    assert abs(np.mean(z1 * z2)) < 4 * se
    assert abs(np.mean(z1 ** 2 * z2 ** 2) - 1.0) < 4 * math.sqrt(8.0) * se          # independent, not just uncorrelated
    r2 = z1 ** 2 + z2 ** 2                                                           # chi-square(2): P(r2 > t) = exp(-t/2)
    for tcut in (0.5, 2.0, 6.0, 12.0):
        pt = math.exp(-tcut / 2)
        assert abs((r2 > tcut).mean() - pt) < 4 * math.sqrt(pt * (1 - pt) / n)
    assert 4.0 < np.abs(z1).max() < 8.6                                              # tail reached; |z| <= sqrt(2*54 ln 2) = 8.65


@pytest.mark.parametrize("mu,ron", [(0.0, 3.0), (0.7, 0.0), (5.0, 3.0), (40.0, 1.0), (63.9, 0.0), (64.0, 0.0), (300.0, 3.0), (4.0e4, 3.0)])
def test_noise_moments(mu, ron):
    """mean = mu + bias, variance = mu + ron^2 (+5/36 in the normal branch), Poisson skewness 1/sqrt(mu); 4-sigma bounds"""
    n = 400_000
    det = Detector(gain=1.0, dark_e=0.0, ron_e=ron, bias=100.0, seed=20200813)
    out = oracle.detector(np.full(n, mu), det) - 100.0
    var_expect = mu + ron * ron + (5.0 / 36.0 if mu >= 64.0 else 0.0)
    assert abs(out.mean() - mu) < 4.0 * math.sqrt(max(var_expect, 1e-30) / n) + 1e-12
    if var_expect > 0:
        # var of sample variance ~ (kurtosis-1) var^2 / n ; Poisson+gaussian excess kurtosis <= 1/mu + small
        kurt = 3.0 + (1.0 / mu if mu > 0 else 0.0)
        assert abs(out.var() - var_expect) < 4.0 * var_expect * math.sqrt((kurt - 1.0) / n)
    if ron == 0.0 and mu > 0:
        assert np.all(out == np.round(out)) and out.min() >= 0
        m3 = np.mean((out - out.mean()) ** 3)
        assert m3 == pytest.approx(mu, rel=0.0, abs=6.0 * math.sqrt(15.0 * var_expect ** 3 / n) + 0.02 * mu)   # third cumulant of Poisson = mu
    if mu == 0.0:
        assert out.var() == pytest.approx(ron * ron, rel=0.02)


@pytest.mark.parametrize("mu", [0.05, 2.5, 20.0, 63.5])
def test_poisson_small_mu_exact_pmf(mu):
    """inversion by sequential search: empirical P(n = k) against the Poisson pmf (chi-square over the bins with
    expectation >= 5, 4-sigma bound), and the count is independent of the read-noise draw of the same pixel"""
    n = 400_000
    out = oracle.detector(np.full(n, mu), Detector(seed=7))
    lo, hi = max(0, int(mu - 6 * math.sqrt(mu) - 2)), int(mu + 6 * math.sqrt(mu) + 6)
    ks = np.arange(lo, hi)
    pmf = np.array([math.exp(-mu + k * math.log(mu) - math.lgamma(k + 1)) for k in ks])
    keep = n * pmf >= 5.0
    obs = np.array([(out == k).sum() for k in ks])
    assert obs.sum() >= n - 50
    chi2 = np.sum((obs[keep] - n * pmf[keep]) ** 2 / (n * pmf[keep]))
    dof = int(keep.sum())
    assert chi2 < dof + 4 * math.sqrt(2 * dof)
    z = oracle.detector(np.zeros(n), Detector(ron_e=1.0, seed=7))                 # z1 of the same pixels
    assert abs(np.corrcoef(out, z)[0, 1]) < 4 / math.sqrt(n)


def test_independent_of_call_split_and_seed_dependent():
    rng = np.random.default_rng(3)
    frame = rng.uniform(0.0, 200.0, 5000)
    det = Detector(gain=1.3, dark_e=0.2, ron_e=3.0, bias=10.0, seed=5005)
    whole = oracle.detector(frame, det)
    for cut in (1234, 1235, 1):                                   # an odd cut puts the two pixels of a pair into different calls
        parts = np.concatenate([oracle.detector(frame[:cut], det, 0), oracle.detector(frame[cut:], det, cut)])
        assert np.array_equal(whole, parts)
    assert np.array_equal(oracle.detector(frame, det, 777)[1:], oracle.detector(frame[1:], det, 778))
    assert not np.array_equal(whole, oracle.detector(frame, Detector(gain=1.3, dark_e=0.2, ron_e=3.0, bias=10.0, seed=5006)))
    # negative flux is clamped: mu = 0 -> pure read noise around the bias
    neg = oracle.detector(np.full(20000, -5.0), Detector(ron_e=2.0, bias=0.0, seed=1))
    assert abs(neg.mean()) < 0.1 and neg.std() == pytest.approx(2.0, rel=0.05)


# ------------------------------------------------------------------------------------------ full detector stage (8(f) 2)
def test_detector_ex_reduces_to_the_basic_stage_bit_for_bit():
    """no maps, no well, no ADC: the extended stage is the (pinned) basic stage, operation for operation"""
    rng = np.random.default_rng(4)
    frame = np.concatenate([rng.uniform(0.0, 120.0, 4000), rng.uniform(0.0, 5.0e4, 4000), [-3.0, 0.0]])
    det = Detector(gain=0.9, dark_e=0.3, ron_e=2.5, bias=50.0, seed=99)
    assert np.array_equal(oracle.detector_ex(frame, det), oracle.detector(frame, det))
    # unit PRNU map and constant dark map = the scalars
    assert np.array_equal(oracle.detector_ex(frame, det, prnu=np.ones_like(frame), dark=np.full_like(frame, 0.3)),
                          oracle.detector(frame, det))


def test_detector_ex_prnu_and_dark_maps_drive_the_poisson_mean():
    """per-pixel mean electrons = gain prnu F + dark: checked column by column of a (prnu, dark) grid, 4 sigma"""
    n = 200_000
    prnu_v, dark_v = [0.0, 0.5, 1.1], [0.0, 7.0]
    F, gain = 200.0, 0.8
    for pr in prnu_v:
        for dk in dark_v:
            out = oracle.detector_ex(np.full(n, F), Detector(gain=gain, dark_e=123.0, ron_e=0.0, bias=0.0, seed=31),
                                     prnu=np.full(n, pr), dark=np.full(n, dk))
            mu = gain * pr * F + dk
            assert np.all(out == np.round(out))
            assert abs(out.mean() - mu) < 4.0 * math.sqrt(max(mu + 5.0 / 36.0, 1e-30) / n) + 1e-12
            if mu == 0.0:
                assert np.all(out == 0.0)


def test_detector_ex_full_well_and_adc():
    n = 100_000
    det = Detector(gain=1.0, dark_e=0.0, ron_e=3.0, bias=100.0, seed=8)
    # ADC: integers in [0, adu_max]; mean = mu / e_per_adu + bias; variance = (mu + ron^2)/e_per_adu^2 + 1/12 (rounding)
    mu, epa = 5000.0, 1.7
    out = oracle.detector_ex(np.full(n, mu), det, e_per_adu=epa, adu_max=65535.0)
    assert np.all(out == np.round(out)) and out.min() >= 0 and out.max() <= 65535
    var = (mu + 5.0 / 36.0 + 9.0) / epa ** 2 + 1.0 / 12.0
    assert abs(out.mean() - (mu / epa + 100.0)) < 4.0 * math.sqrt(var / n)
    assert out.var() == pytest.approx(var, rel=4.0 * math.sqrt(2.0 / n) + 1e-3)
    # quantisation is round-half-up of the unquantised value: reconstruct it from the electrons-valued output
    e_out = oracle.detector_ex(np.full(n, mu), Detector(gain=1.0, ron_e=3.0, bias=0.0, seed=8))
    assert np.array_equal(out, np.clip(np.floor((e_out / epa + 100.0) + 0.5), 0.0, 65535.0))
    # ADC saturation: everything far above adu_max reads adu_max, far below zero reads 0
    assert np.all(oracle.detector_ex(np.full(1000, 1.0e6), det, e_per_adu=1.0, adu_max=65535.0) == 65535.0)
    neg = Detector(gain=1.0, ron_e=3.0, bias=-1000.0, seed=8)
    assert np.all(oracle.detector_ex(np.full(1000, 10.0), neg, e_per_adu=1.0) == 0.0)
    # full well: electrons clipped BEFORE read-out, so with ron = 0 nothing exceeds the well and a bright pixel sits on it
    nr = Detector(gain=1.0, ron_e=0.0, bias=0.0, seed=8)
    sat = oracle.detector_ex(np.concatenate([np.full(1000, 9.0e4), np.full(1000, 100.0)]), nr, full_well=6.0e4)
    assert np.all(sat[:1000] == 6.0e4) and sat[1000:].max() < 200.0
    assert np.array_equal(sat[1000:], oracle.detector(np.concatenate([np.full(1000, 9.0e4), np.full(1000, 100.0)]), nr)[1000:])
    # with read noise the saturated pixels scatter around the well with sigma = ron (noise added after the clip)
    satn = oracle.detector_ex(np.full(50_000, 9.0e4), Detector(ron_e=3.0, seed=8), full_well=6.0e4) - 6.0e4
    assert abs(satn.mean()) < 0.1 and satn.std() == pytest.approx(3.0, rel=0.03)


def test_cross_talk_is_the_port_coupling_matrix():
    """G20: with the electrons-valued video signal v of the no-cross-talk stage (bias 0), the cross-talk output is
    v + (X with its diagonal removed) applied across the ports at equal in-port column -- one matrix product per row;
    X = NULL is the basic stage bit for bit; total signal: sum(out) = sum_b (1 + sum_{a != b} X[a][b]) V_b"""
    rng = np.random.default_rng(9)
    ny, nx, npo = 6, 64, 4
    frame = rng.uniform(0.0, 5.0e4, (ny, nx))
    frame[2, 10:14] = 0.0
    det = Detector(gain=1.0, dark_e=0.2, ron_e=3.0, bias=0.0, seed=4242)
    X = rng.uniform(-2e-4, 1e-3, (npo, npo))
    v = oracle.detector_ex(frame, det)                                            # = (e + 0) + ron z1
    out = oracle.detector_ex(frame, det, xtalk=X)
    Xo = X - np.diag(np.diag(X))
    vp = v.reshape(ny, npo, nx // npo)                                            # [row][port][column in port]
    want = (vp + np.einsum("ab,rbc->rac", Xo, vp)).reshape(ny, nx)
    assert np.allclose(out, want, rtol=1e-15, atol=0.0)
    assert not np.allclose(out, v, rtol=1e-6)
    Vb = vp.sum(axis=(0, 2))
    assert out.sum() == pytest.approx(float(((1.0 + Xo.sum(axis=0)) * Vb).sum()), rel=1e-13)
    # a single bright column in port 1 shows up at the same in-port column of ports 0, 2, 3, scaled by X[a][1]
    f2 = np.zeros((2, nx)); f2[:, 16 + 5] = 4.0e4
    nr = Detector(gain=1.0, ron_e=0.0, seed=1)
    o2 = oracle.detector_ex(f2, nr, xtalk=X)
    e = o2[:, 16 + 5]
    for a in (0, 2, 3):
        assert np.array_equal(o2[:, 16 * a + 5], 0.0 + X[a, 1] * e)
        assert np.all(np.delete(o2[:, 16 * a:16 * a + 16], 5, axis=1) == 0.0)
    # bias and ADC come after the mixing; well clipping before it
    b = Detector(gain=1.0, dark_e=0.2, ron_e=3.0, bias=300.0, seed=4242)
    assert np.allclose(oracle.detector_ex(frame, b, xtalk=X), want + 300.0, rtol=1e-15)
    adc = oracle.detector_ex(frame, b, xtalk=X, e_per_adu=1.7, adu_max=65535.0)
    assert np.array_equal(adc, np.clip(np.floor((out / 1.7 + 300.0) + 0.5), 0.0, 65535.0))
    assert np.array_equal(oracle.detector_ex(frame, b, xtalk=np.zeros((npo, npo))), v + 300.0)
    with pytest.raises(ValueError):
        oracle.detector_ex(frame[:, :63], det, xtalk=X)
    # uint16 output = the ADC branch cast
    a16 = oracle.detector_adu16(frame, b, xtalk=X, e_per_adu=1.7, adu_max=65535.0)
    assert a16.dtype == np.uint16 and np.array_equal(a16.astype(np.float64), adc)


def test_detector_ex_independent_of_call_split():
    rng = np.random.default_rng(5)
    frame = rng.uniform(0.0, 3.0e4, 3000)
    prnu, dark = rng.normal(1.0, 0.02, 3000), rng.uniform(0.0, 2.0, 3000)
    det = Detector(gain=1.0, ron_e=3.0, bias=300.0, seed=77)
    kw = dict(full_well=2.5e4, e_per_adu=0.9, adu_max=65535.0)
    whole = oracle.detector_ex(frame, det, prnu=prnu, dark=dark, **kw)
    parts = np.concatenate([oracle.detector_ex(frame[:700], det, prnu=prnu[:700], dark=dark[:700], pixel_offset=0, **kw),
                            oracle.detector_ex(frame[700:], det, prnu=prnu[700:], dark=dark[700:], pixel_offset=700, **kw)])
    assert np.array_equal(whole, parts)
