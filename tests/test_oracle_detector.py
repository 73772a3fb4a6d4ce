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


def test_self_specified_log_and_exp_match_libm():
    rng = np.random.default_rng(1)
    for x in np.concatenate([rng.uniform(1e-30, 1.0, 300), rng.uniform(0.5, 2.0, 300), [2.0 ** -104, 1.0 - 2.0 ** -53, 0.7071067811865475, 0.7071067811865476]]):
        assert oracle.olog(float(x)) == pytest.approx(math.log(x), rel=4e-16, abs=2e-16)
    for y in np.concatenate([-rng.uniform(0.0, 64.0, 400), rng.uniform(-1.0, 1.0, 100), [0.0, -63.999999]]):
        assert oracle.oexp(float(y)) == pytest.approx(math.exp(y), rel=5e-16)


@pytest.mark.parametrize("mu,ron", [(0.0, 3.0), (0.7, 0.0), (5.0, 3.0), (40.0, 1.0), (64.0, 0.0), (300.0, 3.0), (4.0e4, 3.0)])
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


def test_poisson_small_mu_exact_pmf():
    """multiplication method: empirical P(n = k) against the Poisson pmf at mu = 2.5 (chi-square, 4 sigma)"""
    n = 400_000
    out = oracle.detector(np.full(n, 2.5), Detector(seed=7))
    ks = np.arange(0, 9)
    pmf = np.array([math.exp(-2.5) * 2.5 ** k / math.factorial(k) for k in ks])
    obs = np.array([(out == k).sum() for k in ks])
    chi2 = np.sum((obs - n * pmf) ** 2 / (n * pmf))
    assert chi2 < 9 + 4 * math.sqrt(18)


def test_independent_of_call_split_and_seed_dependent():
    rng = np.random.default_rng(3)
    frame = rng.uniform(0.0, 200.0, 5000)
    det = Detector(gain=1.3, dark_e=0.2, ron_e=3.0, bias=10.0, seed=5005)
    whole = oracle.detector(frame, det)
    parts = np.concatenate([oracle.detector(frame[:1234], det, 0), oracle.detector(frame[1234:], det, 1234)])
    assert np.array_equal(whole, parts)
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
