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
