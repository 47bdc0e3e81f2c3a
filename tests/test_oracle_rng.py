"""Pins for the oracle's random-number layer (SURVEY 8(c) "R", "Pins")."""
from fractions import Fraction

import numpy as np
import pytest
from scipy.special import ndtri
from scipy import stats

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W
from helpers import py_philox, py_draw, read_kat


def test_philox_known_answers():
    for ctr, key, out in read_kat():
        assert list(O.philox4x32_10(ctr, key)) == out
        assert py_philox(ctr, key) == out  # the test-side replay generator is pinned too


def test_philox_matches_independent_python_on_random_counters():
    rng = np.random.default_rng(1)
    for _ in range(200):
        ctr = rng.integers(0, 2**32, 4, dtype=np.uint64)
        key = rng.integers(0, 2**32, 2, dtype=np.uint64)
        assert list(O.philox4x32_10(ctr, key)) == py_philox(ctr, key)


def test_uniforms_are_exact_rationals():
    """DESIGN.md reading R-U: the two-word uniform is (((a<<32|b)>>12) + 1/2) / 2^52, exactly (53 significant bits at
    most), not SURVEY's (>>11, 2^-53) form, whose top value rounds to 1.0."""
    rng = np.random.default_rng(2)
    cases = [(0, 0), (2**32 - 1, 2**32 - 1), (1, 0), (0, 4095), (0, 4096), (0, 2048), (0, 6144), (2**31, 0)]
    cases += [tuple(int(v) for v in rng.integers(0, 2**32, 2, dtype=np.uint64)) for _ in range(200)]
    differs_from_survey_form = 0
    for a, b in cases:
        got = O.u53(a, b)
        assert 0.0 < got < 1.0
        w12 = ((a << 32) | b) >> 12
        assert Fraction(got) == (Fraction(w12) + Fraction(1, 2)) / Fraction(2**52), (a, b)
        survey = (Fraction(((a << 32) | b) >> 11) + Fraction(1, 2)) / Fraction(2**53)
        differs_from_survey_form += Fraction(got) != survey
        exact32 = (Fraction(a) + Fraction(1, 2)) / Fraction(2**32)
        assert Fraction(O.u32(a)) == exact32  # 33 significant bits: exact
    assert differs_from_survey_form > 100          # the two readings are told apart by this test
    assert O.u53(0, 0) == 2.0**-53 and O.u53(2**32 - 1, 2**32 - 1) == 1.0 - 2.0**-53
    assert O.u32(0) == 2.0**-33 and O.u32(2**32 - 1) == 1.0 - 2.0**-33


@pytest.fixture(scope="module")
def orc():
    w = W.make_config(2, scale=1 / 256, particles=False)
    return O.Oracle(w, load=False), w


def test_normal_table_sampler_tracks_inverse_cdf(orc):
    o, w = orc
    rng = np.random.default_rng(3)
    words = rng.integers(0, 2**32, 4000, dtype=np.uint64)
    z = np.array([o.normal(a) for a in words])
    u = (words.astype(np.float64) + 0.5) / 2.0**32
    ref = ndtri(u)
    # piecewise-linear interpolation error h^2/8 * max|d2 ndtri/du2|, h = 1/65536:
    # |z|<1 -> (z/phi^2) <= 17 -> 5e-10; an off-by-one table index is 2e-5..4e-5 there.
    core = np.abs(ref) < 1.0
    assert core.sum() > 2000
    assert np.max(np.abs(z[core] - ref[core])) < 2e-9
    mid = np.abs(ref) < 3.0
    assert np.max(np.abs(z[mid] - ref[mid])) < 1e-5
    # monotone in the word
    ws = np.sort(words)
    zs = np.array([o.normal(a) for a in ws])
    assert np.all(np.diff(zs) >= 0)
    # extreme words stay inside the clamped table
    assert o.normal(0) == pytest.approx(ndtri(2.0**-17), abs=2e-6)
    assert o.normal(2**32 - 1) == pytest.approx(ndtri(1 - 2.0**-17), abs=2e-6)


def test_normal_table_exact_variance():
    # variance of the piecewise-linear inverse CDF: sum over intervals of (a^2+ab+b^2)/(3n);
    # SURVEY 8(c) "Pins" quotes 0.99996617.
    t = W.inv_norm_table()
    a, b = t[:-1], t[1:]
    var = np.sum((a * a + a * b + b * b) / 3.0) / (t.shape[0] - 1)
    assert var == pytest.approx(0.99996617, abs=2e-8)
    assert np.max(np.abs(t)) == pytest.approx(4.325, abs=5e-3)


def test_direction_sampler_is_isotropic(orc):
    o, w = orc
    M = 60000
    n = np.zeros((M, 3))
    fb = 0
    for pid in range(M):
        v, f = o.direction(pid, 5, 4)
        n[pid] = v
        fb += f
    assert fb <= 3  # P(8 rejections) = (1-pi/4)^8 = 4.5e-6 per draw, 0.27 expected in 60000
    norm = np.sqrt((n * n).sum(1))
    assert np.max(np.abs(norm - 1.0)) < 4e-16
    assert np.all(np.abs(n.mean(0)) < 4.0 / np.sqrt(3 * M))
    assert np.all(np.abs((n * n).mean(0) - 1 / 3) < 4 * np.sqrt(4 / 45 / M))
    for k in range(3):  # Archimedes: every coordinate is uniform on (-1, 1)
        assert stats.kstest(n[:, k], "uniform", args=(-1, 2)).pvalue > 1e-3
    # first-attempt acceptance is pi/4: replay attempt 0 with the independent Philox
    acc = 0
    for pid in range(4000):
        wds = py_draw(w.seed, pid, 5, 4)
        p = 2 * (wds[0] + 0.5) / 2**32 - 1
        q = 2 * (wds[1] + 0.5) / 2**32 - 1
        S = p * p + q * q
        if 0 < S < 1:
            acc += 1
            r = np.sqrt(1 - S)
            np.testing.assert_allclose(n[pid], [1 - 2 * S, 2 * p * r, 2 * q * r], rtol=0, atol=1e-15)
    assert abs(acc / 4000 - np.pi / 4) < 4 * np.sqrt(0.785 * 0.215 / 4000)


def test_sigma_lookup_interpolates_and_clamps(orc):
    o, w = orc
    assert o.sigma(0, 37.3) == pytest.approx(1e-19, rel=1e-15)
    assert o.sigma(2, 5e4) == pytest.approx(5e-19, rel=1e-15)
    assert o.sigma(1, 13.0) == 0.0 and o.sigma(1, 13.5) == 0.0
    for E in (14.0, 20.0, 55.5, 400.0):  # table nodes: exactly the Lotz form
        assert o.sigma(1, E) == pytest.approx(4e-18 * np.log(E / 13.6) / (E * 13.6), rel=1e-14)
    E = 100.25  # halfway between nodes 100.0 and 100.5
    lo, hi = o.sigma(1, 100.0), o.sigma(1, 100.5)
    assert o.sigma(1, E) == pytest.approx(0.5 * (lo + hi), rel=1e-14)
    assert o.sigma(1, 1e9) == o.sigma(1, 1000.0)  # clamped above
