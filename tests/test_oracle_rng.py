"""Pins for the oracle's random numbers (pins T6/T7)."""
from pathlib import Path

import numpy as np

import oracle

GOLDEN = Path(__file__).parent / "golden" / "philox4x32_10_kat.txt"


def _kat():
    rows = []
    for line in GOLDEN.read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        w = [int(x, 16) for x in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        got = oracle.philox4x32_10(ctr, key)
        assert [int(x) for x in got] == out


def test_philox_counter_words_are_distinct_streams():
    # each counter word and each key word must matter (a dropped word would alias streams)
    base = oracle.philox4x32_10([1, 2, 3, 0], [1, 0])
    for pos in range(4):
        c = [1, 2, 3, 0]
        c[pos] += 1
        assert not np.array_equal(oracle.philox4x32_10(c, [1, 0]), base)
    assert not np.array_equal(oracle.philox4x32_10([1, 2, 3, 0], [2, 0]), base)
    assert not np.array_equal(oracle.philox4x32_10([1, 2, 3, 0], [1, 1]), base)


def test_uniform_is_x0_of_tag1_mapped_to_open_interval():
    # u = (x0 + 0.5) 2^-32 for counter (walker, k, sweep, 1), key = (seed_lo, seed_hi)
    seed = (7 << 32) | 5
    x = oracle.philox4x32_10([11, 3, 9, 1], [5, 7])
    u = oracle.rng_uniform(seed, 11, 3, 9)
    assert u == (float(x[0]) + 0.5) / 4294967296.0
    assert 0.0 < u < 1.0


def test_gauss3_is_box_muller_of_tag0_words():
    seed = 1
    x = oracle.philox4x32_10([2, 5, 4, 0], [1, 0]).astype(np.float64)
    u = (x + 0.5) / 4294967296.0
    # mpmath-free check with numpy libm: same formula different library -> allow 4 ulp
    chi = oracle.rng_gauss3(seed, 2, 5, 4)
    ref = np.array([np.sqrt(-2 * np.log(u[0])) * np.cos(2 * np.pi * u[1]),
                    np.sqrt(-2 * np.log(u[0])) * np.sin(2 * np.pi * u[1]),
                    np.sqrt(-2 * np.log(u[2])) * np.cos(2 * np.pi * u[3])])
    np.testing.assert_allclose(chi, ref, rtol=1e-14, atol=1e-15)
    # chi_x^2 + chi_y^2 = -2 ln u0 exactly (up to rounding): x and y share one radius
    assert abs(chi[0] ** 2 + chi[1] ** 2 - (-2 * np.log(u[0]))) < 1e-13


def test_gaussian_moments():
    # T7: statistical only.  2e5 triples -> 6e5 samples
    n = 200_000
    out = np.empty((n, 3))
    for i in range(n):
        out[i] = oracle.rng_gauss3(1, i & 0xFFFF, i >> 16, 12345)
    for c in range(3):
        x = out[:, c]
        assert abs(x.mean()) < 5 / np.sqrt(n)
        assert abs(x.var() - 1.0) < 5 * np.sqrt(2.0 / n)
        assert abs((x ** 4).mean() - 3.0) < 5 * np.sqrt(96.0 / n)
    # components uncorrelated
    cc = np.corrcoef(out.T)
    assert np.all(np.abs(cc - np.eye(3)) < 5 / np.sqrt(n))


def test_uniform_moments():
    n = 100_000
    u = np.array([oracle.rng_uniform(1, i & 0xFFF, i >> 12, 7) for i in range(n)])
    assert abs(u.mean() - 0.5) < 5 * np.sqrt(1 / 12 / n)
    assert abs(u.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
    hist, _ = np.histogram(u, bins=10, range=(0, 1))
    assert np.all(np.abs(hist - n / 10) < 5 * np.sqrt(n / 10))
