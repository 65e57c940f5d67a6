"""Pins for the oracle's RNG layer: Philox, CountSketch hash/sign, Gaussian entries.
None of these compare the oracle with itself: KATs are published vectors, the worked example
comes from SURVEY.md section 8(c), the rest are distributional facts."""
import os

import numpy as np
import pytest
from scipy import stats

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _lines(name):
    with open(os.path.join(GOLD, name)) as f:
        for ln in f:
            ln = ln.split("#")[0].strip()
            if ln:
                yield ln.split()


def test_philox_known_answers(orc):
    n = 0
    for t in _lines("philox_kat.txt"):
        v = [int(x, 16) for x in t]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]
        n += 1
    assert n == 3


def test_worked_example_seed42(orc):
    seen = 0
    for t in _lines("sketch_seed42.txt"):
        kind = t[0]
        if kind == "words":
            row = int(t[1].split("=")[1])
            out = orc.philox4x32_10([row & 0xFFFFFFFF, row >> 32, 0, 0], [42, 0])
            assert [int(x) for x in out] == [int(x, 16) for x in t[2:6]]
        elif kind == "bucket_sign":
            s1 = int(t[1].split("=")[1]); row = int(t[2].split("=")[1])
            b, s = orc.hash_sign(42, row, 1, s1)
            assert int(b[0]) == int(t[3]) and int(s[0]) == int(t[4])
        elif kind == "gwords":
            q = int(t[1].split("=")[1])
            words, _, _ = orc.gauss_pair_debug(42, 1, q)
            assert [int(x) for x in words] == [int(x, 16) for x in t[2:6]]
        elif kind == "gu":
            q = int(t[1].split("=")[1])
            _, u, _ = orc.gauss_pair_debug(42, 1, q)
            assert u[0] == float(t[2]) and u[1] == float(t[3])      # exactly representable
        elif kind == "gz":
            q = int(t[1].split("=")[1])
            _, _, z = orc.gauss_pair_debug(42, 1, q)
            assert abs(z[0] - float(t[2])) <= 1e-15 * abs(float(t[2]))
            assert abs(z[1] - float(t[3])) <= 1e-15 * abs(float(t[3]))
        elif kind == "gentry":
            S2 = orc.gauss_matrix(42, 32, 512)
            assert abs(S2[0, 0] - float(t[3])) <= 1e-15 * abs(float(t[3]))
            assert abs(S2[0, 1] - float(t[4])) <= 1e-15 * abs(float(t[4]))
        else:
            raise AssertionError(kind)
        seen += 1
    assert seen >= 15


def test_bucket_is_top_bits_for_power_of_two(orc):
    # (x * 2^k) >> 32 == x >> (32 - k): the multiply-shift map reduces to the top bits
    rows = np.arange(1000, dtype=np.uint64)
    b, _ = orc.hash_sign(7, 0, 1000, 1 << 13)
    for i in rows[:50]:
        out = orc.philox4x32_10([int(i), 0, 0, 0], [7, 0])
        assert int(b[int(i)]) == int(out[0]) >> (32 - 13)


def test_bucket_range_and_uniformity(orc):
    for s1 in (512, 700, 8192):
        cnt = 400 * s1 if s1 < 8192 else 100 * s1
        b, s = orc.hash_sign(123, 5, cnt, s1)
        assert b.min() >= 0 and b.max() < s1
        hist = np.bincount(b, minlength=s1)
        chi2 = ((hist - cnt / s1) ** 2 / (cnt / s1)).sum()
        # chi-square with s1-1 dof: mean s1-1, sd sqrt(2(s1-1)); 6 sigma
        assert abs(chi2 - (s1 - 1)) < 6 * np.sqrt(2 * (s1 - 1))
        assert set(np.unique(s)) == {-1, 1}
        assert abs(s.astype(np.float64).mean()) < 6 / np.sqrt(cnt)
        # sign independent of bucket parity
        assert abs(np.corrcoef(s.astype(float), (b & 1).astype(float))[0, 1]) < 6 / np.sqrt(cnt)


def test_hash_depends_on_global_row_index(orc):
    b0, s0 = orc.hash_sign(42, 0, 100, 512)
    b1, s1_ = orc.hash_sign(42, 40, 60, 512)
    assert np.array_equal(b0[40:], b1) and np.array_equal(s0[40:], s1_)
    b2, _ = orc.hash_sign(43, 0, 100, 512)
    assert not np.array_equal(b0, b2)


def test_gaussian_moments_and_ks(orc):
    z = orc.gauss_z(2024, 1, 0, 2_000_000)
    n = z.size
    assert abs(z.mean()) < 5 / np.sqrt(n)
    assert abs(z.var() - 1.0) < 5 * np.sqrt(2.0 / n)
    assert abs(stats.skew(z)) < 5 * np.sqrt(6.0 / n)
    assert abs(stats.kurtosis(z)) < 5 * np.sqrt(24.0 / n)
    # Kolmogorov-Smirnov against the N(0,1) CDF (would fail for a dropped factor 2, a wrong
    # angle range, cos/sin of pi*u instead of 2*pi*u ...)
    assert stats.kstest(z[:200_000], "norm").pvalue > 1e-4
    # even/odd members of a pair are uncorrelated, and so are neighbours
    assert abs(np.corrcoef(z[0::2], z[1::2])[0, 1]) < 5 / np.sqrt(n / 2)
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 5 / np.sqrt(n)
    # streams differ
    z3 = orc.gauss_z(2024, 3, 0, 1000)
    assert not np.allclose(z[:1000], z3)


def test_gaussian_matrix_scaling_and_norm_preservation(orc):
    s2, s1 = 64, 4096
    S2 = orc.gauss_matrix(9, s2, s1)
    # entries N(0, 1/s2)  (PAPER.md:89 S = G / sqrt(p))
    assert abs(S2.var() * s2 - 1.0) < 5 * np.sqrt(2.0 / S2.size)
    z = orc.gauss_z(9, 1, 0, s2 * s1).reshape(s2, s1)
    assert np.allclose(S2 * np.sqrt(s2), z, rtol=1e-15, atol=0)
    # E ||S2 x||^2 = ||x||^2  (eq. (1), in expectation)
    rng = np.random.default_rng(0)
    x = rng.standard_normal((s1, 200))
    ratio = (np.linalg.norm(S2 @ x, axis=0) / np.linalg.norm(x, axis=0)) ** 2
    assert abs(ratio.mean() - 1.0) < 5 * np.sqrt(2.0 / s2) / np.sqrt(200)


def test_gauss_entry_indexing_is_row_major_pairs(orc):
    # entry e = r*s1 + c lives in pair e>>1; an odd s1 makes rows straddle pairs
    s2, s1 = 3, 5
    S2 = orc.gauss_matrix(77, s2, s1)
    flat = orc.gauss_z(77, 1, 0, s2 * s1) / np.sqrt(s2)
    assert np.array_equal(S2.ravel(), flat)
    _, _, z = orc.gauss_pair_debug(77, 1, 3)       # entries 6, 7 = (1,1), (1,2)
    assert S2[1, 1] == z[0] / np.sqrt(3) and S2[1, 2] == z[1] / np.sqrt(3)
