"""Pins of the oracle's dense Rademacher S2 ("dense Rademacher sketch
matrices in place of dense Gaussian sketches"; reading S21).  CPU only.

What fixes a Rademacher sketch: entries are exactly +-1/sqrt(s2), signs are fair and independent (so
E S^T S = I and E ||S x||^2 = ||x||^2), the bits come from the pinned Philox (known answers in
tests/golden/philox_kat.txt) in the stated order, and the sketch W = S2 W1 is a plain matrix product.
"""
import numpy as np
import pytest

from paper_2309_05868_b200 import inputs


def test_entries_are_plus_minus_inv_sqrt_s2(orc):
    for s2, s1 in [(16, 300), (25, 128), (7, 129)]:
        S = orc.rademacher_matrix(9, s2, s1)
        assert np.array_equal(np.abs(S), np.full((s2, s1), 1.0 / np.sqrt(s2)))
        # every row has squared norm s1 / s2 and every column squared norm 1, exactly up to rounding
        assert np.allclose((S * S).sum(axis=0), 1.0, rtol=0, atol=1e-14)


def test_sign_bits_follow_the_philox_words(orc):
    """Bit (c mod 128) of philox(idx = r * ceil(s1/128) + c div 128, stream 4), word b div 32, bit b mod 32.
    The Philox itself is pinned by the Random123 known answers; here its words are unpacked with numpy's
    unpackbits (little-endian bit order) instead of shifts, for a ragged s1 that is not a multiple of 128."""
    seed, s2, s1 = 42, 5, 300
    S = orc.rademacher_matrix(seed, s2, s1)
    ng = (s1 + 127) // 128
    key = (seed & 0xFFFFFFFF, seed >> 32)
    for r in range(s2):
        bits = []
        for g in range(ng):
            idx = r * ng + g
            o = orc.philox4x32_10((idx & 0xFFFFFFFF, idx >> 32, 4, 0), key)
            words = np.array(o, dtype="<u4")
            bits.append(np.unpackbits(words.view(np.uint8), bitorder="little"))
        bits = np.concatenate(bits)[:s1]
        assert np.array_equal(S[r] < 0, bits.astype(bool))


def test_groups_do_not_repeat_across_rows_or_seeds(orc):
    A = orc.rademacher_matrix(1, 8, 256)
    B = orc.rademacher_matrix(2, 8, 256)
    assert not np.array_equal(A, B)
    # no two rows equal or opposite, no two 128-column groups equal
    for i in range(8):
        for j in range(i + 1, 8):
            assert 0.2 < np.mean(A[i] * A[j] > 0) < 0.8
    assert not np.array_equal(A[:, :128], A[:, 128:])


def test_signs_are_fair_and_pairwise_uncorrelated(orc):
    s2, s1 = 64, 4096
    S = orc.rademacher_matrix(7, s2, s1) * np.sqrt(s2)            # +-1
    N = s2 * s1
    assert abs(S.mean()) <= 4.0 / np.sqrt(N)                       # 4 sigma
    # row-row and column-column correlations: off-diagonal entries of S S^T / s1 are ~ N(0, 1/s1)
    C = S @ S.T / s1
    off = C[~np.eye(s2, dtype=bool)]
    assert np.abs(off).max() <= 5.0 / np.sqrt(s1)
    assert abs(np.mean(off ** 2) * s1 - 1.0) <= 0.15
    D = S.T[:512] @ S.T[:512].T / s2                               # 512 columns
    offd = D[~np.eye(512, dtype=bool)]
    assert abs(np.mean(offd ** 2) * s2 - 1.0) <= 0.05
    # adjacent bits of one Philox word
    assert abs(np.mean(S[:, :-1] * S[:, 1:])) <= 4.0 / np.sqrt(N)


def test_norm_preservation_in_expectation(orc):
    """E ||S x||^2 = ||x||^2 and Var = 2 (||x||^4 - sum x_i^4) / s2 for a Rademacher sketch."""
    rng = np.random.default_rng(0)
    s2, s1 = 32, 512
    x = rng.standard_normal(s1)
    vals = np.array([np.sum((orc.rademacher_matrix(seed, s2, s1) @ x) ** 2) for seed in range(200)])
    nx2 = np.sum(x * x)
    var = 2.0 * (nx2 ** 2 - np.sum(x ** 4)) / s2
    assert abs(vals.mean() - nx2) <= 4.0 * np.sqrt(var / 200)
    assert 0.7 * var <= vals.var() <= 1.3 * var


def test_embeds_a_random_subspace(orc):
    """eq. (1) PAPER.md:55 for S = S2: singular values of S2 U in [sqrt(1-eps), sqrt(1+eps)] with the eps
    a Gaussian sketch of the same size has (s2 = 2 n gives eps well below 0.9; Marchenko-Pastur edge
    (1 +- sqrt(n / s2))^2)."""
    rng = np.random.default_rng(3)
    n, s1 = 16, 2 * 16 * 16
    s2 = 8 * n
    U, _ = np.linalg.qr(rng.standard_normal((s1, n)))
    sv = np.linalg.svd(orc.rademacher_matrix(11, s2, s1) @ U, compute_uv=False)
    edge = np.sqrt(n / s2)
    assert (1 - edge) - 0.1 <= sv.min() and sv.max() <= (1 + edge) + 0.1


def test_rademacher_sketch_equals_numpy_matmul(orc):
    rng = np.random.default_rng(1)
    W1 = rng.standard_normal((700, 9))
    W = orc.rademacher_sketch(W1, 20, 42)
    ref = orc.rademacher_matrix(42, 20, 700) @ W1
    assert np.abs(W - ref).max() <= 1e-13 * np.abs(ref).max()
    # integer data: +-sums are exact, so W sqrt(s2) is an integer matrix
    Wi = orc.rademacher_sketch(np.rint(W1 * 8), 16, 5) * 4.0
    assert np.array_equal(Wi, np.rint(Wi))


@pytest.mark.parametrize("kappa", [1e0, 1e8, 1e12, 1e15])
def test_rand_cholqr_with_rademacher_S2_meets_thm_5_3(orc, kappa):
    """The analysis covers any (eps, d, m) multisketch: the Thm 5.3 bars
    must hold with S2 Rademacher as they do with S2 Gaussian, and R is the R factor of V either way."""
    m, n = 4000, 12
    V = inputs.make_V(m, n, kappa, 5).numpy()
    Q, R, info = orc.rand_cholqr(V, 2 * n * n, 2 * n, 42, rademacher=True)
    assert info == 0
    assert np.linalg.norm(Q.T @ Q - np.eye(n)) <= 1e-13
    assert np.linalg.norm(V - Q @ R) / np.linalg.norm(V) <= 1e-14
    assert np.all(np.diag(R) > 0)
    parts = orc.rand_cholqr(V, 2 * n * n, 2 * n, 42, want_parts=True, rademacher=True)
    assert np.linalg.cond(parts["V1"]) <= 10.0                      # Thm 5.2: kappa(V1) = O(1)
    _, Rg, _ = orc.rand_cholqr(V, 2 * n * n, 2 * n, 42)
    if kappa <= 1e8:
        assert np.linalg.norm(R - Rg) / np.linalg.norm(Rg) <= 1e-6  # same R up to kappa u
    assert not np.array_equal(parts["W"], orc.rand_cholqr(V, 2 * n * n, 2 * n, 42, want_parts=True)["W"])
