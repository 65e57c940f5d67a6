"""Pins for the oracle's per-step functions against library routines, exact integer cases
and invariants (PAPER.md citations inline)."""
import numpy as np
import pytest
import scipy.linalg as sla

from paper_2309_05868_b200 import inputs


def _np(t):
    return t.numpy()


def test_countsketch_equals_dense_S1_times_V(orc):
    m, n, s1, seed = 3000, 12, 200, 42
    V = _np(inputs.make_V(m, n, 1e4, 1))
    b, s = orc.hash_sign(seed, 0, m, s1)
    S1 = np.zeros((s1, m))
    S1[b, np.arange(m)] = s                       # one +-1 per column
    assert (np.abs(S1).sum(axis=0) == 1).all()
    W1 = orc.countsketch(V, s1, seed)
    ref = S1 @ V
    assert np.abs(W1 - ref).max() <= 1e-14 * np.abs(V).max() * (m / s1) * 4
    # column sums: sum_h W1[h,:] = sum_i sigma_i V[i,:]
    assert np.allclose(W1.sum(axis=0), (s[:, None] * V).sum(axis=0), rtol=0, atol=1e-12)
    # unscaled: ||S1||_F = sqrt(m)
    assert np.isclose(np.linalg.norm(S1), np.sqrt(m))


def test_countsketch_integer_exact_and_row_offset(orc):
    m, n, s1, seed = 5000, 7, 64, 9
    V = _np(inputs.make_integer_V(m, n, 3))
    b, s = orc.hash_sign(seed, 0, m, s1)
    ref = np.zeros((s1, n))
    np.add.at(ref, b, s[:, None] * V)
    W1 = orc.countsketch(V, s1, seed)
    assert np.array_equal(W1, ref)                # exact: order-independent
    # block rows with global row indices sum to the whole (footnote 3)
    Wa = orc.countsketch(V[:1234], s1, seed, row0=0)
    Wb = orc.countsketch(V[1234:], s1, seed, row0=1234)
    assert np.array_equal(Wa + Wb, W1)
    # empty buckets stay zero
    Ws = orc.countsketch(V[:10], 4096, seed)
    assert (np.abs(Ws).sum(axis=1) > 0).sum() <= 10


def test_countsketch_embedding_norm(orc):
    # eq. (3): ||S V||_F within sqrt(1 +- eps) ||V||_F
    V = _np(inputs.make_V(20000, 16, 1e3, 5))
    W1 = orc.countsketch(V, 512, 42)
    r = np.linalg.norm(W1) / np.linalg.norm(V)
    assert 0.7 < r < 1.3


def test_gauss_sketch_equals_numpy_matmul(orc):
    rng = np.random.default_rng(1)
    W1 = rng.standard_normal((700, 9))
    W = orc.gauss_sketch(W1, 20, 42)
    S2 = orc.gauss_matrix(42, 20, 700)
    ref = S2 @ W1
    assert np.abs(W - ref).max() <= 1e-13 * np.abs(ref).max()
    # a transposed operand or wrong stride would fail this non-square case


def test_dense_gauss_sketch_equals_numpy_matmul(orc):
    rng = np.random.default_rng(2)
    V = rng.standard_normal((1000, 6))
    s = 14
    W = orc.dense_gauss_sketch(V, s, 5)
    S = (orc.gauss_z(5, 3, 0, s * 1000) / np.sqrt(s)).reshape(s, 1000)
    assert np.abs(W - S @ V).max() <= 1e-13 * np.abs(W).max()
    # row-sharded halves with global indexing add up
    Wa = orc.dense_gauss_sketch(V[:400], s, 5, row0=0, m_total=1000)
    Wb = orc.dense_gauss_sketch(V[400:], s, 5, row0=400, m_total=1000)
    assert np.abs(Wa + Wb - W).max() <= 1e-13 * np.abs(W).max()


@pytest.mark.parametrize("rows,n", [(32, 16), (128, 64), (50, 7), (9, 9)])
def test_hhqr_r_matches_lapack(orc, rows, n):
    rng = np.random.default_rng(rows + n)
    W = rng.standard_normal((rows, n)) * np.logspace(0, -8, n)
    R, info = orc.hhqr_r(W)
    assert info == 0
    Rl = np.linalg.qr(W, mode="r")
    Rl = Rl * np.sign(np.diag(Rl))[:, None]
    assert np.linalg.norm(R - Rl) <= 1e-13 * np.linalg.norm(Rl)
    assert (np.diag(R) > 0).all()
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R))
    assert np.linalg.norm(R.T @ R - W.T @ W) <= 1e-13 * np.linalg.norm(W) ** 2


def test_hhqr_full_matches_lapack_and_flags_zero_column(orc):
    rng = np.random.default_rng(3)
    V = rng.standard_normal((300, 10))
    Q, R, info = orc.hhqr_full(V)
    assert info == 0
    Ql, Rl = np.linalg.qr(V)
    sg = np.sign(np.diag(Rl))
    assert np.linalg.norm(R - Rl * sg[:, None]) <= 1e-13 * np.linalg.norm(Rl)
    assert np.linalg.norm(Q - Ql * sg[None, :]) <= 1e-12
    assert np.linalg.norm(Q.T @ Q - np.eye(10)) <= 1e-14 * 10
    assert np.linalg.norm(Q @ R - V) <= 1e-14 * np.linalg.norm(V)
    V0 = np.zeros((20, 4)); V0[:, 0] = 1; V0[:, 2] = 2; V0[3, 3] = 1
    _, info = orc.hhqr_r(V0)
    assert info == orc.ORC_SINGULAR + 2


@pytest.mark.parametrize("n,dec", [(16, 0), (64, 6), (33, 12)])
def test_trsm_matches_scipy(orc, n, dec):
    R = _np(inputs.make_upper(n, 4, dec))
    rng = np.random.default_rng(n)
    V = rng.standard_normal((500, n))
    X = orc.trsm(V, R)
    ref = sla.solve_triangular(R, V.T, trans="T", lower=False).T       # x R = v
    assert np.abs(X - ref).max() <= 1e-9 * np.abs(ref).max() if dec else np.allclose(X, ref, rtol=1e-12)
    # row-wise backward stability (eq. (42)): x R = v to O(n u) |x||R|
    resid = np.abs(X @ R - V)
    assert (resid <= 4 * n * 2.0 ** -53 * (np.abs(X) @ np.abs(R)) + 1e-300).all()


def test_trsm_integer_exact(orc):
    # R unit upper triangular with integer entries: substitution is exact
    n = 6
    R = np.triu(np.arange(1, n * n + 1).reshape(n, n) % 5, 1) + np.eye(n)
    X0 = np.arange(1, 4 * n + 1, dtype=np.float64).reshape(4, n) % 7 - 3
    V = X0 @ R
    assert np.array_equal(orc.trsm(V, R), X0)


def test_gram_matches_numpy_and_integer_exact(orc):
    A = _np(inputs.make_V(5000, 24, 1e5, 8))
    G = orc.gram(A)
    ref = A.T @ A
    assert np.linalg.norm(G - ref) <= 1e-14 * np.linalg.norm(ref)
    assert np.array_equal(G, G.T)
    Ai = _np(inputs.make_integer_V(1000, 9, 2))
    assert np.array_equal(orc.gram(Ai), Ai.T @ Ai)
    # ragged block tail (m not a multiple of the 256-row summation block) and m < block
    assert np.array_equal(orc.gram(Ai[:257]), Ai[:257].T @ Ai[:257])
    assert np.array_equal(orc.gram(Ai[:3]), Ai[:3].T @ Ai[:3])


def test_chol_matches_numpy_and_fails_on_indefinite(orc):
    rng = np.random.default_rng(5)
    B = rng.standard_normal((200, 32))
    G = B.T @ B
    R, info = orc.chol(G)
    assert info == 0
    ref = np.linalg.cholesky(G).T
    assert np.linalg.norm(R - ref) <= 1e-13 * np.linalg.norm(ref)
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R)) and (np.diag(R) > 0).all()
    Rs, info = orc.chol(G, shift=2.5)
    assert info == 0 and np.linalg.norm(Rs.T @ Rs - (G + 2.5 * np.eye(32))) <= 1e-13 * np.linalg.norm(G)
    Gbad = G.copy(); Gbad[5, 5] = -1.0
    _, info = orc.chol(Gbad)
    assert info == orc.ORC_NOT_SPD + 6
    Gn = G.copy(); Gn[0, 0] = np.nan
    _, info = orc.chol(Gn)
    assert info == orc.ORC_NOT_SPD + 1
    # exact integer case: G = R^T R with small-integer R
    Ri = np.triu(np.arange(16).reshape(4, 4) % 3 + 1.0)
    R2, info = orc.chol(Ri.T @ Ri)
    assert info == 0 and np.array_equal(R2, Ri)


def test_triu_mul_matches_numpy(orc):
    R1 = _np(inputs.make_upper(20, 1)); R0 = _np(inputs.make_upper(20, 2, 5))
    R = orc.triu_mul(R1, R0)
    assert np.linalg.norm(R - R1 @ R0) <= 1e-15 * np.linalg.norm(R1 @ R0) * 20
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R))
    # order matters: R1 R0, not R0 R1 (Alg. 3 step 3)
    assert np.linalg.norm(R - R0 @ R1) > 1e-3 * np.linalg.norm(R)
