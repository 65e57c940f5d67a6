"""Closed forms printed in the paper, used as oracle-side checks (TEST INFRASTRUCTURE).

Paper letters inside this file: V is n x m (n rows), sketches p1, p2.
Each function cites the equation it restates; tests/test_oracle_theory.py pins them to
the constants the paper prints (PAPER.md:839 "12.07", :883 "0.9490", "1.8310").
"""
import math


def eps_L(e1: float, e2: float) -> float:
    """Proposition 4.1: eps_L = e1 + e2 - e1 e2."""
    return e1 + e2 - e1 * e2


def eps_H(e1: float, e2: float) -> float:
    """Proposition 4.1: eps_H = e1 + e2 + e1 e2."""
    return e1 + e2 + e1 * e2


def d_total(d1: float, d2: float) -> float:
    """d = d1 + d2 - d1 d2, so that 1 - d = (1 - d1)(1 - d2)."""
    return d1 + d2 - d1 * d2


def kappa_bound_randqr(eL: float, eH: float) -> float:
    """Theorem 5.2 eq. (73): kappa(Q0) <= 33 / (25 sqrt((1-eL)/(1+eH)) - 3)."""
    return 33.0 / (25.0 * math.sqrt((1.0 - eL) / (1.0 + eH)) - 3.0)


def kappa_bound_exact(eL: float, eH: float) -> float:
    """Exact-arithmetic bound on kappa(Q0).  The paper prints eq. (13)/(14), PAPER.md:174-180,
    with the factor sqrt((1-eL)/(1+eH)) < 1, which cannot bound a condition number >= 1;
    from (12), the factor is sqrt((1+eH)/(1-eL)) (reading S11)."""
    return math.sqrt((1.0 + eH) / (1.0 - eL))


def orth_bound_rand_cholqr(n_rows: int, m_cols: int, eL: float, eH: float, u: float = 2.0 ** -52) -> float:
    """Theorem 5.3 eq. (74): ||Q^T Q - I||_2 <= 5445/(25 sqrt((1-eL)/(1+eH)) - 3)^2
    (n m + m (m+1)) u   (paper letters: n rows, m columns; u = 2^-52 as in PAPER.md:303)."""
    c = 25.0 * math.sqrt((1.0 - eL) / (1.0 + eH)) - 3.0
    return 5445.0 / (c * c) * (n_rows * m_cols + m_cols * (m_cols + 1)) * u


def countsketch_rows(m_cols: int, eps: float, d: float) -> float:
    """eq. (7): p >= (m^2 + m) / (eps^2 d)."""
    return (m_cols * m_cols + m_cols) / (eps * eps * d)


# ---- flop models, PAPER.md:220-226 (paper letters: n rows, m columns, p sketch rows) ----

def flops_randqr_dense(n_rows: int, m_cols: int, p: int) -> float:
    """p m (2n-1) + 2 p m^2 - (2/3) m^3 + n m^2."""
    return p * m_cols * (2 * n_rows - 1) + 2 * p * m_cols ** 2 - (2.0 / 3.0) * m_cols ** 3 + n_rows * m_cols ** 2


def flops_rand_cholqr_dense(n_rows: int, m_cols: int, p: int) -> float:
    """randQR + 2 n m^2 (cholQR) + m^2 (2m - 1) (matrix mult.)."""
    return flops_randqr_dense(n_rows, m_cols, p) + 2 * n_rows * m_cols ** 2 + m_cols ** 2 * (2 * m_cols - 1)


def flops_cholqr2(n_rows: int, m_cols: int) -> float:
    """2 n m^2 + 2 n m^2 + m^2 (2m - 1)."""
    return 4 * n_rows * m_cols ** 2 + m_cols ** 2 * (2 * m_cols - 1)


def flops_rand_cholqr_multisketch(n_rows: int, m_cols: int, p1: int, p2: int) -> float:
    """Count-Gauss: the dense sketching term p m (2n-1) of PAPER.md:220 is replaced by the
    CountSketch adds n m ("O(nm)") plus the S2 gemm 2 p2 p1 m;
    the rest as in PAPER.md:220-222 with p = p2."""
    hh = 2 * p2 * m_cols ** 2 - (2.0 / 3.0) * m_cols ** 3
    return (n_rows * m_cols + 2.0 * p2 * p1 * m_cols + hh + n_rows * m_cols ** 2
            + 2 * n_rows * m_cols ** 2 + m_cols ** 3 / 3.0 + m_cols ** 2 * (2 * m_cols - 1))
