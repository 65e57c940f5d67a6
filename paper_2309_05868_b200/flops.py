"""Algorithmic work of one rand_cholQR factorization (BASELINE letters: V is m x n).

Flop model: the paper's with the dense sketching term replaced by the
Count-Gauss terms.  Byte model: SURVEY.md section 8(d) -- what the method
itself must move through HBM: A1 reads V, A4 reads V, A6 reads and writes m x n.
"""


def rand_cholqr_flops(m: int, n: int, s1: int, s2: int) -> float:
    return (m * n                               # CountSketch adds
            + 2.0 * s2 * s1 * n                 # W = S2 W1
            + 2.0 * s2 * n * n - (2.0 / 3.0) * n ** 3   # Householder QR
            + m * n * n                         # V1 = V R0^-1
            + 2.0 * m * n * n                   # cholQR: Gram + solve
            + n ** 3 / 3.0                      # Cholesky
            + n * n * (2.0 * n - 1))            # R = R1 R0


def rand_cholqr_bytes(m: int, n: int, s1: int, s2: int) -> float:
    return 8.0 * (4.0 * m * n + 2.0 * s1 * n + s2 * s1 + 2.0 * s2 * n + 6.0 * n * n)


def cholqr2_flops(m: int, n: int) -> float:
    return 4.0 * m * n * n + n * n * (2.0 * n - 1)


def trsm_gram_flops(m: int, n: int) -> float:
    return 2.0 * m * n * n                               # m n^2 solve + m n^2 symmetric Gram


def step_bytes(m: int, n: int) -> dict:
    return {"countsketch": 8.0 * m * n, "trsm_gram": 8.0 * m * n, "apply": 16.0 * m * n}
