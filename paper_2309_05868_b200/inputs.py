"""Seeded synthetic inputs, shared by the CUDA path's tests/bench and by the CPU oracle's tests.

This module holds NONE of the method's arithmetic (no sketch, no hash, no triangular solve,
no Gram, no Cholesky): it only builds test matrices with plain torch float64 library ops, so
that both sides see identical bits.  It imports neither the CUDA binding nor oracle/.

Recipe ("V := L Sigma R^T using random orthogonal
matrices L, R and a diagonal Sigma with log-equispaced entries"; BASELINE.json configs):
  V = U diag(sigma) W^T,  U (m x n) and W (n x n) Haar (Q factor of the Householder QR of an
  i.i.d. Gaussian, sign-fixed so that diag(R) > 0),  sigma_j = kappa^(-j/(n-1)), j = 0..n-1
  (BASELINE: "log-spaced from 1 to 1/kappa"; a pure rescaling of the paper's
  [kappa^-1/2, kappa^1/2]).
"""
from __future__ import annotations

import torch

# BASELINE.json `configs`.  s1 = 2 n^2, s2 = 2 n.
CONFIGS = {
    "C1": dict(m=20_000, n=16, kappa=1e10),
    "C2": dict(m=1 << 20, n=64, kappa=1e6),
    "C3": dict(m=1 << 23, n=64, kappa=1e12),
    "C4": dict(m=1 << 21, n=256, kappa=1e14),
}
MATRIX_SEED_BASE = 1234
SKETCH_SEEDS = (42, 43, 44)


def sketch_sizes(n: int) -> tuple[int, int]:
    """BASELINE.json: CountSketch s1 = 2 n^2, Gaussian s2 = 2 n."""
    return 2 * n * n, 2 * n


def config(name: str) -> dict:
    c = dict(CONFIGS[name])
    c["s1"], c["s2"] = sketch_sizes(c["n"])
    c["seed"] = MATRIX_SEED_BASE + list(CONFIGS).index(name)
    return c


def _haar(rows: int, cols: int, gen: torch.Generator, device) -> torch.Tensor:
    a = torch.randn(rows, cols, generator=gen, dtype=torch.float64, device=device)
    q, r = torch.linalg.qr(a, mode="reduced")
    d = torch.sign(torch.diagonal(r))
    d = torch.where(d == 0, torch.ones_like(d), d)
    return q * d


def singular_values(n: int, kappa: float, device="cpu") -> torch.Tensor:
    j = torch.arange(n, dtype=torch.float64, device=device)
    if n == 1:
        return torch.ones(1, dtype=torch.float64, device=device)
    return torch.pow(torch.tensor(float(kappa), dtype=torch.float64, device=device), -j / (n - 1))


def make_V(m: int, n: int, kappa: float, seed: int, device="cpu") -> torch.Tensor:
    """m x n float64, row-major contiguous, singular values kappa^(-j/(n-1))."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    U = _haar(m, n, gen, device)
    W = _haar(n, n, gen, device)
    sig = singular_values(n, kappa, device)
    V = (U * sig) @ W.T
    return V.contiguous()


def make_config_V(name: str, device="cpu") -> torch.Tensor:
    c = config(name)
    return make_V(c["m"], c["n"], c["kappa"], c["seed"], device)


def make_integer_V(m: int, n: int, seed: int, lo: int = -8, hi: int = 8, device="cpu") -> torch.Tensor:
    """Small integers: every partial sum of a CountSketch or Gram is exact in float64, so the
    result is independent of summation order (exactness pin K4)."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    return torch.randint(lo, hi + 1, (m, n), generator=gen, device=device).to(torch.float64).contiguous()


def make_graded_V(m: int, n: int, decades: float, seed: int, device="cpu") -> torch.Tensor:
    """Column-graded stress input: Gaussian columns scaled by 10^(-j*decades/(n-1))."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    a = torch.randn(m, n, generator=gen, dtype=torch.float64, device=device)
    j = torch.arange(n, dtype=torch.float64, device=device)
    return (a * torch.pow(torch.tensor(10.0, dtype=torch.float64, device=device),
                          -j * decades / max(n - 1, 1))).contiguous()


def make_vandermonde_V(m: int, n: int, device="cpu") -> torch.Tensor:
    """Numerically rank-deficient stress input: V[i, j] = x_i^j, x equispaced in [0, 1]."""
    x = torch.linspace(0.0, 1.0, m, dtype=torch.float64, device=device)
    j = torch.arange(n, dtype=torch.float64, device=device)
    return torch.pow(x[:, None], j[None, :]).contiguous()


def make_upper(n: int, seed: int, cond_decades: float = 0.0, device="cpu") -> torch.Tensor:
    """Random upper-triangular n x n with positive, optionally graded, diagonal."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    a = torch.randn(n, n, generator=gen, dtype=torch.float64, device=device) / (n ** 0.5)
    r = torch.triu(a, diagonal=1)
    j = torch.arange(n, dtype=torch.float64, device=device)
    d = (1.0 + torch.rand(n, generator=gen, dtype=torch.float64, device=device)) * torch.pow(
        torch.tensor(10.0, dtype=torch.float64, device=device), -j * cond_decades / max(n - 1, 1))
    return (r + torch.diag(d)).contiguous()


def make_V_reflectors(m: int, n: int, kappa: float, seed: int, device="cpu", k: int = 4) -> torch.Tensor:
    """Same recipe with a cheaper orthonormal U for the largest sweep points (2^24, 2^25 rows), where a
    library QR of an m x n Gaussian needs more workspace than the matrix: U = H_1 ... H_k D E with
    E = sqrt(n/m) [I_n; I_n; ...] (stacked identities: orthonormal columns, all rows of equal norm, like a
    Haar U), D random signs, and k random Householder reflectors (Gaussian vectors): orthonormal to rounding
    by construction ("Haar-like"); W Haar as in make_V.  O(k m n) work, in place.
    (If n does not divide m the columns of E have counts that differ by one and are normalised one by one.)"""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    sgn = torch.randint(0, 2, (m,), generator=gen, device=device).to(torch.float64) * 2.0 - 1.0
    U = torch.zeros(m, n, dtype=torch.float64, device=device)
    idx = torch.arange(m, device=device)
    col = idx % n
    cnt = torch.bincount(col, minlength=n).to(torch.float64)
    U[idx, col] = sgn / torch.sqrt(cnt[col])
    del idx, sgn, col, cnt
    for _ in range(k):
        v = torch.randn(m, generator=gen, dtype=torch.float64, device=device)
        v /= torch.linalg.norm(v)
        w = v @ U                                   # n
        U.addr_(v, w, alpha=-2.0)                   # U -= 2 v (v^T U)
    W = _haar(n, n, gen, device)
    sig = singular_values(n, kappa, device)
    U *= sig
    V = U @ W.T
    del U
    return V.contiguous()


def make_coherent_V(m: int, n: int, kappa: float, seed: int, device="cpu", k: int = 4) -> torch.Tensor:
    """Stress input: same singular values, but U = H_1 ... H_k [I_n; 0]: the first n rows carry almost all of
    the mass (maximal coherence).  Hard for a CountSketch (heavy rows may share a bucket) and for long
    floating-point accumulations (the sums reach their final size in the first row-block)."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    U = torch.zeros(m, n, dtype=torch.float64, device=device)
    U[:n] = torch.eye(n, dtype=torch.float64, device=device)
    for _ in range(k):
        v = torch.randn(m, generator=gen, dtype=torch.float64, device=device)
        v /= torch.linalg.norm(v)
        U.addr_(v, v @ U, alpha=-2.0)
    W = _haar(n, n, gen, device)
    U *= singular_values(n, kappa, device)
    V = U @ W.T
    del U
    return V.contiguous()
