"""ctypes/numpy front end of the CPU oracle (oracle/rqr_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares nothing with the
CUDA path in paper_2309_05868_b200/ and never imports it.

Every function is a thin marshalling layer: the arithmetic is in rqr_oracle.c, each C
function citing the PAPER.md passage it follows.  Matrices are C-contiguous float64,
V is m x n (BASELINE.json letters; the paper writes n x m).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rqr_oracle.c")
_LIB = os.path.join(_HERE, "librqr_oracle.so")

ORC_OK = 0
ORC_NOT_SPD = 1000
ORC_SINGULAR = 2000


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP) if needed; returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_num_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


_i64 = ctypes.c_int64
_u64 = ctypes.c_uint64
_u32 = ctypes.c_uint32
_int = ctypes.c_int
_dbl = ctypes.c_double


def num_threads() -> int:
    return int(lib().orc_num_threads())


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def hash_sign(seed, row0, count, s1):
    b = np.zeros(count, dtype=np.uint32)
    s = np.zeros(count, dtype=np.int8)
    lib().orc_hash_sign(_u64(seed), _u64(row0), _i64(count), _u64(s1), _p(b), _p(s))
    return b, s


def countsketch(V, s1, seed, row0=0):
    V = _f64(V)
    m, n = V.shape
    W1 = np.empty((s1, n), dtype=np.float64)
    lib().orc_countsketch(_p(V), _i64(m), _int(n), _i64(n), _i64(s1), _u64(seed), _u64(row0), _p(W1))
    return W1


def gauss_z(seed, stream, first, count):
    z = np.empty(count, dtype=np.float64)
    lib().orc_gauss_z(_u64(seed), _u32(stream), _u64(first), _i64(count), _p(z))
    return z


def gauss_pair_debug(seed, stream, q):
    words = np.zeros(4, dtype=np.uint32)
    u = np.zeros(2, dtype=np.float64)
    z = np.zeros(2, dtype=np.float64)
    lib().orc_gauss_pair_debug(_u64(seed), _u32(stream), _u64(q), _p(words), _p(u), _p(z))
    return words, u, z


def gauss_matrix(seed, s2, s1):
    S2 = np.empty((s2, s1), dtype=np.float64)
    lib().orc_gauss_matrix(_u64(seed), _int(s2), _i64(s1), _p(S2))
    return S2


def gauss_sketch(W1, s2, seed):
    W1 = _f64(W1)
    s1, n = W1.shape
    W = np.empty((s2, n), dtype=np.float64)
    lib().orc_gauss_sketch(_p(W1), _i64(s1), _int(n), _int(s2), _u64(seed), _p(W))
    return W


def rademacher_matrix(seed, s2, s1):
    """N4: dense Rademacher S2, entries +-1/sqrt(s2) from Philox stream 4."""
    S2 = np.empty((s2, s1), dtype=np.float64)
    lib().orc_rademacher_matrix(_u64(seed), _int(s2), _i64(s1), _p(S2))
    return S2


def rademacher_sketch(W1, s2, seed):
    W1 = _f64(W1)
    s1, n = W1.shape
    W = np.empty((s2, n), dtype=np.float64)
    lib().orc_rademacher_sketch(_p(W1), _i64(s1), _int(n), _int(s2), _u64(seed), _p(W))
    return W


def dense_gauss_sketch(V, s, seed, row0=0, m_total=None):
    V = _f64(V)
    m, n = V.shape
    W = np.empty((s, n), dtype=np.float64)
    lib().orc_dense_gauss_sketch(_p(V), _i64(m), _int(n), _i64(n), _int(s), _u64(seed), _u64(row0),
                                 _u64(m if m_total is None else m_total), _p(W))
    return W


def hhqr_r(W):
    """R factor (diag > 0) of the Householder QR of W; returns (R, info)."""
    A = _f64(W).copy()
    rows, n = A.shape
    R = np.empty((n, n), dtype=np.float64)
    info = lib().orc_hhqr(_p(A), _i64(rows), _int(n), _p(R), ctypes.c_void_p(0))
    return R, int(info)


def hhqr_full(V):
    """Brute-force Householder QR with explicit thin Q; returns (Q, R, info)."""
    A = _f64(V).copy()
    rows, n = A.shape
    R = np.empty((n, n), dtype=np.float64)
    Q = np.empty((rows, n), dtype=np.float64)
    info = lib().orc_hhqr(_p(A), _i64(rows), _int(n), _p(R), _p(Q))
    return Q, R, int(info)


def trsm(V, R):
    V = _f64(V)
    R = _f64(R)
    m, n = V.shape
    X = np.empty_like(V)
    lib().orc_trsm(_p(V), _i64(m), _int(n), _i64(n), _p(R), _p(X), _i64(n))
    return X


def gram(A):
    A = _f64(A)
    m, n = A.shape
    G = np.empty((n, n), dtype=np.float64)
    lib().orc_gram(_p(A), _i64(m), _int(n), _i64(n), _p(G))
    return G


def chol(G, shift=0.0):
    G = _f64(G)
    n = G.shape[0]
    R = np.empty((n, n), dtype=np.float64)
    info = lib().orc_chol(_p(G), _int(n), _dbl(shift), _p(R))
    return R, int(info)


def triu_mul(R1, R0):
    R1 = _f64(R1)
    R0 = _f64(R0)
    n = R1.shape[0]
    R = np.empty((n, n), dtype=np.float64)
    lib().orc_triu_mul(_p(R1), _p(R0), _int(n), _p(R))
    return R


def rand_cholqr(V, s1, s2, seed, want_parts=False, rademacher=False):
    """Alg. 3 with Count-Gauss (rademacher=True: Count-Rademacher, N4).  Returns (Q, R, info) or, with
    want_parts, a dict that also holds R0, R1, V1, W1, W."""
    V = _f64(V)
    fn = lib().orc_rand_cholqr_rademacher if rademacher else lib().orc_rand_cholqr
    m, n = V.shape
    Q = np.empty_like(V)
    R = np.zeros((n, n), dtype=np.float64)
    if not want_parts:
        z = ctypes.c_void_p(0)
        info = fn(_p(V), _i64(m), _int(n), _i64(s1), _int(s2), _u64(seed), _p(Q), _p(R), z, z, z, z, z)
        return Q, R, int(info)
    R0 = np.zeros((n, n)); R1 = np.zeros((n, n)); V1 = np.empty_like(V)
    W1 = np.empty((s1, n)); W = np.empty((s2, n))
    info = fn(_p(V), _i64(m), _int(n), _i64(s1), _int(s2), _u64(seed),
              _p(Q), _p(R), _p(R0), _p(R1), _p(V1), _p(W1), _p(W))
    return dict(Q=Q, R=R, R0=R0, R1=R1, V1=V1, W1=W1, W=W, info=int(info))


def gauss_rand_cholqr(V, s, seed):
    V = _f64(V)
    m, n = V.shape
    Q = np.empty_like(V)
    R = np.zeros((n, n), dtype=np.float64)
    info = lib().orc_gauss_rand_cholqr(_p(V), _i64(m), _int(n), _int(s), _u64(seed), _p(Q), _p(R))
    return Q, R, int(info)


def cholqr2(V):
    V = _f64(V)
    m, n = V.shape
    Q = np.empty_like(V)
    R = np.zeros((n, n), dtype=np.float64)
    info = lib().orc_cholqr2(_p(V), _i64(m), _int(n), _p(Q), _p(R))
    return Q, R, int(info)


def scholqr3(V):
    V = _f64(V)
    m, n = V.shape
    Q = np.empty_like(V)
    R = np.zeros((n, n), dtype=np.float64)
    shift = _dbl(0.0)
    info = lib().orc_scholqr3(_p(V), _i64(m), _int(n), _p(Q), _p(R), ctypes.byref(shift))
    return Q, R, int(info), float(shift.value)
