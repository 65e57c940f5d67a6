"""Pins for the oracle's factorizations against what the paper proves or prints:
Thm 5.3, Thm 5.2 (:697-699), Thm 5.1 (:627-641), Fig. 4 (:903, :913),
uniqueness of the QR factorization with positive diagonal (Alg. 3, :200-206)."""
import numpy as np
import pytest

from oracle import theory
from paper_2309_05868_b200 import inputs

ORTH_TOL = 1e-12      # BASELINE.json north_star
RES_TOL = 1e-13


def _np(t):
    return t.numpy()


def orth_err(Q):
    return np.linalg.norm(Q.T @ Q - np.eye(Q.shape[1]))


def resid(V, Q, R):
    return np.linalg.norm(V - Q @ R) / np.linalg.norm(V)


def check_R(R):
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R))
    assert (np.diag(R) > 0).all()


@pytest.mark.parametrize("kappa", [1e0, 1e3, 1e6, 1e9, 1e12, 1e15])
def test_rand_cholqr_invariants_over_kappa(orc, kappa):
    m, n = 65536, 32
    s1, s2 = inputs.sketch_sizes(n)
    V = _np(inputs.make_V(m, n, kappa, 11))
    out = orc.rand_cholqr(V, s1, s2, 42, want_parts=True)
    assert out["info"] == 0
    Q, R = out["Q"], out["R"]
    assert orth_err(Q) <= ORTH_TOL                     # Thm 5.3 (74): O(u)
    assert resid(V, Q, R) <= RES_TOL                   # Thm 5.3 (75): O(u)||V||
    check_R(R); check_R(out["R0"]); check_R(out["R1"])
    # Thm 5.2: kappa(V1) = O(1); bound (73) with the paper's eps is 92.8; measured ~4-6
    kV1 = np.linalg.cond(out["V1"])
    assert kV1 < 100.0
    # R = R1 R0 (Alg. 3 step 3) and Q R1 = V1 (Alg. 2)
    assert np.linalg.norm(out["R1"] @ out["R0"] - R) <= 1e-14 * np.linalg.norm(R)
    assert np.linalg.norm(Q @ out["R1"] - out["V1"]) <= 1e-14 * np.linalg.norm(out["V1"])
    # W = S2 S1 V (Alg. 1 step 1) against dense library products
    assert np.allclose(out["W"], orc.gauss_matrix(42, s2, s1) @ out["W1"], rtol=0,
                       atol=1e-13 * np.abs(out["W"]).max())


@pytest.mark.parametrize("name", ["C1"])
def test_rand_cholqr_R_matches_householder_on_tiny(orc, name):
    # K7: in exact arithmetic rand_cholQR returns THE thin QR with positive diagonal
    c = inputs.config(name)
    V = _np(inputs.make_config_V(name))
    Q, R, info = orc.rand_cholqr(V, c["s1"], c["s2"], 42)
    assert info == 0
    Rl = np.linalg.qr(V, mode="r")
    Rl = Rl * np.sign(np.diag(Rl))[:, None]
    assert np.linalg.norm(R - Rl) <= 1e-12 * np.linalg.norm(Rl)
    Qh, Rh, info = orc.hhqr_full(V)
    assert info == 0 and np.linalg.norm(R - Rh) <= 1e-12 * np.linalg.norm(Rh)
    assert orth_err(Q) <= ORTH_TOL and resid(V, Q, R) <= RES_TOL
    # different sketch seeds give the same R norm-wise (any embedding works)
    _, R43, _ = orc.rand_cholqr(V, c["s1"], c["s2"], 43)
    assert np.linalg.norm(R - R43) <= 1e-12 * np.linalg.norm(R)


def test_randqr_S_orthogonality_grows_with_kappa(orc):
    # Thm 5.1 (69): ||(S2 S1 V1)^T (S2 S1 V1) - I|| <= 3 delta, delta ~ u kappa(V); and
    # Remark 4.1: S2 S1 V1 = Q_tmp (orthonormal) in exact arithmetic
    m, n = 20000, 16
    s1, s2 = inputs.sketch_sizes(n)
    errs = []
    for kappa in (1e2, 1e6, 1e10):
        V = _np(inputs.make_V(m, n, kappa, 3))
        out = orc.rand_cholqr(V, s1, s2, 42, want_parts=True)
        SV1 = orc.gauss_matrix(42, s2, s1) @ orc.countsketch(out["V1"], s1, 42)
        e = np.linalg.norm(SV1.T @ SV1 - np.eye(n), 2)
        errs.append(e)
        assert e <= 1e-13 * kappa                     # O(u) kappa(V), constant ~1e3 u
        # (67): ||V - V1 R0|| <= (delta/10) sigma_min(V)  =>  O(u) ||V||
        assert np.linalg.norm(V - out["V1"] @ out["R0"]) <= 1e-13 * np.linalg.norm(V)
    assert errs[2] > 100 * errs[0]                    # it really grows with kappa


def test_cholqr2_threshold(orc):
    # Fig. 4: cholQR2's line ends at kappa = 1e8; PAPER.md:23 kappa >~ u^-1/2
    m, n = 65536, 32
    for kappa in (1e0, 1e3, 1e6):
        V = _np(inputs.make_V(m, n, kappa, 21))
        Q, R, info = orc.cholqr2(V)
        assert info == 0 and orth_err(Q) <= ORTH_TOL and resid(V, Q, R) <= RES_TOL
        check_R(R)
    for kappa in (1e10, 1e13):
        V = _np(inputs.make_V(m, n, kappa, 21))
        Q, R, info = orc.cholqr2(V)
        assert info >= orc.ORC_NOT_SPD or orth_err(Q) > 1e3 * ORTH_TOL


def test_scholqr3_threshold(orc):
    # Fig. 4: sCholQR3 works through 1e12 and fails beyond
    m, n = 65536, 32
    for kappa in (1e6, 1e10, 1e12):
        V = _np(inputs.make_V(m, n, kappa, 22))
        Q, R, info, shift = orc.scholqr3(V)
        assert info == 0 and shift > 0
        assert orth_err(Q) <= ORTH_TOL and resid(V, Q, R) <= RES_TOL
        check_R(R)
    V = _np(inputs.make_V(m, n, 1e15, 22))
    Q, R, info, _ = orc.scholqr3(V)
    assert info >= orc.ORC_NOT_SPD or orth_err(Q) > 10 * ORTH_TOL
    # rand_cholQR is fine on the same matrix (the paper's point)
    s1, s2 = inputs.sketch_sizes(n)
    Q, R, info = orc.rand_cholqr(V, s1, s2, 42)
    assert info == 0 and orth_err(Q) <= ORTH_TOL


def test_gauss_rand_cholqr_single_sketch(orc):
    m, n = 8192, 16
    V = _np(inputs.make_V(m, n, 1e12, 31))
    Q, R, info = orc.gauss_rand_cholqr(V, 2 * n, 42)
    assert info == 0 and orth_err(Q) <= ORTH_TOL and resid(V, Q, R) <= RES_TOL
    check_R(R)
    Rl = np.linalg.qr(V, mode="r"); Rl = Rl * np.sign(np.diag(Rl))[:, None]
    assert np.linalg.norm(R - Rl) <= 1e-12 * np.linalg.norm(Rl)


def test_rank_deficient_reports_singular(orc):
    V = np.zeros((1000, 8)); V[:, 0] = 1.0
    _, _, info = orc.rand_cholqr(V, 128, 16, 42)
    assert info >= orc.ORC_SINGULAR


def test_stress_inputs(orc):
    n = 24
    s1, s2 = inputs.sketch_sizes(n)
    for V in (_np(inputs.make_graded_V(30000, n, 14, 5)), _np(inputs.make_vandermonde_V(30000, n))):
        Q, R, info = orc.rand_cholqr(V, s1, s2, 42)
        assert info == 0
        assert resid(V, Q, R) <= RES_TOL
        check_R(R)
    # column-graded input is only badly scaled, not ill-conditioned after scaling: O(u)
    Q, R, _ = orc.rand_cholqr(_np(inputs.make_graded_V(30000, n, 14, 5)), s1, s2, 42)
    assert orth_err(Q) <= ORTH_TOL


def test_H1_recomputed_V1_breaks_orthogonality(orc):
    # K13: cholQR only cleans up the matrix it was GIVEN.  Applying R1^-1 to a V1 that was
    # re-formed with a different rounding (here: via an explicit inverse) loses ~u kappa.
    m, n, kappa = 20000, 16, 1e10
    s1, s2 = inputs.sketch_sizes(n)
    V = _np(inputs.make_V(m, n, kappa, 3))
    out = orc.rand_cholqr(V, s1, s2, 42, want_parts=True)
    good = orth_err(out["Q"])
    V1_other = V @ np.linalg.inv(out["R0"])
    Q_other = orc.trsm(V1_other, out["R1"])
    Q_comb = V @ np.linalg.inv(out["R1"] @ out["R0"])
    assert good <= ORTH_TOL
    assert orth_err(Q_other) > 100 * good
    assert orth_err(Q_comb) > 100 * good
