"""Closed forms (oracle/theory.py) against the constants the paper prints."""
import math
import os

from oracle import theory

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def consts():
    out = {}
    with open(GOLD) as f:
        for ln in f:
            ln = ln.split("#")[0].split()
            if len(ln) == 2:
                out[ln[0]] = float(ln[1])
    return out


def test_eps_composition_printed_values():
    c = consts()
    assert abs(theory.eps_L(c["eps1"], c["eps2"]) - c["eps_L"]) < 5e-5
    assert abs(theory.eps_H(c["eps1"], c["eps2"]) - c["eps_H"]) < 5e-5
    assert abs(theory.d_total(0.15, 1 / 70) - (1 - 0.85 * (1 - 1 / 70))) < 1e-15


def test_kappa_bound_printed_value():
    c = consts()
    # PAPER.md:839 prints the bound rounded UP to 12.07 (the value is 12.0641)
    assert 0 <= c["kappa_bound_eps0.9"] - theory.kappa_bound_randqr(0.9, 0.9) < 1e-2
    # Assumptions 5.1 hold for the paper's multisketch and (72) follows
    eL, eH = theory.eps_L(0.9, 0.49), theory.eps_H(0.9, 0.49)
    assert 0 <= eL < 616 / 625 - 9 / 625 * eH
    assert theory.kappa_bound_exact(eL, eH) < c["sqrt_ratio_max"]
    assert 90 < theory.kappa_bound_randqr(eL, eH) < 95
    # single sketch limit 616/634: the bound blows up there
    assert abs(616 / 634 - c["eps_single_max"]) < 1e-7
    e = 616 / 634 - 1e-9
    assert theory.kappa_bound_randqr(e, e) > 1e6


def test_orth_bound_is_O_u():
    eL, eH = theory.eps_L(0.9, 0.49), theory.eps_H(0.9, 0.49)
    b = theory.orth_bound_rand_cholqr(10 ** 7, 70, eL, eH)
    assert 0 < b < 1        # (74) is meaningful at the paper's largest problem
    assert b == theory.orth_bound_rand_cholqr(10 ** 7, 70, eL, eH, 2.0 ** -52)


def test_flop_models():
    n, m, p = 10 ** 7, 70, 140
    # with p ~ 2m rand_cholQR ~ 7 n m^2 ; cholQR2 ~ 4 n m^2
    assert abs(theory.flops_rand_cholqr_dense(n, m, p) / (7 * n * m * m) - 1) < 0.01
    assert abs(theory.flops_cholqr2(n, m) / (4 * n * m * m) - 1) < 1e-4
    assert theory.flops_randqr_dense(4, 2, 3) == 3 * 2 * 7 + 2 * 3 * 4 - (2 / 3) * 8 + 16
    # multisketch ~ 3 n m^2 + n m + 2 p2 p1 m
    p1, p2 = 2 * m * m, 2 * m
    f = theory.flops_rand_cholqr_multisketch(n, m, p1, p2)
    assert abs(f / (3 * n * m * m + n * m + 2 * p2 * p1 * m) - 1) < 1e-3
    # CountSketch size, eq. (7): 8.24 (m^2+m) <-> eps = 0.9, d = 0.15
    assert abs(theory.countsketch_rows(70, 0.9, 0.15) / (8.24 * (70 * 70 + 70)) - 1) < 2e-3


def test_printed_speedups_follow_from_tables():
    c = consts()
    assert abs(c["t_cholqr2_1e7_70"] / c["t_multi_1e7_70"] - c["speedup_vs_cholqr2"]) < 5e-3
    assert abs(c["t_scholqr3_1e7_70"] / c["t_multi_1e7_70"] - c["speedup_vs_scholqr3"]) < 5e-3
