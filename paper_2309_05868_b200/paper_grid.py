"""The paper's own grid: m = 1e5, 1e6, 1e7 rows, n = 10, 20, ..., 100 columns, with
the paper's "Multi (eps1 = 0.9, eps2 = 0.49)" sketch sizes s1 = ceil(8.24 (n^2 + n)), s2 = ceil(74.3 log s1)
(natural log presumed, reading S17), sketch generation off the clock.

  python -m paper_2309_05868_b200.paper_grid [--m 100000 1000000 10000000] [--reps 5] [--out grid.jsonl]

One JSON line per (m, n): seconds of rand_cholQR, CholeskyQR2 and shifted CholeskyQR3 on one B200 next to the
seconds the paper prints for one A100 (Tables 1-3: "Multi (.9,.49)", "cholQR2", "sCholQR3").
The A100 numbers are context, not a target (another machine, vendor libraries).  Non-power-of-two shapes: ragged
row tiles, padded column blocks and the general bucket map are what this grid exercises.
"""
from __future__ import annotations

import argparse
import json
import math
import sys

import torch

from . import binding as rq, inputs

KAPPA = 1e6          # the paper does not state the conditioning of its timing matrices; CholeskyQR2 must succeed

# seconds printed in the paper's Appendix A for n = 10, 20, ..., 100
PAPER_A100 = {
    100_000: {"rand_cholqr": [.0004, .0006, .0008, .0011, .0014, .0017, .0022, .0025, .0027, .0034],
              "cholqr2": [.0003, .0004, .0006, .0009, .0011, .0013, .0018, .0019, .0021, .0024],
              "scholqr3": [.0005, .0009, .0011, .0014, .0018, .0020, .0028, .0029, .0032, .0037]},
    1_000_000: {"rand_cholqr": [.0021, .0034, .0046, .0069, .0094, .0108, .0147, .0161, .0181, .0208],
                "cholqr2": [.0015, .0031, .0042, .0065, .0087, .0099, .0150, .0161, .0179, .0199],
                "scholqr3": [.0024, .0047, .0068, .0100, .0134, .0152, .0226, .0244, .0270, .0301]},
    10_000_000: {"rand_cholqr": [.0185, .0312, .0427, .0650, .0889, .1019, .1378, .1508, .1706, .1962],
                 "cholqr2": [.0134, .0287, .0396, .0625, .0848, .0964, .1433, .1545, .1724, .1958],
                 "scholqr3": [.0206, .0433, .0598, .0942, .1278, .1453, .2158, .2328, .2603, .2955]},
}


def paper_sketch_sizes(n: int) -> tuple[int, int]:
    s1 = math.ceil(8.24 * (n * n + n))
    return s1, math.ceil(74.3 * math.log(s1))


def _time(fn, reps):
    for _ in range(2):
        fn()
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps * 1e-3


def run_point(m, n, reps):
    s1, s2 = paper_sketch_sizes(n)
    gen = inputs.make_V if m <= 2_000_000 else inputs.make_V_reflectors
    V = gen(m, n, KAPPA, inputs.MATRIX_SEED_BASE + 5, device="cuda")
    Q = torch.empty_like(V)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, s1, s2)
    info = rq.new_info()
    rq.sketch_prepare(m, n, s1, s2, 42, work)
    eye = torch.eye(n, dtype=torch.float64, device="cuda")
    out = {"m": m, "n": n, "s1": s1, "s2": s2, "kappa": KAPPA}
    algs = {"rand_cholqr": lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, work, info, 0, rq.FLAG_PREPARED),
            "cholqr2": lambda: rq.cholqr2(V, Q, R, work, info),
            "scholqr3": lambda: rq.scholqr3(V, Q, R, work, info)}
    j = n // 10 - 1
    for name, fn in algs.items():
        sec = _time(fn, reps)
        st = int(info.item())
        orth = float(torch.linalg.norm(Q.T @ Q - eye)) if st == 0 else None
        paper = PAPER_A100.get(m, {}).get(name)
        out[name] = {"seconds": sec, "info": st, "orth_err": orth,
                     "paper_a100_seconds": paper[j] if paper and 0 <= j < 10 and n % 10 == 0 else None}
    del V, Q, work
    torch.cuda.empty_cache()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--m", type=int, nargs="+", default=[100_000, 1_000_000, 10_000_000])
    ap.add_argument("--n", type=int, nargs="+", default=list(range(10, 101, 10)))
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--out", default=None)
    a = ap.parse_args(argv)
    rq.lib()
    torch.cuda.set_device(0)
    f = open(a.out, "w") if a.out else None
    for m in a.m:
        for n in a.n:
            r = run_point(m, n, a.reps)
            print(json.dumps(r))
            sys.stdout.flush()
            if f:
                f.write(json.dumps(r) + "\n")
                f.flush()
    if f:
        f.close()


if __name__ == "__main__":
    main()
