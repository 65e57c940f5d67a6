"""Effect of a larger distortion factor eps (second half; section 6.4, Figs 5-7).

  python -m paper_2309_05868_b200.eps_sweep [--m 100000 1000000 10000000] [--n 10 ... 100] [--reps 5] [--out f.jsonl]

The paper times rand_cholQR with the SMALL sketch a large distortion allows against the LARGE sketch eps = 0.49 needs
and plots the speedup, one panel per sketch family (natural log presumed, reading S17):

  (a) one Gaussian sketch     eps = 0.99: s  = ceil(36.01 log n)      eps = 0.49: s  = ceil(74.3 log n)
  (b) one CountSketch         eps = 0.99: s1 = ceil(6.8 (n^2 + n))    eps = 0.49: s1 = ceil(27.8 (n^2 + n))
  (c) Count-Gauss multisketch eps1 = 0.9: s1 = ceil(8.24 (n^2 + n))   eps1 = 0.49: s1 = ceil(27.8 (n^2 + n)) PAPER.md:919
      with eps2 = 0.49 fixed:  s2 = ceil(74.3 log s1)

(the paper's m is our n, its n our m).  One JSON line per (m, n): seconds, info and ||I - Q^T Q||_F of
both sketch sizes of every family and the speedup large / small, sketch generation off the clock.
Figures 5-7 are images and their values are not in PAPER.md, so there is no paper number beside ours; the claim
under test is qualitative ("a larger eps allows for significant runtime improvements").  A sketch
with more rows than V has (s1 > m at m = 1e5, n >= 60 for the large CountSketch) is not an embedding of anything and
the library rejects it: such points are reported as skipped.
"""
from __future__ import annotations

import argparse
import json
import math
import sys

import torch

from . import binding as rq, inputs

KAPPA = 1e6          # as in paper_grid: the paper does not state the conditioning of its timing matrices


def gauss_size(n: int, eps: float) -> int:
    return math.ceil({0.99: 36.01, 0.49: 74.3}[eps] * math.log(n))


def count_size(n: int, eps: float) -> int:
    return math.ceil({0.99: 6.8, 0.9: 8.24, 0.49: 27.8}[eps] * (n * n + n))


def multi_sizes(n: int, eps1: float) -> tuple[int, int]:
    s1 = count_size(n, eps1)
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


def _measure(fn, reps, Q, info, eye):
    try:
        sec = _time(fn, reps)
    except rq.RqrError as e:                 # a size the library does not take: reported, not hidden
        return {"rejected": str(e)}
    st = int(info.item())
    return {"seconds": sec, "info": st, "orth_err": float(torch.linalg.norm(Q.T @ Q - eye)) if st == 0 else None}


def run_point(m, n, reps, seed=42):
    gen = inputs.make_V if m <= 2_000_000 else inputs.make_V_reflectors
    V = gen(m, n, KAPPA, inputs.MATRIX_SEED_BASE + 6, device="cuda")
    Q = torch.empty_like(V)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    info = rq.new_info()
    eye = torch.eye(n, dtype=torch.float64, device="cuda")
    out = {"m": m, "n": n, "kappa": KAPPA}

    def pair(name, small, large, run):
        rec = {}
        for tag, size in (("small", small), ("large", large)):
            rec[tag] = run(size)
        a, b = rec["small"], rec["large"]
        rec["speedup"] = b["seconds"] / a["seconds"] if "seconds" in a and "seconds" in b else None
        out[name] = rec

    def run_gauss(s):
        if s > m or s > rq.MAX_S2 or s < n:
            return {"s": s, "skipped": "s outside [n, min(m, %d)]" % rq.MAX_S2}
        work = rq.alloc_workspace(m, n, n, s)
        r = _measure(lambda: rq.gauss_randcholqr(V, s, seed, Q, R, work, info), reps, Q, info, eye)
        return {"s": s, **r}

    def run_count(s1):
        if s1 > m:
            return {"s1": s1, "skipped": "s1 > m"}
        work = rq.alloc_workspace(m, n, s1, 2 * n)
        rq.sketch_prepare(m, n, s1, 2 * n, seed, work)
        r = _measure(lambda: rq.count_randcholqr(V, s1, seed, Q, R, work, info, 0, rq.FLAG_PREPARED), reps, Q, info, eye)
        return {"s1": s1, **r}

    def run_multi(ss):
        s1, s2 = ss
        if s1 > m or s2 > rq.MAX_S2:
            return {"s1": s1, "s2": s2, "skipped": "s1 > m" if s1 > m else "s2 > %d" % rq.MAX_S2}
        work = rq.alloc_workspace(m, n, s1, s2)
        rq.sketch_prepare(m, n, s1, s2, seed, work)
        r = _measure(lambda: rq.rand_cholqr(V, s1, s2, seed, Q, R, work, info, 0, rq.FLAG_PREPARED), reps, Q, info, eye)
        return {"s1": s1, "s2": s2, **r}

    pair("gauss", gauss_size(n, 0.99), gauss_size(n, 0.49), run_gauss)
    torch.cuda.empty_cache()
    pair("count", count_size(n, 0.99), count_size(n, 0.49), run_count)
    torch.cuda.empty_cache()
    pair("multi", multi_sizes(n, 0.9), multi_sizes(n, 0.49), run_multi)
    del V, Q
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
