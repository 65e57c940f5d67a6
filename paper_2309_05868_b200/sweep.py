"""C5 sweep (BASELINE.json configs[4]): m in {2^17..2^25} x n in {32, 64, 128}, sigma log-spaced 1 -> 1e-12;
rand_cholQR (Count-Gauss, s1 = 2n^2, s2 = 2n) vs single-Gaussian-sketch rand_cholQR vs CholeskyQR2 vs shifted
CholeskyQR3 and single-CountSketch rand_cholQR on the same kernels, each reported as a fraction of its own FP64/HBM roofline.

  python -m paper_2309_05868_b200.sweep [--n 32 64 128] [--logm 17 25] [--reps 10] [--out sweep.jsonl]

One JSON line per (m, n).  Sketch generation is off the clock.  Peaks: HBM from
MEASURED_PEAKS.json, FP64 from the library's DMMA/DFMA probe measured in this run.  The checks (orthogonality,
residual) use torch float64 library ops on the device, not the library under test.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import torch

from . import bench_probe as probe, binding as rq, flops, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KAPPA = 1e12


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
    return e0.elapsed_time(e1) / reps


def _fp64_peak():
    sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device="cuda")
    best = 0.0
    for kind in (probe.DFMA, probe.DMMA):
        fl = probe.probe_fp64(kind, 20000, 148 * 8, sink)
        ms = _time(lambda: probe.probe_fp64(kind, 20000, 148 * 8, sink), 5)
        best = max(best, fl / (ms * 1e-3) / 1e12)
    return best


def _hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


def _checks(V, Q, R):
    n = V.shape[1]
    eye = torch.eye(n, dtype=torch.float64, device=V.device)
    # Q^T Q by pairwise summation of 2^20-row pieces: a single library GEMM over 2^25 rows has a rounding
    # error of its own (measured 3e-12 on a coherent Q) that would be charged to the factorization
    parts = [Q[i:i + (1 << 20)].T @ Q[i:i + (1 << 20)] for i in range(0, Q.shape[0], 1 << 20)]
    while len(parts) > 1:
        parts = [parts[i] + parts[i + 1] if i + 1 < len(parts) else parts[i] for i in range(0, len(parts), 2)]
    orth = float(torch.linalg.norm(parts[0] - eye))
    num = 0.0
    step = 1 << 21
    for i0 in range(0, V.shape[0], step):
        num += float(torch.linalg.norm(V[i0:i0 + step] - Q[i0:i0 + step] @ R)) ** 2
    return orth, num ** 0.5 / float(torch.linalg.norm(V))


def run_point(m, n, reps, p64, hbm):
    s1, s2 = inputs.sketch_sizes(n)
    seed = inputs.MATRIX_SEED_BASE + 4
    V = (inputs.make_V if m <= (1 << 23) else inputs.make_V_reflectors)(m, n, KAPPA, seed, device="cuda")
    Q = torch.empty_like(V)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, s1, s2)
    info = rq.new_info()
    rq.sketch_prepare(m, n, s1, s2, 42, work)
    out = {"m": m, "n": n, "kappa": KAPPA, "s1": s1, "s2": s2}
    models = {
        "rand_cholqr": (flops.rand_cholqr_flops(m, n, s1, s2), flops.rand_cholqr_bytes(m, n, s1, s2),
                        lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, work, info, 0, rq.FLAG_PREPARED)),
        "gauss_rand_cholqr": (2.0 * m * n * s2 + 3.0 * m * n * n, 32.0 * m * n,
                              lambda: rq.gauss_randcholqr(V, s2, 42, Q, R, work, info)),
        "cholqr2": (flops.cholqr2_flops(m, n), 32.0 * m * n, lambda: rq.cholqr2(V, Q, R, work, info)),
        # one CountSketch, Householder QR of the s1 x n sketch itself (the paper's "Sparse" rows)
        "count_rand_cholqr": (m * n + 2.0 * s1 * n * n - 2.0 * n ** 3 / 3.0 + 3.0 * m * n * n, 32.0 * m * n,
                              lambda: rq.count_randcholqr(V, s1, 42, Q, R, work, info, 0, rq.FLAG_PREPARED)),
        "scholqr3": (6.0 * m * n * n, 48.0 * m * n, lambda: rq.scholqr3(V, Q, R, work, info)),
    }
    for name, (F, B, fn) in models.items():
        ms = _time(fn, reps if name != "gauss_rand_cholqr" else max(1, reps // 5))   # the dense sketch is slow
        st = int(info.item())
        t_roof = max(F / (p64 * 1e12), B / (hbm * 1e9))
        orth, res = _checks(V, Q, R) if st == 0 else (None, None)
        out[name] = {"ms": ms, "gflops": F / ms / 1e6, "gbs": B / ms / 1e6, "roofline_frac": t_roof / (ms * 1e-3),
                     "info": st, "orth_err": orth, "resid": res}
    del V, Q, work
    torch.cuda.empty_cache()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, nargs="+", default=[32, 64, 128])
    ap.add_argument("--logm", type=int, nargs=2, default=[17, 25])
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--out", default=None)
    a = ap.parse_args(argv)
    rq.lib()
    torch.cuda.set_device(0)
    p64 = _fp64_peak()
    hbm, src = _hbm_peak()
    f = open(a.out, "w") if a.out else None
    head = {"fp64_peak_tflops": p64, "hbm_gbs": hbm, "hbm_source": src}
    print(json.dumps(head))
    if f:
        f.write(json.dumps(head) + "\n")
    for n in a.n:
        for lm in range(a.logm[0], a.logm[1] + 1):
            m = 1 << lm
            if 2 * 8 * m * n + rq.workspace_bytes(m, n, *inputs.sketch_sizes(n)) > 150e9:
                continue
            r = run_point(m, n, a.reps if lm < 24 else max(3, a.reps // 3), p64, hbm)
            print(json.dumps(r))
            sys.stdout.flush()
            if f:
                f.write(json.dumps(r) + "\n")
                f.flush()
    if f:
        f.close()


if __name__ == "__main__":
    main()
