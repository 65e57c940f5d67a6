"""Per-step timings of the C-ABI entry points at one shape ("per-kernel times alongside").

  python -m paper_2309_05868_b200.stepbench --m 8388608 --n 64 [--reps 10]

Prints one JSON line: CUDA-event time of every step called on its own (A0 sketch generation, A1 in both
CountSketch variants, A2 with the Gaussian and with the on-the-fly Rademacher S2 (N4), A3, A4 with and without R0,
A5, A6 stored / recomputed, A7, the dense Gaussian sketch of B'' and its draw alone, the one-shot with either S2), with the achieved
GB/s or TFLOP/s of the m-sized passes against their algorithmic work.  The input is a
plain Gaussian matrix: timings do not depend on the values.
"""
from __future__ import annotations

import argparse
import json

import torch

from . import binding as rq, inputs


def _time(fn, reps):
    for _ in range(3):
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


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--m", type=int, default=1 << 23)
    ap.add_argument("--n", type=int, default=64)
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--s1", type=int, default=0, help="CountSketch rows (default 2 n^2)")
    ap.add_argument("--s2", type=int, default=0, help="Gaussian sketch rows (default 2 n)")
    a = ap.parse_args(argv)
    m, n, reps = a.m, a.n, a.reps
    s1, s2 = inputs.sketch_sizes(n)
    s1, s2 = (a.s1 or s1), (a.s2 or s2)
    rq.lib()
    torch.cuda.set_device(0)
    f = dict(dtype=torch.float64, device="cuda")
    torch.manual_seed(0)
    V = torch.randn(m, n, **f)
    Q = torch.empty_like(V)
    W1 = torch.empty(s1, n, **f)
    W = torch.empty(s2, n, **f)
    R0 = torch.empty(n, n, **f)
    R1 = torch.empty(n, n, **f)
    R = torch.empty(n, n, **f)
    G = torch.empty(n, n, **f)
    work = rq.alloc_workspace(m, n, s1, s2)
    info = rq.new_info()
    P = rq.FLAG_PREPARED
    out = {"m": m, "n": n, "s1": s1, "s2": s2, "ms": {}}
    t = out["ms"]
    t["A0_sketch_prepare"] = _time(lambda: rq.sketch_prepare(m, n, s1, s2, 42, work), max(2, reps // 3))
    t["A1_countsketch_sorted"] = _time(lambda: rq.countsketch(V, s1, 42, W1, work, rq.VARIANT_SORTED, P), reps)
    t["A1_countsketch_scatter"] = _time(lambda: rq.countsketch(V, s1, 42, W1, work, rq.VARIANT_SCATTER, 0), reps)
    t["A1_countsketch_stream"] = _time(lambda: rq.countsketch(V, s1, 42, W1, work, rq.VARIANT_STREAM, 0), reps)
    rq.countsketch(V, s1, 42, W1, work, rq.VARIANT_SORTED, P)
    t["A2_gauss_sketch"] = _time(lambda: rq.gauss_sketch(W1, s2, 42, W, work, P), reps)
    Wc = W.clone()

    def geqrf():
        W.copy_(Wc)                     # A3 destroys W
        rq.small_geqrf(W, R0, info)
    t_copy = _time(lambda: W.copy_(Wc), reps)
    t["A3_small_geqrf"] = _time(geqrf, reps) - t_copy
    t["A4_trsm_gram_store_V1"] = _time(lambda: rq.trsm_gram(V, R0, G, Q, work), reps)
    if n <= 64:
        t["A4_trsm_gram_no_store"] = _time(lambda: rq.trsm_gram(V, R0, G, None, work), reps)
    t["A4_gram_only"] = _time(lambda: rq.trsm_gram(V, None, G, None, work), reps)
    rq.trsm_gram(V, R0, G, Q, work)
    t["A5_chol"] = _time(lambda: rq.chol(G, R1, info), reps)
    t["A6_apply_in_place"] = _time(lambda: rq.apply(Q, None, R1, Q, work), reps)
    if n <= 64:
        t["A6_apply_recompute_V1"] = _time(lambda: rq.apply(V, R0, R1, Q, work), reps)
    t["A7_triu_mul"] = _time(lambda: rq.triu_mul(R1, R0, R), reps)
    # B'': the single dense Gaussian sketch (s = s2 rows) and the draw of its s x m Gaussians alone
    t["Bpp_dense_gauss_sketch"] = _time(lambda: rq.dense_gauss_sketch(V, s2, 42, W, work), max(1, reps // 3))
    if n % 2 == 0:
        t["Bpp_draw_only"] = _time(lambda: rq.debug_dense_gauss_draw_only(m, n, s2, 42, work), max(1, reps // 3))
    t["Bpp_gauss_randcholqr"] = _time(lambda: rq.gauss_randcholqr(V, s2, 42, Q, R, work, info), max(1, reps // 3))
    # N4: Rademacher S2 generated on the fly (no S2 in the workspace), and the one-shot with either S2
    RAD = rq.S2_RADEMACHER
    t["one_shot_stream_variant"] = _time(lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, work, info, rq.VARIANT_STREAM, P), reps)
    t["one_shot_gauss_S2"] = _time(lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, work, info, 0, P), reps)
    if n <= 64:
        t["one_shot_store_V1"] = _time(lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, work, info, 0, P | rq.FLAG_STORE_V1), reps)
        t["one_shot_recompute_V1"] = _time(lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, work, info, 0, P | rq.FLAG_RECOMPUTE_V1), reps)
        t["cholqr2"] = _time(lambda: rq.cholqr2(V, Q, R, work, info), reps)
    del work
    workr = rq.alloc_workspace(m, n, s1, s2, RAD)
    t["A0_sketch_prepare_rademacher"] = _time(lambda: rq.sketch_prepare(m, n, s1, s2, 42, workr, RAD), max(2, reps // 3))
    t["A2_rademacher_sketch"] = _time(lambda: rq.gauss_sketch(W1, s2, 42, W, workr, P | RAD), reps)
    t["one_shot_rademacher_S2"] = _time(lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, workr, info, RAD, P), reps)
    out["workspace_bytes"] = {"gauss_S2": rq.workspace_bytes(m, n, s1, s2, 0), "rademacher_S2": rq.workspace_bytes(m, n, s1, s2, RAD)}
    mn = float(m) * n
    out["achieved"] = {
        "A1_sorted_GBs": 8.0 * mn / t["A1_countsketch_sorted"] / 1e6,
        "A1_scatter_GBs": 8.0 * mn / t["A1_countsketch_scatter"] / 1e6,
        "A1_stream_GBs": 8.0 * mn / t["A1_countsketch_stream"] / 1e6,
        "A4_TFLOPs": 2.0 * mn * n / t["A4_trsm_gram_store_V1"] / 1e9,
        "A4_GBs": 16.0 * mn / t["A4_trsm_gram_store_V1"] / 1e6,
        "A6_GBs": 16.0 * mn / t["A6_apply_in_place"] / 1e6,
        "A6_TFLOPs": mn * n / t["A6_apply_in_place"] / 1e9,
        "A2_TFLOPs": 2.0 * s2 * s1 * n / t["A2_gauss_sketch"] / 1e9,
        "Bpp_sketch_TFLOPs": 2.0 * mn * s2 / t["Bpp_dense_gauss_sketch"] / 1e9,
    }
    out["info"] = int(info.item())
    print(json.dumps(out))


if __name__ == "__main__":
    main()
