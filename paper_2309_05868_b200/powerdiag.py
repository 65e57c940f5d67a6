"""Sustained time, energy and SM clock of the m-sized kernels and of the one-shots.

  python -m paper_2309_05868_b200.powerdiag [--m 8388608] [--n 64] [--seconds 1.5]

Every entry point is called back to back for about `seconds`; printed per entry: ms per call (CUDA events), joules per
call and average watts from the board's energy counter (NVML nvmlDeviceGetTotalEnergyConsumption), and the median SM
clock sampled every 10 ms.  A B200 board is capped at 1 kW: a kernel that reaches the cap is clocked down until it fits,
so under sustained load time = energy / 1 kW, and a 10-30-repetition timing understates it.
"""
from __future__ import annotations

import argparse
import json
import threading
import time

import torch

from . import binding as rq, dist as rdist, inputs


def main(argv=None):
    import pynvml
    ap = argparse.ArgumentParser()
    ap.add_argument("--m", type=int, default=1 << 23)
    ap.add_argument("--n", type=int, default=64)
    ap.add_argument("--seconds", type=float, default=1.5)
    a = ap.parse_args(argv)
    rq.lib()
    pynvml.nvmlInit()
    h = pynvml.nvmlDeviceGetHandleByIndex(0)
    m, n = a.m, a.n
    s1, s2 = inputs.sketch_sizes(n)
    V = torch.randn(m, n, dtype=torch.float64, device="cuda")
    Q = torch.empty_like(V)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    b = rdist.alloc_bufs(rq, m, n, s1, s2, "cuda")
    info = b["info"]
    rq.sketch_prepare(m, n, s1, s2, 42, b["work"])
    P = rq.FLAG_PREPARED
    rq.countsketch(V, s1, 42, b["W1"], b["work"], 0, P)
    rq.gauss_sketch(b["W1"], s2, 42, b["W"], b["work"], P)
    rq.small_geqrf(b["W"], b["R0"], info)
    rq.trsm_gram(V, b["R0"], b["G"], Q, b["work"])
    rq.chol(b["G"], b["R1"], info)
    src = torch.empty(1 << 28, dtype=torch.float64, device="cuda") if 16 * m * n < (40 << 30) else None
    dst = torch.empty_like(src) if src is not None else None
    fns = [("A1 countsketch (sorted)", lambda: rq.countsketch(V, s1, 42, b["W1"], b["work"], 0, P)),
           ("A4 trsm_gram, V1 stored", lambda: rq.trsm_gram(V, b["R0"], b["G"], Q, b["work"])),
           ("A6 apply in place", lambda: rq.apply(Q, None, b["R1"], Q, b["work"])),
           ("one-shot rand_cholqr", lambda: rq.rand_cholqr(V, s1, s2, 42, Q, R, b["work"], info, 0, P)),
           ("cholqr2", lambda: rq.cholqr2(V, Q, R, b["work"], info))]
    if n <= 64:
        fns.insert(2, ("A4 trsm_gram, no V1 store", lambda: rq.trsm_gram(V, b["R0"], b["G"], None, b["work"])))
        fns.insert(4, ("A6 apply two-pass", lambda: rq.apply(V, b["R0"], b["R1"], Q, b["work"])))
    if src is not None:
        fns.append(("device copy of 2 GiB (torch)", lambda: dst.copy_(src)))
    out = {"m": m, "n": n, "power_limit_w": pynvml.nvmlDeviceGetEnforcedPowerLimit(h) / 1e3,
           "sm_max_mhz": pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM), "entries": []}
    for name, fn in fns:
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        fn()
        torch.cuda.synchronize()
        reps = max(20, int(a.seconds / max(time.perf_counter() - t0, 1e-5)))
        clk, stop = [], [False]

        def samp():
            while not stop[0]:
                clk.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                time.sleep(0.01)
        th = threading.Thread(target=samp)
        th.start()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        en0 = pynvml.nvmlDeviceGetTotalEnergyConsumption(h)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        en1 = pynvml.nvmlDeviceGetTotalEnergyConsumption(h)
        stop[0] = True
        th.join()
        ms = e0.elapsed_time(e1) / reps
        c = sorted(clk[5:]) or [0]
        out["entries"].append({"name": name, "ms": ms, "reps": reps, "joule_per_call": (en1 - en0) / 1e3 / reps,
                               "watts": (en1 - en0) / (ms * reps), "sm_mhz_median": c[len(c) // 2]})
    print(json.dumps(out))


if __name__ == "__main__":
    main()
