#!/usr/bin/env python
"""bench.py -- rand_cholQR (Count-Gauss) FP64 throughput on B200, one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl ours|reference]

A "step" is one whole factorization (all SURVEY.md 8(a) rows A1..A7) of one synthetic matrix
V = U diag(sigma) W^T of the named workload (default C3, 2^23 x 64: the m >= 2^22 target configuration and the
largest n = 64 configuration of BASELINE.json).  Sketch generation A0 is OFF the clock, the paper's convention
(PAPER.md:883); `ms_with_sketch_gen` reports the time including it.
`value` = algorithmic GFLOP/s (paper_2309_05868_b200/flops.py) with V resident in HBM, from the MEDIAN of the K
per-step CUDA-event times of the timed region (median of >= 20 repetitions; the mean is beside it);
`e2e` = the same through host buffers (every step uploads its V from pinned host memory and reads Q and R back
inside the timed region; steps double-buffered over three streams, the one-stream serial figure beside it).
`roofline` = the dominant kernel (A4), `roofline.per_step` = every m-sized kernel against its own roof.
N > 1: the rows are sharded over ranks (PAPER.md:228 footnote 3), weak scaling.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_ncu_traffic.csv")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--seed", type=int, default=42)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the other configurations and the sweep points")
    ap.add_argument("--v1", default="auto", choices=["auto", "store", "recompute"],
                    help="V1 = V R0^-1 stored in A4 or recomputed in A6 (auto: the library chooses per n)")
    ap.add_argument("--no-probe", action="store_true", help="skip the FP64 peak probe (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="time direct calls instead of CUDA-graph replays")
    ap.add_argument("--force-sharded", action="store_true",
                    help="run the row-sharded N > 1 code path even at one rank (self-test of that path)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed regions run."""

    def __init__(self, index=0, period=0.02):
        super().__init__(daemon=True)
        self.period = period
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml_unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


def launches_per_step(n, m=0, s1=0):
    """Kernels of ours launched by one rqr_rand_cholqr with a prepared sketch (sorted variant):
    countsketch 1 (+ 1 partial reduction when the bucket lists are split, 2 s1 <= 1184), Gaussian GEMM + reduce 2,
    Householder 1, A4 2 (n <= 64: fused kernel + partial reduce) or 4 (n > 64: fragment build, panel substitution,
    syrk, reduce), Cholesky 1 (the product R = R1 R0 is fused into it for n <= 128; a separate launch above),
    A6 1 (n > 64: + fragment build).  Stored or recomputed V1: the same count."""
    split = 1 if (s1 and 2 * s1 <= 1184) else 0
    if n <= 64:
        return 8 + split + max(0, -(-m // (1 << 23)) - 1)          # one more A4 launch per further 2^23-row chunk
    return (11 if n <= 128 else 12) + max(0, -(-m // (1 << 21)) - 1)   # the syrk runs per 2^21-row chunk


def load_traffic(workload, kernel_prefix):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel from the committed ncu --set full summary
    (profiles/r2_ncu_traffic.csv: workload,kernel,dram_read_bytes,dram_write_bytes,source)."""
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    tot, src = 0.0, None
    with open(TRAFFIC_CSV) as f:
        for row in csv.DictReader(r for r in f if not r.startswith("#")):
            if row["workload"] == workload and row["kernel"].startswith(kernel_prefix):
                tot += float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
                src = row["source"]
    return (tot, src) if src else (None, None)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d.get("hbm_gbs"), "bf16_tflops": d.get("bf16_tflops"),
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained"), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def config_dict(args, c, name, v1_mode):
    m, n = c["m"], c["n"]
    return {"workload": name, "m": m, "n": n, "kappa": c["kappa"], "s1": c["s1"], "s2": c["s2"],
            "l2": "inputs_exceed_L2" if 8 * m * n > 126e6 else "L2_resident_not_flushed",
            "sketch_generation": "off_the_clock (PAPER.md:883)",
            "launch": "direct calls" if args.no_graph else "CUDA-graph replay of one rqr_rand_cholqr call",
            "v1": v1_mode}


def v1_mode_of(args, n):
    if args.v1 != "auto":
        return args.v1 + "d" if args.v1 == "store" else "recomputed"
    return "recomputed (auto, n <= 24)" if n <= 24 else "stored (auto, n > 24)"


# ------------------------------------------------------------------------------------------
ORACLE_SAMPLE_ROWS = 1 << 22      # bounds the CPU leg: a few seconds of oracle work per call at n = 64


def oracle_sample(V_host, n, seed):
    """Times the CPU oracle, as it stands, on a bounded sample (the first rows) of the workload."""
    from oracle import rqr_oracle as orc
    from paper_2309_05868_b200 import flops, inputs
    orc.build()
    ms = V_host.shape[0]
    s1, s2 = inputs.sketch_sizes(n)
    t0 = time.perf_counter()
    Q, R, info = orc.rand_cholqr(V_host, s1, s2, seed)
    dt = time.perf_counter() - t0
    fl = flops.rand_cholqr_flops(ms, n, s1, s2)
    return {"value": fl / dt / 1e9, "unit": "GFLOP/s", "cores": orc.num_threads(), "kind": "oracle",
            "sample": "one whole factorization of the first %d rows of the workload (x %d cols, s1=%d s2=%d), "
                      "%.2f s wall, info=%d" % (ms, n, s1, s2, dt, info)}, dt


def run_reference(args):
    """--impl reference: the oracle on the host cores, on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2309_05868_b200 import inputs
    c = inputs.config(args.workload)
    n = c["n"]
    ms = min(c["m"], ORACLE_SAMPLE_ROWS)
    V = inputs.make_V(ms, n, c["kappa"], c["seed"]).numpy()
    oracle_sample(V, n, args.seed)                       # one warm-up (library build, page faults)
    vals, dts = [], []
    r = None
    for _ in range(max(1, min(args.steps, 5))):
        r, dt = oracle_sample(V, n, args.seed)
        vals.append(r["value"]); dts.append(dt)
    r["value"] = sum(vals) / len(vals)
    r["sample"] += "; %d timed repetitions of that sample per run" % len(vals)
    line = {"impl": "reference", "metric": "rand_cholQR FP64 GFLOP/s", "value": r["value"], "unit": "GFLOP/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(dts) / len(dts),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(args, c, args.workload, v1_mode_of(args, n)),
            "cpu_baseline": r,
            "e2e": {"value": r["value"], "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    _emit(line)


# ------------------------------------------------------------------------------------------
def time_region(torch, fn, steps):
    """CUDA-event time (ms) of `steps` calls of fn on the current stream, synchronised both sides."""
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def time_steps(torch, fn, steps, barrier=None):
    """One timed region of exactly `steps` calls on the current stream (synchronised, and a barrier over the ranks,
    on both sides) with an event after every call: returns (total ms, per-step ms list)."""
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    if barrier:
        barrier()
    torch.cuda.synchronize()
    ev[0].record()
    for i in range(steps):
        fn()
        ev[i + 1].record()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    return ev[0].elapsed_time(ev[steps]), [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]


def median(v):
    s = sorted(v)
    k = len(s)
    return s[k // 2] if k % 2 else 0.5 * (s[k // 2 - 1] + s[k // 2])


def gpu_energy_mj(index=0):
    """Total energy counter of the board (NVML, millijoules) or None."""
    try:
        import pynvml
        pynvml.nvmlInit()
        return pynvml.nvmlDeviceGetTotalEnergyConsumption(pynvml.nvmlDeviceGetHandleByIndex(index))
    except Exception:
        return None


def probe_hbm_sustained(torch, seconds=1.0):
    """Sustained device copy bandwidth (GB/s, read + write bytes) over >= `seconds` of back-to-back copies of 2 GiB:
    what the HBM delivers once the board sits at its power cap (MEASURED_PEAKS.json holds the burst figure)."""
    a = torch.empty(1 << 28, dtype=torch.float64, device="cuda")
    b = torch.empty_like(a)
    b.copy_(a)
    ms1 = time_region(torch, lambda: b.copy_(a), 3) / 3
    reps = max(3, int(seconds * 1e3 / ms1))
    ms = time_region(torch, lambda: b.copy_(a), reps) / reps
    del a, b
    torch.cuda.empty_cache()
    return 2.0 * (1 << 28) * 8 / ms / 1e6


def probe_fp64_peak(torch):
    """Measured FP64 peak (TFLOP/s): best of a DFMA chain and a DMMA chain, >= 0.25 s each."""
    from paper_2309_05868_b200 import bench_probe as probe
    sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device="cuda")
    out = {}
    for kind, name in ((probe.DFMA, "dfma"), (probe.DMMA, "dmma"), (probe.MIX, "dfma_dmma_mixed")):
        iters = 20000
        fl = probe.probe_fp64(kind, iters, 148 * 8, sink)        # warm-up
        ms = time_region(torch, lambda: probe.probe_fp64(kind, iters, 148 * 8, sink), 1)
        reps = max(1, int(250.0 / max(ms, 1e-3)))
        ms = time_region(torch, lambda: probe.probe_fp64(kind, iters, 148 * 8, sink), reps)
        out[name] = fl * reps / (ms * 1e-3) / 1e12
    return out


def breakdown(torch, rq, Vd, c, seed, Q, R, bufs, steps, recompute, row0=0):
    """Per-step CUDA-event times (medians over `steps` runs) of the sequence the one-shot runs, called as the
    separate step entry points (the one-shot itself fuses A7 into A5)."""
    names = ["countsketch", "gauss_sketch", "small_geqrf", "trsm_gram", "chol", "apply", "triu_mul"]
    acc = {k: [] for k in names}
    s1, s2 = c["s1"], c["s2"]
    P = rq.FLAG_PREPARED
    for _ in range(steps):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(len(names) + 1)]
        ev[0].record()
        rq.countsketch(Vd, s1, seed, bufs["W1"], bufs["work"], 0, P, row0); ev[1].record()
        rq.gauss_sketch(bufs["W1"], s2, seed, bufs["W"], bufs["work"], P); ev[2].record()
        rq.small_geqrf(bufs["W"], bufs["R0"], bufs["info"]); ev[3].record()
        rq.trsm_gram(Vd, bufs["R0"], bufs["G"], None if recompute else Q, bufs["work"]); ev[4].record()
        rq.chol(bufs["G"], bufs["R1"], bufs["info"]); ev[5].record()
        if recompute:
            rq.apply(Vd, bufs["R0"], bufs["R1"], Q, bufs["work"])
        else:
            rq.apply(Q, None, bufs["R1"], Q, bufs["work"])
        ev[6].record()
        rq.triu_mul(bufs["R1"], bufs["R0"], R); ev[7].record()
        torch.cuda.synchronize()
        for i, k in enumerate(names):
            acc[k].append(ev[i].elapsed_time(ev[i + 1]))
    return {k: median(v) for k, v in acc.items()}      # medians: robust against a host hiccup


def per_step_roofline(bd, m, n, p64, hbm, recompute, workload):
    """Every m-sized kernel against its own roof (algorithmic work per launch): A1 reads V
    (8mn bytes); A4 does 2mn^2 flops (n^2 substitution + n^2 symmetric Gram per row) on 16mn bytes (8mn when V1 is
    not stored); A6 moves 16mn bytes and does mn^2 flops (2mn^2 executed when V1 is recomputed, mn^2 credited)."""
    mn = float(m) * n
    rows = []

    def entry(step, kernel, t_ms, bytes_, flops_):
        t = t_ms * 1e-3
        hb = {"achieved": bytes_ / t / 1e9, "peak": hbm, "unit": "GB/s", "frac": bytes_ / t / 1e9 / hbm}
        e = {"step": step, "kernel": kernel, "ms": t_ms, "algorithmic_bytes": bytes_, "algorithmic_flops": flops_}
        if flops_ / (p64 * 1e12) > bytes_ / (hbm * 1e9):
            tn = {"achieved": flops_ / t / 1e12, "peak": p64, "unit": "TFLOP/s", "frac": flops_ / t / 1e12 / p64}
            e.update({"bound": "tensor", **tn, "hbm": hb})
        else:
            e.update({"bound": "hbm", **hb})
            if flops_ > mn:
                e["tensor"] = {"achieved": flops_ / t / 1e12, "peak": p64, "unit": "TFLOP/s",
                               "frac": flops_ / t / 1e12 / p64}
        tr, src = load_traffic(workload, kernel)
        e["traffic"] = tr
        if src:
            e["traffic_source"] = src
        return e
    rows.append(entry("A1", "rqr_countsketch", bd["countsketch"], 8.0 * mn, mn))
    rows.append(entry("A4", "rqr_trsm_gram", bd["trsm_gram"], (8.0 if recompute else 16.0) * mn, 2.0 * mn * n))
    rows.append(entry("A6", "rqr_apply", bd["apply"], 16.0 * mn, mn * n))
    return rows


def make_step(torch, rq, rdist, Vd, c, seed, Q, R, bufs, flags, shard):
    """The timed call: one rqr_rand_cholqr, or (sharded) one row-sharded factorization of this rank's rows."""
    s1, s2 = c["s1"], c["s2"]
    if shard is None:
        return lambda: rq.rand_cholqr(Vd, s1, s2, seed, Q, R, bufs["work"], bufs["info"], 0, flags)
    world, rank, row0 = shard
    return lambda: rdist.rand_cholqr_sharded(rq, Vd, row0, s1, s2, seed, Q, R, bufs, None, flags, 0,
                                             m_total=Vd.shape[0] * world)


def run_config(torch, rq, name, args, peaks, p64, want_e2e=True, want_breakdown=True, steps=None, shard=None,
               shape=None, want_comparators=False):
    """Measures one workload.  shard = (world, rank, row0): this rank's block rows of the row-sharded job (weak
    scaling: `m` rows per rank); timings are then the max over ranks.  shape = (m, n, kappa): a sweep point."""
    from paper_2309_05868_b200 import dist as rdist, flops, inputs
    steps = steps or args.steps
    if shape is None:
        c = inputs.config(name)
    else:
        c = {"m": shape[0], "n": shape[1], "kappa": shape[2], "seed": inputs.MATRIX_SEED_BASE + 4}
        c["s1"], c["s2"] = inputs.sketch_sizes(shape[1])
    m, n, s1, s2 = c["m"], c["n"], c["s1"], c["s2"]
    seed = args.seed
    world, rank, row0 = shard if shard else (1, 0, 0)
    barrier = None
    if shard is not None:
        import torch.distributed as dist
        barrier = dist.barrier if dist.is_initialized() and world > 1 else None
    Vd = inputs.make_V(m, n, c["kappa"], c["seed"] + 1000 * rank, device="cuda")
    Q = torch.empty_like(Vd)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    bufs = rdist.alloc_bufs(rq, m, n, s1, s2, "cuda")
    work, info = bufs["work"], bufs["info"]
    v1f = {"auto": 0, "store": rq.FLAG_STORE_V1, "recompute": rq.FLAG_RECOMPUTE_V1}[args.v1]
    recompute = (n <= 64) and (args.v1 == "recompute" or (args.v1 == "auto" and n <= 24))
    flags = rq.FLAG_PREPARED | v1f

    def prep():
        rq.sketch_prepare(m, n, s1, s2, seed, work, 0, row0)
    prep()
    _, tp = time_steps(torch, prep, 5)
    t_prep = median(tp)

    step = make_step(torch, rq, rdist, Vd, c, seed, Q, R, bufs, flags, shard)
    for _ in range(args.warmup):
        step()
    timed_step = step
    if not args.no_graph:
        # the C ABI neither synchronises nor allocates: the whole factorization (8 launches + a memset, and the two
        # all-reduces of the sharded form) is captured once and replayed, which removes the host launch gaps
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            with torch.cuda.graph(graph, stream=side):
                step()
        torch.cuda.synchronize()
        timed_step = graph.replay
        for _ in range(2):
            timed_step()
    en0 = gpu_energy_mj(torch.cuda.current_device())
    total_ms, per = time_steps(torch, timed_step, steps, barrier)
    en1 = gpu_energy_mj(torch.cuda.current_device())
    ms_med, ms_mean = median(per), total_ms / steps
    if barrier:                                     # every rank reports the slowest rank's figures
        import torch.distributed as dist
        t = torch.tensor([ms_med, ms_mean], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_med, ms_mean = float(t[0]), float(t[1])
    assert int(info.item()) == 0, "numerical failure: info=%d" % int(info.item())
    eye = torch.eye(n, dtype=torch.float64, device="cuda")
    Vn2 = torch.linalg.norm(Vd) ** 2

    def checks():
        QtQ = Q.T @ Q
        num = torch.linalg.norm(Vd - Q @ R) ** 2
        den = Vn2.clone()
        if barrier:
            import torch.distributed as dist
            dist.all_reduce(QtQ); dist.all_reduce(num); dist.all_reduce(den)
        return float(torch.linalg.norm(QtQ - eye)), float(torch.sqrt(num / den))
    orth, res = checks()
    # the other sketch seeds of the recipe: correctness only, worst error reported
    worst_orth, worst_res = orth, res
    for sd in inputs.SKETCH_SEEDS:
        if sd == seed:
            continue
        make_step(torch, rq, rdist, Vd, c, sd, Q, R, bufs, flags & ~rq.FLAG_PREPARED, shard)()
        assert int(info.item()) == 0, "numerical failure at sketch seed %d: info=%d" % (sd, int(info.item()))
        o, r_ = checks()
        worst_orth, worst_res = max(worst_orth, o), max(worst_res, r_)
    prep()                                                      # restore the timed seed's sketch
    mt = m * world
    F = flops.rand_cholqr_flops(mt, n, s1, s2)
    B = flops.rand_cholqr_bytes(mt, n, s1, s2)
    # roofline of the whole job: N GPUs have N times the peaks
    t_roof = max(F / (world * p64 * 1e12), B / (world * peaks["hbm_gbs"] * 1e9))
    out = {"workload": name, "m": m, "n": n, "kappa": c["kappa"], "s1": s1, "s2": s2,
           "ms_per_step": ms_med, "ms_per_step_mean": ms_mean, "timing": "median of %d per-step CUDA-event times "
           "of one timed region (mean beside it)" % steps, "steps": steps,
           "gflops": F / ms_med / 1e6, "gbs": B / ms_med / 1e6,
           "roofline_frac_whole_path": t_roof / (ms_med * 1e-3), "orth_err": orth, "resid": res,
           "orth_err_worst_of_seeds": worst_orth, "resid_worst_of_seeds": worst_res,
           "sketch_seeds": list(inputs.SKETCH_SEEDS), "v1": "recomputed" if recompute else "stored",
           "sketch_gen_ms": t_prep, "ms_with_sketch_gen": ms_med + t_prep}
    if en0 is not None and en1 is not None and total_ms > 0:
        # the board's energy counter over the timed region: the path runs AT the 1 kW power cap
        out["energy_j_per_step"] = (en1 - en0) / 1e3 / steps
        out["power_w_avg_timed_region"] = (en1 - en0) / total_ms
    if shard is None or world == 1:
        # comparator on the same kernels, same V (CholeskyQR2, Alg. 4): same V1 policy, same timing method
        def step_c2():
            rq.cholqr2(Vd, Q, R, work, info)
        for _ in range(2):
            step_c2()
        kc = max(5, steps // 2)
        _, pc = time_steps(torch, step_c2, kc)
        out["cholqr2_ms"] = median(pc)
        out["cholqr2_info"] = int(info.item())
        out["no_slower_than_cholqr2"] = bool(ms_med <= out["cholqr2_ms"])
        if want_comparators:
            # the other in-run comparators of BASELINE.json configs 2, 3 and 5 on the same V and the same kernels:
            # shifted CholeskyQR3 (6 m n^2 flops, 48 m n bytes) and rand_cholQR with ONE dense Gaussian sketch
            # (2 m n s2 + 3 m n^2 flops, 32 m n bytes), each against its own FP64 / HBM roofline (models of sweep.py)
            comp = {"cholqr2": {"ms": out["cholqr2_ms"], "info": out["cholqr2_info"],
                                "roofline_frac": max(flops.cholqr2_flops(m, n) / (p64 * 1e12), 32.0 * m * n / (peaks["hbm_gbs"] * 1e9))
                                / (out["cholqr2_ms"] * 1e-3)}}
            for cname, fn, Fc, Bc, reps_c in (
                    ("scholqr3", lambda: rq.scholqr3(Vd, Q, R, work, info), 6.0 * m * n * n, 48.0 * m * n, 5),
                    ("gauss_rand_cholqr", lambda: rq.gauss_randcholqr(Vd, s2, seed, Q, R, work, info),
                     2.0 * m * n * s2 + 3.0 * m * n * n, 32.0 * m * n, 3)):
                fn()
                _, pcc = time_steps(torch, fn, reps_c)
                st = int(info.item())
                e = {"ms": median(pcc), "info": st,
                     "roofline_frac": max(Fc / (p64 * 1e12), Bc / (peaks["hbm_gbs"] * 1e9)) / (median(pcc) * 1e-3)}
                if st == 0:
                    e["orth_err"], e["resid"] = checks()
                comp[cname] = e
            out["comparators"] = comp
    if want_breakdown:
        out["breakdown_ms"] = breakdown(torch, rq, Vd, c, seed, Q, R, bufs, max(5, steps // 3), recompute, row0)
    if want_e2e:
        # End to end through host buffers.  Every step copies its V from pinned host memory and reads its Q and R
        # back; the steps are pipelined the way a caller streaming panels would run them: double-buffered device
        # arrays, H2D / factorization / D2H on three streams, so step i's read-back overlaps step i+1's upload
        # (PCIe is full duplex; the factorization itself is ~30x shorter than either copy).  The serial figure
        # (one step start to finish on one stream) is reported beside it.
        Vh = torch.empty(Vd.shape, dtype=torch.float64, pin_memory=True)
        Vh.copy_(Vd)
        Qh = [torch.empty(Vd.shape, dtype=torch.float64, pin_memory=True) for _ in range(2)]
        Rh = [torch.empty(n, n, dtype=torch.float64, pin_memory=True) for _ in range(2)]
        Vin = [torch.empty_like(Vd), Vd]            # Vd is not needed any more: second input buffer
        Qd = [Q, torch.empty_like(Vd)]
        Rd = [R, torch.empty_like(R)]
        steps_of = [make_step(torch, rq, rdist, Vin[b], c, seed, Qd[b], Rd[b], bufs, flags, shard) for b in range(2)]

        def step_serial():
            Vin[0].copy_(Vh, non_blocking=True)
            steps_of[0]()
            Qh[0].copy_(Qd[0], non_blocking=True)
            Rh[0].copy_(Rd[0], non_blocking=True)
        step_serial()
        k = max(2, min(steps, 5))
        ms_serial = time_region(torch, step_serial, k) / k

        s_in, s_cmp, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()

        def run_pipeline(nsteps):
            ev_in = [None, None]; ev_cmp = [None, None]; ev_out = [None, None]
            if barrier:
                barrier()
            torch.cuda.synchronize()
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(s_in):
                e0.record()
            for i in range(nsteps):
                b = i & 1
                with torch.cuda.stream(s_in):
                    if ev_cmp[b] is not None:
                        s_in.wait_event(ev_cmp[b])              # the factorization that read Vin[b] is done
                    Vin[b].copy_(Vh, non_blocking=True)
                    ev_in[b] = torch.cuda.Event(); ev_in[b].record()
                with torch.cuda.stream(s_cmp):
                    s_cmp.wait_event(ev_in[b])
                    if ev_out[b] is not None:
                        s_cmp.wait_event(ev_out[b])             # Qd[b], Rd[b] have been read back
                    steps_of[b]()
                    ev_cmp[b] = torch.cuda.Event(); ev_cmp[b].record()
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_cmp[b])
                    Qh[b].copy_(Qd[b], non_blocking=True)
                    Rh[b].copy_(Rd[b], non_blocking=True)
                    ev_out[b] = torch.cuda.Event(); ev_out[b].record()
            with torch.cuda.stream(s_out):
                s_out.wait_stream(s_in); s_out.wait_stream(s_cmp)
                e1.record()
            torch.cuda.synchronize()
            if barrier:
                barrier()
            return e0.elapsed_time(e1)
        run_pipeline(3)
        ke = max(4, min(steps, 20))
        ms_e = run_pipeline(ke) / ke
        if barrier:
            import torch.distributed as dist
            t = torch.tensor([ms_e, ms_serial], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms_e, ms_serial = float(t[0]), float(t[1])
        ok = bool(int(info.item()) == 0 and torch.equal(Qh[0], Qh[1]) and torch.equal(Rh[0], Rh[1]))
        out["e2e"] = {"value": F / ms_e / 1e6, "unit": "GFLOP/s", "ms_per_step": ms_e, "steps": ke,
                      "h2d_bytes_per_step": int(8 * mt * n), "d2h_bytes_per_step": int(8 * mt * n + 8 * n * n * world),
                      "pipeline": "double-buffered; H2D, factorization, D2H on three streams; whole region timed "
                                  "from the first upload to the last read-back",
                      "serial_ms_per_step": ms_serial, "serial_value": F / ms_serial / 1e6,
                      "results_identical_across_buffers": ok}
        out["_V_host_sample"] = None if args.no_cpu_baseline else Vh[: min(m, ORACLE_SAMPLE_ROWS)].numpy().copy()
        del Vh, Qh, Vin, Qd, steps_of
    else:
        out["_V_host_sample"] = None if args.no_cpu_baseline else Vd[: min(m, ORACLE_SAMPLE_ROWS)].cpu().numpy()
    del Vd, Q, bufs, step, timed_step
    torch.cuda.empty_cache()
    return out, F


_JSON_FD = None


def _claim_stdout():
    """stdout carries exactly ONE line, the JSON record.  Libraries loaded below write to file descriptor 1 on their
    own (NCCL prints "NCCL version ..." there on the first communicator, whatever NCCL_DEBUG_FILE says): keep a
    private duplicate of the real stdout for the record and point descriptor 1 at stderr for everything else."""
    global _JSON_FD
    if _JSON_FD is None:
        sys.stdout.flush()
        _JSON_FD = os.dup(1)
        os.dup2(2, 1)


def _emit(line):
    sys.stdout.flush()
    data = (json.dumps(line) + "\n").encode()
    if _JSON_FD is None:
        os.write(1, data)
    else:
        os.write(_JSON_FD, data)


def main():
    args = parse()
    _claim_stdout()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import __graft_entry__ as ge
    from paper_2309_05868_b200 import binding as rq, flops, inputs
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if rank == 0:
        ge.build()
    sharded = world > 1 or args.force_sharded
    if sharded:
        import torch.distributed as dist
        # NCCL writes its "NCCL version ..." / debug lines to stdout: send them to stderr, stdout is the one JSON line
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        os.environ.setdefault("RANK", "0")
        os.environ.setdefault("WORLD_SIZE", "1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()                                   # rank 0 has built the libraries
    rq.lib()
    peaks = measured_peaks()
    sampler = ClockSampler(local)
    sampler.start()
    p64s = {"dfma": 34.2, "dmma": 37.2, "note": "not probed in this run"} if args.no_probe else probe_fp64_peak(torch)
    ratio_peak = (peaks["bf16_tflops"] or 1590.0) * (45.0 / 2250.0)   # guide's nominal FP64:bf16 ratio
    p64 = max(p64s["dfma"], p64s["dmma"], 1e-3)
    hbm_sustained = None if args.no_probe else probe_hbm_sustained(torch)
    c = inputs.config(args.workload)
    m, n = c["m"], c["n"]
    shard = (world, rank, rank * m) if sharded else None
    main_out, F = run_config(torch, rq, args.workload, args, peaks, p64, want_e2e=not args.no_e2e, shard=shard,
                             want_comparators=not args.no_extra)
    sampler.stop()
    sampler.join(timeout=1.0)
    clocks = sampler.summary()
    extra = None
    if not args.no_extra and not sharded and rank == 0:
        # the other BASELINE configurations that fit the time budget, and three sweep points at m = 2^22 (C5): the
        # ">= 60% of the roofline and no slower than CholeskyQR2 for m >= 2^22" claim, printed by this process
        extra = {"configs": {}, "sweep_m_2p22": []}
        for nm, st in (("C2", 20), ("C4", 10)):
            if nm == args.workload:
                continue
            o, _ = run_config(torch, rq, nm, args, peaks, p64, want_e2e=False, want_breakdown=True, steps=st,
                              want_comparators=(nm == "C2"))
            o.pop("_V_host_sample", None)
            extra["configs"][nm] = o
        for nn in (32, 64, 128):
            o, _ = run_config(torch, rq, "C5", args, peaks, p64, want_e2e=False, want_breakdown=False, steps=20,
                              shape=(1 << 22, nn, 1e12))
            o.pop("_V_host_sample", None)
            extra["sweep_m_2p22"].append({k: o[k] for k in ("m", "n", "kappa", "ms_per_step", "gflops",
                                                           "roofline_frac_whole_path", "orth_err", "v1",
                                                           "cholqr2_ms", "cholqr2_info", "no_slower_than_cholqr2")})
    bd = main_out["breakdown_ms"]
    recompute = main_out["v1"] == "recomputed"
    per_step = per_step_roofline(bd, m, n, p64, peaks["hbm_gbs"], recompute, args.workload)
    dom = max(per_step, key=lambda e: e["ms"])
    roof = {"kernel": dom["kernel"], "bound": dom["bound"], "achieved": dom["achieved"], "peak": dom["peak"],
            "unit": dom["unit"], "frac": dom["frac"], "traffic": dom["traffic"],
            "traffic_source": dom.get("traffic_source"),
            "algorithmic": "A4: 2 m n^2 flops per launch (n^2 substitution + n^2 symmetric Gram per row), 16 m n bytes "
                           "(read V, write V1; 8 m n when V1 is not stored)" + ("; n > 64: two kernels, the syrk re-reads V1 (24 m n)" if n > 64 else "")
                           + "; A1: 8 m n bytes; A6: 16 m n bytes, m n^2 flops",
            "peak_source": "tensor: FP64 probe measured live in this run (max of DFMA %.1f / DMMA %.1f TFLOP/s; "
                           "MEASURED_PEAKS.json has no FP64 figure; bf16 x nominal ratio would give %.1f); "
                           "hbm: MEASURED_PEAKS.json hbm_gbs (%s)" % (p64s["dfma"], p64s["dmma"], ratio_peak, peaks["source"]),
            "per_step": per_step}
    cpu = None
    cpu_other = {}
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        cpu, _ = oracle_sample(main_out.pop("_V_host_sample"), n, args.seed)
        if not args.no_extra:
            # SURVEY.md 8(d) "oracle beside it": also C1 (whole) and C2 (whole)
            for nm in ("C1", "C2"):
                if nm == args.workload:
                    continue
                cc = inputs.config(nm)
                Vh = inputs.make_V(min(cc["m"], ORACLE_SAMPLE_ROWS), cc["n"], cc["kappa"], cc["seed"]).numpy()
                cpu_other[nm], _ = oracle_sample(Vh, cc["n"], args.seed)
    main_out.pop("_V_host_sample", None)
    if rank != 0:
        if sharded:
            import torch.distributed as dist
            dist.destroy_process_group()
        return
    nl = launches_per_step(n, m, c["s1"])          # the sharded one-shot launches the same kernels (+ 2 all-reduces)
    line = {"metric": "rand_cholQR FP64 GFLOP/s", "value": main_out["gflops"], "unit": "GFLOP/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": main_out["ms_per_step"],
            "ms_per_step_mean": main_out["ms_per_step_mean"], "timing": main_out["timing"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(args, c, args.workload, v1_mode_of(args, n)),
            "gbs": main_out["gbs"], "roofline_frac_whole_path": main_out["roofline_frac_whole_path"],
            "orth_err": main_out["orth_err"], "resid": main_out["resid"],
            "orth_err_worst_of_seeds": main_out["orth_err_worst_of_seeds"],
            "resid_worst_of_seeds": main_out["resid_worst_of_seeds"], "sketch_seeds": main_out["sketch_seeds"],
            "cholqr2_ms": main_out.get("cholqr2_ms"), "cholqr2_info": main_out.get("cholqr2_info"),
            "no_slower_than_cholqr2": main_out.get("no_slower_than_cholqr2"),
            "comparators": main_out.get("comparators"),
            "sketch_gen_ms": main_out["sketch_gen_ms"], "ms_with_sketch_gen": main_out["ms_with_sketch_gen"],
            "breakdown_ms": bd, "fp64_peak_tflops": p64s, "e2e": main_out.get("e2e"),
            "gpu_launches": nl * args.steps * world, "roofline": roof, "cpu_baseline": cpu,
            "cpu_baseline_other_configs": cpu_other or None, "clocks": clocks,
            # the path runs at the board's power cap: energy counter over the timed region, and the
            # sustained device-copy bandwidth (1 s loop) beside the burst figure of MEASURED_PEAKS.json
            "power": {"energy_j_per_step": main_out.get("energy_j_per_step"),
                      "power_w_avg_timed_region": main_out.get("power_w_avg_timed_region"),
                      "hbm_sustained_gbs": hbm_sustained, "hbm_burst_gbs": peaks["hbm_gbs"],
                      "note": "every m-sized kernel of the step runs at the 1 kW cap (sw_power_cap): the burst peaks of the "
                              "roofline (FP64 probe at ~600 W, device copy) are not reachable together under it"},
            "extra": extra}
    if sharded:
        line["config"].update({"m_per_gpu": m, "m_total": m * world,
                               "parallelism": "row-sharded, 2 all-reduces (W, G) per step"})
    _emit(line)
    if sharded:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
