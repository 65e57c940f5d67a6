"""Builds librqr.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librqr.so")
PROBE_DIR = os.path.join(HERE, "bench_probe")
PROBE_LIB = os.path.join(HERE, "librqr_probe.so")       # bench-only FP64 peak probe, not part of librqr.so
SOURCES = ["rqr_sketch.cu", "rqr_gauss_mma.cu", "rqr_dense_mma.cu", "rqr_small.cu", "rqr_tall.cu", "rqr_tall_mma.cu", "rqr_tall_panel.cu", "rqr_api.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("RQR_EXTRA_NVCC_FLAGS", "").split()


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [
        os.path.join(HERE, "..", "include", f) for f in os.listdir(os.path.join(HERE, "..", "include"))]
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)

    def compile_one(src):
        obj = os.path.join(HERE, "build", src.replace(".cu", ".o"))
        cmd = ["nvcc", *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s" % (src, r.stderr))
        return obj, r.stderr

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
        done = list(ex.map(compile_one, SOURCES))
    objs = [o for o, _ in done]
    log = [e for _, e in done]
    cmd = ["nvcc", "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stderr)
    with open(os.path.join(HERE, "build", "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


def build_probe(force: bool = False) -> str:
    """The FP64 peak probe of bench.py / sweep.py (bench_probe/): its own small shared object."""
    src = os.path.join(PROBE_DIR, "rqr_probe.cu")
    if not force and os.path.exists(PROBE_LIB) and all(
            os.path.getmtime(os.path.join(PROBE_DIR, f)) <= os.path.getmtime(PROBE_LIB) for f in os.listdir(PROBE_DIR)):
        return PROBE_LIB
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
           "-shared", src, "-o", PROBE_LIB]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for the probe:\n" + r.stderr)
    return PROBE_LIB


if __name__ == "__main__":
    print(build_lib(force=True, verbose=True))
    print(build_probe(force=True))
