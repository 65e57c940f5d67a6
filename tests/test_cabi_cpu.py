"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol the headers
declare, and rejects bad arguments before touching the GPU.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2309_05868_b200 import build
    build.build_lib()
    from paper_2309_05868_b200 import binding
    return binding.lib()


def declared_symbols():
    names = set()
    inc = os.path.join(ROOT, "include")
    for f in os.listdir(inc):
        if f.endswith(".h"):
            src = open(os.path.join(inc, f)).read()
            src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
            names |= set(re.findall(r"\b(rqr_[a-zA-Z0-9_]+)\s*\(", src))
    return names


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert {"rqr_countsketch", "rqr_gauss_sketch", "rqr_small_geqrf", "rqr_trsm_gram", "rqr_chol",
            "rqr_apply", "rqr_rand_cholqr", "rqr_cholqr2", "rqr_scholqr3"} <= names
    for n in names:
        assert hasattr(lib, n), n
    from paper_2309_05868_b200 import binding
    assert names == set(binding.SIGNATURES), names ^ set(binding.SIGNATURES)


def test_version_and_workspace(lib):
    assert b"rqr" in lib.rqr_version()
    b1 = lib.rqr_workspace_bytes(1 << 20, 64, 8192, 128, 0)
    b2 = lib.rqr_workspace_bytes(1 << 23, 64, 8192, 128, 0)
    assert 0 < b1 < b2 < (1 << 30)
    # only the sorted row list, its radix-sort twin and the sort's tile counts grow with m: 8 bytes per row + ~2 MB
    assert 8 * ((1 << 23) - (1 << 20)) <= b2 - b1 <= 8 * ((1 << 23) - (1 << 20)) + (4 << 20)
    assert lib.rqr_workspace_bytes(100, 1, 10, 10, 0) == 0   # n < 2
    assert lib.rqr_workspace_bytes(100, 300, 10, 10, 0) == 0


def test_argument_validation_without_gpu(lib):
    one = ctypes.c_void_p(16)   # non-null dummy, never dereferenced: checks come first
    z = ctypes.c_void_p(0)
    assert lib.rqr_countsketch(z, 10, 4, 4, 0, 8, 1, one, one, 0, 0, z) == -1
    assert lib.rqr_countsketch(one, 10, 1, 4, 0, 8, 1, one, one, 0, 0, z) == -3
    assert lib.rqr_countsketch(one, 10, 4, 3, 0, 8, 1, one, one, 0, 0, z) == -4     # ldv < n
    assert lib.rqr_countsketch(one, 10, 4, 4, 0, 8, 1, one, one, 7, 0, z) == -10
    assert lib.rqr_gauss_sketch(one, 8, 4, 9, 1, one, one, 0, z) == -4              # s2 > s1
    assert lib.rqr_small_geqrf(one, 3, 4, one, z, z) == -3                          # n > s2
    assert lib.rqr_trsm_gram(one, 10, 4, 2, z, one, z, 4, one, z) == -4
    assert lib.rqr_chol(z, 4, 0.0, one, z, z) == -1
    assert lib.rqr_apply(one, 10, 4, 4, z, z, one, 4, z, z) == -6
    assert lib.rqr_triu_mul(one, one, 4, one, z) == -4                              # aliasing
    # eq. (20): 1 < n <= s2 <= s1 <= m
    assert lib.rqr_rand_cholqr(one, 100, 8, 200, 16, 1, one, one, one, z, 0, 0, z) == -4   # s1 > m
    assert lib.rqr_rand_cholqr(one, 100, 8, 64, 4, 1, one, one, one, z, 0, 0, z) == -5     # s2 < n
    assert lib.rqr_rand_cholqr(one, 100, 8, 64, 80, 1, one, one, one, z, 0, 0, z) == -5    # s2 > s1
    assert lib.rqr_rand_cholqr(one, 4, 8, 4, 8, 1, one, one, one, z, 0, 0, z) == -3        # n > m
    assert lib.rqr_cholqr2(z, 100, 8, one, one, one, z, z) == -1
    assert lib.rqr_sketch_prepare(100, 8, 0, 64, 600, 1, 0, one, z) == -5
    # batched / strided one-shot and the Rademacher test hook
    assert lib.rqr_rand_cholqr_batched(one, 100, 8, 0, 800, 64, 16, 1, one, 800, one, one, z, 0, 1, z) == -4     # batch < 1
    assert lib.rqr_rand_cholqr_batched(one, 100, 8, 2, 799, 64, 16, 1, one, 800, one, one, z, 0, 1, z) == -5     # stride < m n
    assert lib.rqr_rand_cholqr_batched(z, 100, 8, 2, 800, 64, 16, 1, one, 800, one, one, z, 0, 1, z) == -1
    # row-sharded one-shot: V m row0 m_total n s1 s2 seed Q R work info variant flags allreduce ctx stream
    assert lib.rqr_rand_cholqr_sharded(one, 100, -1, 200, 8, 64, 16, 1, one, one, one, z, 0, 0, z, z, z) == -3      # row0 < 0
    assert lib.rqr_rand_cholqr_sharded(one, 100, 150, 200, 8, 64, 16, 1, one, one, one, z, 0, 0, z, z, z) == -4     # past m_total
    assert lib.rqr_rand_cholqr_sharded(one, 100, 0, 200, 8, 300, 16, 1, one, one, one, z, 0, 0, z, z, z) == -6      # s1 > m_total
    assert lib.rqr_rand_cholqr_sharded(one, 4, 0, 200, 8, 64, 4, 1, one, one, one, z, 0, 0, z, z, z) == -7          # s2 < n (a 4-row shard is fine)
    assert lib.rqr_rand_cholqr_sharded(z, 100, 0, 200, 8, 64, 16, 1, one, one, one, z, 0, 0, z, z, z) == -1
    assert lib.rqr_debug_rademacher(1, 100, 2000, 0, 10, one, z) == -3                                          # row
    assert lib.rqr_debug_rademacher(1, 100, 3, 95, 10, one, z) == -4                                            # past s1
    # the Rademacher S2 needs no S2 slot: 8 * 1024 * ld bytes less
    full = lib.rqr_workspace_bytes(1 << 20, 64, 8192, 128, 0)
    lean = lib.rqr_workspace_bytes(1 << 20, 64, 8192, 128, 16)
    assert full - lean == 8 * 1024 * 8192
    assert lib.rqr_rand_cholqr(one, 100, 8, 64, 16, 1, one, one, one, z, 3, 0, z) == -11                         # variant
    assert lib.rqr_rand_cholqr(one, 100, 8, 64, 16, 1, one, one, one, z, 32, 0, z) == -11


def test_noalloc_entry_point_limits_without_gpu(lib):
    """rqr_trsm_gram_noalloc: the limits of its built-in scratch are checked from the sizes alone, before the device
    is touched, and the header's constants are the binding's."""
    from paper_2309_05868_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "rqr.h")).read()
    assert int(re.search(r"#define RQR_NOALLOC_MAX_N (\d+)", hdr).group(1)) == binding.NOALLOC_MAX_N == 64
    assert re.search(r"#define RQR_NOALLOC_MAX_M \(\(int64_t\)1 << (\d+)\)", hdr).group(1) == "23"
    assert binding.NOALLOC_MAX_M == 1 << 23
    assert int(re.search(r"#define RQR_ERR_SCRATCH_LIMIT \((-\d+)\)", hdr).group(1)) == binding.ERR_SCRATCH_LIMIT
    one = ctypes.c_void_p(16)
    z = ctypes.c_void_p(0)
    f = lib.rqr_trsm_gram_noalloc
    assert f(one, 100, 66, 66, z, one, z, 66, z) == binding.ERR_SCRATCH_LIMIT
    assert f(one, (1 << 23) + 1, 64, 64, z, one, z, 64, z) == binding.ERR_SCRATCH_LIMIT
    assert f(z, 100, 64, 64, z, one, z, 64, z) == -1
    assert f(one, 0, 64, 64, z, one, z, 64, z) == -2
    assert f(one, 100, 1, 64, z, one, z, 64, z) == -3
    assert f(one, 100, 64, 63, z, one, z, 64, z) == -4
    assert f(one, 100, 64, 64, z, z, z, 64, z) == -6
    assert f(one, 100, 64, 64, z, one, one, 63, z) == -8


def test_binding_refuses_cpu_tensors(lib):
    import torch
    from paper_2309_05868_b200 import binding
    V = torch.zeros(8, 4, dtype=torch.float64)
    with pytest.raises(binding.RqrError):
        binding.countsketch(V, 4, 1, torch.zeros(4, 4, dtype=torch.float64), None)


def test_product_does_not_import_oracle():
    bad = re.compile(r"^\s*(import|from)\s+\S*oracle|#include.*oracle|librqr_oracle|CDLL\(.*oracle")
    pkg = os.path.join(ROOT, "paper_2309_05868_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                for ln in open(os.path.join(dirpath, f)).read().splitlines():
                    assert not bad.search(ln), (f, ln)
    bad2 = re.compile(r"^\s*(import|from)\s+paper_2309_05868_b200|#include\s+\"[^\"]*(rqr\.h|csrc|\.cuh)|CDLL\(.*librqr\.so")
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py") or f.endswith(".c"):
            for ln in open(os.path.join(ROOT, "oracle", f)).read().splitlines():
                assert not bad2.search(ln), (f, ln)


def test_eps_sweep_sketch_sizes():
    """Sketch sizes of the eps sweep: constants as printed, natural log (S17).
    The eps = 0.9 multisketch sizes are the paper grid's; a larger eps always means a smaller sketch."""
    import math
    from paper_2309_05868_b200 import eps_sweep as es, paper_grid
    assert es.gauss_size(100, 0.99) == math.ceil(36.01 * math.log(100)) == 166
    assert es.gauss_size(100, 0.49) == 343
    assert es.count_size(10, 0.99) == 748 and es.count_size(10, 0.49) == 3058      # 6.8 * 110, 27.8 * 110
    for n in range(10, 101, 10):
        assert es.multi_sizes(n, 0.9) == paper_grid.paper_sketch_sizes(n)
        assert es.gauss_size(n, 0.99) < es.gauss_size(n, 0.49)
        assert es.count_size(n, 0.99) < es.count_size(n, 0.9) < es.count_size(n, 0.49)
        s1, s2 = es.multi_sizes(n, 0.49)
        assert n <= s2 <= s1 and s2 <= 1024                                      # eq. (20) ordering, library limit
