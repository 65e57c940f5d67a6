"""GPU parity, step by step: every C-ABI entry point against the CPU oracle on the same seeded
inputs (element by element where the result is unique, invariants where it is not).
Tolerances: integer/index work bit-exact; Gaussian entries 1e-15
(north_star); sums and triangular solves with well-conditioned factors 1e-13 relative."""
import numpy as np
import pytest
import torch

from paper_2309_05868_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rq():
    from paper_2309_05868_b200 import binding
    binding.lib()
    assert torch.cuda.is_available()
    return binding


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def host(t):
    return t.detach().cpu().numpy()


@pytest.mark.parametrize("s1,row0,count", [(512, 0, 5000), (8192, 0, 70000), (9940, 123, 4097),
                                           (8192, (1 << 33) + 5, 300), (131072, 7, 20000)])
def test_hash_sign_bit_exact(rq, orc, s1, row0, count):
    b, s = rq.debug_hash_sign(42, row0, count, s1)
    bo, so = orc.hash_sign(42, row0, count, s1)
    assert np.array_equal(host(b).astype(np.uint32), bo)
    assert np.array_equal(host(s), so)


def test_gauss_entries_within_1e15(rq, orc):
    for stream, first, count in [(1, 0, 200001), (3, (1 << 40) + 1, 50001), (1, 12345, 7)]:
        z = host(rq.debug_gauss(42, stream, first, count))
        zo = orc.gauss_z(42, stream, first, count)
        assert np.all(np.abs(z - zo) <= 1e-15 * np.maximum(np.abs(zo), 1.0))
        assert np.max(np.abs(z - zo) / np.maximum(np.abs(zo), 1e-3)) < 1e-12


def test_prepared_S2_matches_oracle(rq, orc):
    m, n = 4096, 16
    s1, s2 = 700, 33                      # odd sizes: pairs straddle rows
    work = rq.alloc_workspace(m, n, s1, s2)
    rq.sketch_prepare(m, n, s1, s2, 43, work)
    S2 = host(rq.workspace_S2(work, n, s1, s2))
    S2o = orc.gauss_matrix(43, s2, s1)
    assert np.all(np.abs(S2 - S2o) <= 1e-15 * np.maximum(np.abs(S2o), 1.0 / np.sqrt(s2)))


@pytest.mark.parametrize("m,s1,row0", [(100000, 8192, 0), (70001, 9940, 12345), (300000, 200, 0), (5000, 131072, 7),
                                       (1 << 21, 2048, 1 << 33)])
def test_sorted_row_list_is_the_stable_sort(rq, orc, m, s1, row0):
    """A0: the row list rqr_sketch_prepare writes must be, bit for bit, the STABLE sort of the rows by the oracle's
    bucket (ascending row inside a bucket) with the oracle's sign in bit 31, and the offsets the bucket histogram's
    exclusive scan ("sorted row list: bit-exact")."""
    n = 16
    s2 = 32
    work = rq.alloc_workspace(m, n, s1, s2)
    rq.sketch_prepare(m, n, s1, s2, 42, work, 0, row0)
    off, ent = rq.workspace_rows(work, m, n, s1)
    off = host(off).view(np.uint32); ent = host(ent).view(np.uint32)
    bo, so = orc.hash_sign(42, row0, m, s1)
    order = np.argsort(bo, kind="stable").astype(np.uint32)
    expect = order | ((so[order] < 0).astype(np.uint32) << np.uint32(31))
    assert np.array_equal(ent, expect)
    assert np.array_equal(off, np.concatenate([[0], np.cumsum(np.bincount(bo, minlength=s1))]).astype(np.uint32))


@pytest.mark.parametrize("m,n,s1", [(20000, 16, 512), (100000, 70, 9940), (65536, 64, 8192),
                                    (5000, 33, 64), (3000, 256, 4000), (37, 8, 16), (8192, 2, 8),
                                    # few buckets: every bucket's row list is split over several CTAs (two-stage sum)
                                    (200000, 10, 200), (150001, 16, 64), (120000, 7, 37), (300000, 24, 500)])
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_countsketch_parity(rq, orc, m, n, s1, variant):
    V = inputs.make_V(m, n, 1e8, 7)
    Vd = V.cuda()
    W1 = torch.empty(s1, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, s1, min(2 * n, s1))
    rq.countsketch(Vd, s1, 42, W1, work, variant=variant)
    W1o = orc.countsketch(V.numpy(), s1, 42)
    scale = np.abs(W1o).max()
    assert np.abs(host(W1) - W1o).max() <= 1e-13 * scale
    if variant == 0:                      # sorted variant is bit-reproducible
        W1b = torch.empty_like(W1)
        rq.countsketch(Vd, s1, 42, W1b, work, variant=0)
        assert torch.equal(W1, W1b)
    # integer input: every partial sum exact => bit-exact whatever the order (K4)
    Vi = inputs.make_integer_V(m, n, 3)
    rq.countsketch(Vi.cuda(), s1, 42, W1, work, variant=variant)
    assert np.array_equal(host(W1), orc.countsketch(Vi.numpy(), s1, 42))


def test_countsketch_strided_and_row_offset(rq, orc):
    m, n, s1 = 6000, 24, 300
    big = inputs.make_integer_V(m, n + 6, 5).cuda()
    V = big[:, :n]                        # ldv = n + 6
    W1 = torch.empty(s1, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, s1, 2 * n)
    for variant in (0, 1, 2):
        rq.countsketch(V, s1, 9, W1, work, variant=variant, row0=1000)
        ref = orc.countsketch(host(V), s1, 9, row0=1000)
        assert np.array_equal(host(W1), ref)


@pytest.mark.parametrize("m,n,ld,s1,row0", [(70001, 12, 15, 300, 1000), (50000, 19, 19, 700, (1 << 33) + 3),
                                            (33, 20, 22, 1400, 5), (100000, 3, 3, 9333, 0)])
def test_countsketch_stream_tile_form(rq, orc, m, n, ld, s1, row0):
    """RQR_VARIANT_STREAM with a sketch that fits shared memory (n <= 20, 8 s1 n <= 224 KB): the shared-memory
    bucket-tile kernel (k_countsketch_tile): strided V, odd n, row offsets, odd s1 n (element-wise flush), a tile at the
    size limit (1400 x 20) and a ragged last group."""
    big = inputs.make_integer_V(m, ld, 6).cuda()
    V = big[:, :n]
    W1 = torch.full((s1, n), float("nan"), dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, s1, min(2 * n, s1))
    rq.countsketch(V, s1, 11, W1, work, variant=2, row0=row0)
    assert np.array_equal(host(W1), orc.countsketch(host(V), s1, 11, row0=row0))
    Vr = inputs.make_V(m, n, 1e6, 8) if m >= n else inputs.make_graded_V(m, n, 1, 8)
    rq.countsketch(Vr.cuda(), s1, 11, W1, work, variant=2, row0=row0)
    W1o = orc.countsketch(Vr.numpy(), s1, 11, row0=row0)
    assert np.abs(host(W1) - W1o).max() <= 1e-13 * np.abs(W1o).max()


def test_new_kernels_write_only_their_outputs(rq, orc):
    """Guard bands around the outputs of the kernels added in round 2 (compute-sanitizer is not available on the pool):
    the shared-memory-tile CountSketch (bulk-reduction flush and element-wise flush), the DMMA sketch GEMM below
    n = 96 and the four-columns-per-warp Householder kernel must leave every sentinel outside their output intact."""
    SENT = 1234.5
    def guarded(rows, cols, g=64):
        buf = torch.full(((rows + 2 * g) * cols,), SENT, dtype=torch.float64, device="cuda")
        return buf, buf[g * cols:(g + rows) * cols].view(rows, cols)
    def intact(buf, rows, cols, g=64):
        return bool((buf[:g * cols] == SENT).all()) and bool((buf[(g + rows) * cols:] == SENT).all())
    for m, n, s1 in [(50000, 20, 1400), (70001, 7, 37), (33, 12, 5)]:
        V = inputs.make_integer_V(m, n, 9).cuda()
        buf, W1 = guarded(s1, n)
        work = rq.alloc_workspace(m, n, s1, min(2 * n, s1))
        rq.countsketch(V, s1, 3, W1, work, variant=2)
        torch.cuda.synchronize()
        assert intact(buf, s1, n)
        assert np.array_equal(host(W1), orc.countsketch(host(V), s1, 3))
    for s1, n, s2 in [(13514, 40, 707), (9001, 34, 900), (8192, 64, 128)]:
        rng = np.random.default_rng(s1)
        W1 = dev(rng.standard_normal((s1, n)))
        buf, W = guarded(s2, n)
        work = rq.alloc_workspace(s1, n, s1, s2)
        rq.gauss_sketch(W1, s2, 42, W, work)
        torch.cuda.synchronize()
        assert intact(buf, s2, n)
        Wo = orc.gauss_sketch(host(W1), s2, 42)
        assert np.abs(host(W) - Wo).max() <= 1e-13 * np.abs(Wo).max()
    for s2, n in [(64, 32), (20, 10), (128, 30), (37, 13)]:
        rng = np.random.default_rng(s2 + n)
        Wm = rng.standard_normal((s2, n))
        buf, R0 = guarded(n, n)
        info = rq.new_info()
        rq.small_geqrf(dev(Wm), R0, info)
        torch.cuda.synchronize()
        assert intact(buf, n, n) and int(info.item()) == 0
        Ro, _ = orc.hhqr_r(Wm)
        assert np.linalg.norm(host(R0) - Ro) <= 1e-13 * np.linalg.norm(Ro)


@pytest.mark.parametrize("s1,n,s2", [(512, 16, 32), (8192, 64, 128), (9940, 70, 140), (300, 5, 7),
                                     (4096, 256, 512), (32768, 128, 256), (9984, 200, 401), (40000, 98, 130),
                                     (65536, 256, 512), (40953, 70, 789),
                                     # 32 <= n < 96 with a large product: the DMMA GEMM with 8 / 10 / 12 column blocks
                                     (13514, 40, 707), (30159, 60, 767), (9001, 34, 900), (12000, 88, 333)])
def test_gauss_sketch_parity(rq, orc, s1, n, s2):
    rng = np.random.default_rng(s1 + n)
    W1 = rng.standard_normal((s1, n))
    W = torch.empty(s2, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(s1, n, s1, s2)
    rq.gauss_sketch(dev(W1), s2, 42, W, work)
    Wo = orc.gauss_sketch(W1, s2, 42)
    assert np.abs(host(W) - Wo).max() <= 1e-13 * np.abs(Wo).max()


@pytest.mark.parametrize("m,n,s,row0,m_total", [(5000, 20, 40, 0, None), (4099, 10, 83, 0, None), (3001, 64, 128, 0, None),
                                                 (2500, 100, 166, 0, None), (1500, 200, 343, 0, None), (1000, 256, 300, 0, None),
                                                 (2001, 33, 70, 999, 3001), (2000, 16, 33, 1, 2001), (37, 9, 12, 0, None)])
def test_dense_gauss_sketch_parity(rq, orc, m, n, s, row0, m_total):
    """One dense Gaussian sketch W = S V, every column-slot / row-blocking variant of the
    kernel; odd m_total and odd row0 make the first entry of a row tile fall on the second output of a Box-Muller
    pair (the unpaired path); row0 / m_total is the row-sharded call of dist.py."""
    V = inputs.make_V(m, n, 1e3, 2)
    W = torch.empty(s, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, 2 * n * n, 2 * n)
    rq.dense_gauss_sketch(V.cuda(), s, 5, W, work, row0, m_total)
    Wo = orc.dense_gauss_sketch(V.numpy(), s, 5, row0, m_total)
    assert np.abs(host(W) - Wo).max() <= 1e-13 * np.abs(Wo).max()


@pytest.mark.parametrize("s2,n", [(32, 16), (128, 64), (140, 70), (256, 128), (512, 256), (9, 9),
                                  (64, 2), (300, 37), (789, 70), (1000, 100), (700, 30), (1024, 128), (600, 200),
                                  (1024, 256), (900, 150), (513, 129), (140, 69), (512, 255), (200, 97)])
def test_small_geqrf_parity(rq, orc, s2, n):
    rng = np.random.default_rng(s2 * 1000 + n)
    W = rng.standard_normal((s2, n)) * np.logspace(0, -10, n)
    R0 = torch.full((n, n), np.nan, dtype=torch.float64, device="cuda")
    info = rq.new_info()
    rq.small_geqrf(dev(W), R0, info)
    Ro, io = orc.hhqr_r(W)
    R = host(R0)
    assert int(info.item()) == 0 and io == 0
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R))
    assert (np.diag(R) > 0).all()
    assert np.linalg.norm(R - Ro) <= 1e-13 * np.linalg.norm(Ro)
    # row-wise too: row j of R is determined to ~u relative to ||W[:, j:]|| scaling
    assert np.all(np.linalg.norm(R - Ro, axis=1) <= 1e-12 * np.linalg.norm(Ro, axis=1) + 1e-300)


def test_small_geqrf_flags_rank_deficiency(rq, orc):
    W = np.zeros((20, 4)); W[:, 0] = 1; W[:, 2] = 2; W[3, 3] = 1
    info = rq.new_info()
    R0 = torch.empty(4, 4, dtype=torch.float64, device="cuda")
    rq.small_geqrf(dev(W), R0, info)
    _, io = orc.hhqr_r(W)
    assert int(info.item()) == rq.INFO_SINGULAR + 2 == io - orc.ORC_SINGULAR + rq.INFO_SINGULAR


SHAPES_TALL = [(20000, 16), (4099, 64), (10000, 70), (3000, 32), (2500, 128), (700, 256), (65, 8), (5, 2),
               (40003, 128), (30011, 200), (20000, 256), (9001, 66),
               # last panel of 16 / 48 columns at 2, 3 and 4 panels (panel_last_nb = 2, 6)
               (3001, 80), (3001, 100), (2003, 112), (2000, 140), (2000, 176), (1500, 208), (1500, 240),
               # 5 and 6 column blocks (32 < n <= 48; 5 blocks: X staging row padded from 40 to 48 doubles)
               (5000, 40), (4099, 36), (5003, 48), (3001, 44),
               # 3 column blocks (16 < n <= 24): the X staging row is padded to 32 doubles
               (5000, 20), (4099, 24), (3001, 18),
               # 7 column blocks (48 < n <= 56)
               (5000, 50), (4099, 56), (3001, 52)]


@pytest.mark.parametrize("m,n", SHAPES_TALL)
@pytest.mark.parametrize("generic", [False, True])
def test_trsm_gram_parity(rq, orc, m, n, generic):
    rq.force_generic(generic)
    try:
        V = inputs.make_V(m, n, 1e3, 11) if m >= n else inputs.make_graded_V(m, n, 1, 11)
        R0 = inputs.make_upper(n, 5)                      # well conditioned: X is unique to ~1e-13
        Vd = V.cuda()
        G = torch.empty(n, n, dtype=torch.float64, device="cuda")
        V1 = torch.empty_like(Vd)
        work = rq.alloc_workspace(m, n, max(n, 2), 2)
        rq.trsm_gram(Vd, R0.cuda(), G, V1, work)
        Xo = orc.trsm(V.numpy(), R0.numpy())
        Go = orc.gram(Xo)
        assert np.abs(host(V1) - Xo).max() <= 1e-12 * np.abs(Xo).max()
        assert np.linalg.norm(host(G) - Go) <= 1e-13 * np.linalg.norm(Go)
        assert torch.equal(G, G.T)
        # R0 = NULL: plain Gram; V1 = NULL: nothing stored; integer input: exact
        Vi = inputs.make_integer_V(m, n, 4)
        rq.trsm_gram(Vi.cuda(), None, G, None, work)
        assert np.array_equal(host(G), orc.gram(Vi.numpy()))
        # in place (V1 == V)
        Vc = Vd.clone()
        rq.trsm_gram(Vc, R0.cuda(), G, Vc, work)
        assert torch.equal(Vc, V1)
    finally:
        rq.force_generic(False)


@pytest.mark.parametrize("m,n", SHAPES_TALL)
@pytest.mark.parametrize("generic", [False, True])
def test_apply_parity_and_bit_identical_recompute(rq, orc, m, n, generic):
    rq.force_generic(generic)
    try:
        V = inputs.make_V(m, n, 1e3, 12) if m >= n else inputs.make_graded_V(m, n, 1, 12)
        R0 = inputs.make_upper(n, 6); R1 = inputs.make_upper(n, 7)
        Vd = V.cuda()
        G = torch.empty(n, n, dtype=torch.float64, device="cuda")
        V1 = torch.empty_like(Vd)
        work = rq.alloc_workspace(m, n, max(n, 2), 2)
        rq.trsm_gram(Vd, R0.cuda(), G, V1, work)
        Qa = torch.empty_like(Vd); Qb = torch.empty_like(Vd)
        rq.apply(V1, None, R1.cuda(), Qa, work)              # stored V1
        rq.apply(Vd, R0.cuda(), R1.cuda(), Qb, work)         # V1 re-formed inside
        assert torch.equal(Qa, Qb)                           # H1: same bits
        Qo = orc.trsm(orc.trsm(V.numpy(), R0.numpy()), R1.numpy())
        assert np.abs(host(Qa) - Qo).max() <= 1e-12 * np.abs(Qo).max()
        Vc = V1.clone()
        rq.apply(Vc, None, R1.cuda(), Vc, work)              # in place
        assert torch.equal(Vc, Qa)
    finally:
        rq.force_generic(False)


@pytest.mark.parametrize("m,n,pad", [(5003, 20, 4), (4099, 32, 2), (3001, 64, 8), (2500, 100, 6), (777, 10, 2)])
def test_strided_V_and_Q_take_the_per_row_staging(rq, orc, m, n, pad):
    """ld > n: the rows of an 8-row block are not contiguous, so the DMMA kernels stage them with one bulk copy per row
    (ld = n takes the one-copy-per-block mode, covered by the shapes above); both must give the oracle's X and G, and
    the same bits as the contiguous call."""
    V = inputs.make_V(m, n, 1e3, 13)
    R0 = inputs.make_upper(n, 5).cuda(); R1 = inputs.make_upper(n, 7).cuda()
    big = torch.zeros(m, n + pad, dtype=torch.float64, device="cuda")
    big[:, :n] = V.cuda()
    Vs = big[:, :n]                                   # ldv = n + pad
    qbig = torch.full((m, n + pad), float("nan"), dtype=torch.float64, device="cuda")
    Qs = qbig[:, :n]
    G = torch.empty(n, n, dtype=torch.float64, device="cuda")
    Gc = torch.empty_like(G)
    work = rq.alloc_workspace(m, n, max(n, 2), 2)
    rq.trsm_gram(Vs, R0, G, Qs, work)
    Vc = V.cuda(); X = torch.empty_like(Vc)
    rq.trsm_gram(Vc, R0, Gc, X, work)
    assert torch.equal(Qs, X) and torch.equal(G, Gc)
    assert bool(torch.isnan(qbig[:, n:]).all())       # nothing written past the n columns
    Xo = orc.trsm(V.numpy(), host(R0))
    assert np.abs(host(X) - Xo).max() <= 1e-12 * np.abs(Xo).max()
    rq.apply(Qs, None, R1, Qs, work)                  # in place, strided
    Qc = torch.empty_like(Vc)
    rq.apply(X, None, R1, Qc, work)
    assert torch.equal(Qs, Qc)
    rq.apply(Vs, R0, R1, Qs, work)                    # two-pass from the strided V
    assert torch.equal(Qs, Qc)


def test_trsm_rowwise_backward_error_with_graded_R(rq):
    # eq. (42): each row solves x (R + dR) = v with |dR| <= c n u |R|.
    # R0 = R factor of a column-graded matrix (12 decades), as randQR meets at kappa = 1e12.
    m, n = 3000, 64
    Rg = torch.linalg.qr(inputs.make_graded_V(500, n, 12, 8), mode="r").R
    Rg = (Rg * torch.sign(torch.diagonal(Rg))[:, None]).contiguous()
    X0 = inputs.make_graded_V(m, n, 0, 9)
    R0 = Rg.cuda()
    V = (X0 @ Rg).contiguous().cuda()
    for generic in (False, True):
        rq.force_generic(generic)
        try:
            G = torch.empty(n, n, dtype=torch.float64, device="cuda")
            V1 = torch.empty_like(V)
            work = rq.alloc_workspace(m, n, n, 2)
            rq.trsm_gram(V, R0, G, V1, work)
            resid = (V1 @ R0 - V).abs()
            bound = 16 * n * 2.0 ** -53 * (V1.abs() @ R0.abs())
            assert bool((resid <= bound + 1e-300).all())
            assert float(torch.linalg.norm(G - V1.T @ V1) / torch.linalg.norm(G)) <= 1e-13
        finally:
            rq.force_generic(False)


@pytest.mark.parametrize("n", [2, 16, 64, 70, 128, 129, 136, 200, 250, 256])
def test_chol_parity_and_failure(rq, orc, n):
    A = inputs.make_V(4 * n + 3, n, 30.0, n).numpy()
    Gm = A.T @ A
    R1 = torch.empty(n, n, dtype=torch.float64, device="cuda")
    info = rq.new_info()
    rq.chol(dev(Gm), R1, info)
    Ro, io = orc.chol(Gm)
    assert int(info.item()) == 0 and io == 0
    R = host(R1)
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R)) and (np.diag(R) > 0).all()
    assert np.linalg.norm(R - Ro) <= 1e-13 * np.linalg.norm(Ro)
    rq.chol(dev(Gm), R1, info, shift=0.75)
    Rs, _ = orc.chol(Gm, 0.75)
    assert np.linalg.norm(host(R1) - Rs) <= 1e-13 * np.linalg.norm(Rs)
    bad = Gm.copy(); j = n // 2; bad[j, j] = -1.0
    rq.chol(dev(bad), R1, info)
    _, io = orc.chol(bad)
    assert int(info.item()) == rq.INFO_NOT_SPD + j + 1 == io - orc.ORC_NOT_SPD + rq.INFO_NOT_SPD
    info.zero_()
    nan = Gm.copy(); nan[0, 0] = np.nan
    rq.chol(dev(nan), R1, info)
    assert int(info.item()) == rq.INFO_NOT_SPD + 1


@pytest.mark.parametrize("n", [2, 16, 70, 256])
def test_triu_mul_parity(rq, orc, n):
    R1 = inputs.make_upper(n, 1); R0 = inputs.make_upper(n, 2, 6)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    rq.triu_mul(R1.cuda(), R0.cuda(), R)
    Ro = orc.triu_mul(R1.numpy(), R0.numpy())
    assert np.abs(host(R) - Ro).max() <= 1e-15 * n * np.abs(Ro).max()
    assert np.array_equal(np.tril(host(R), -1), np.zeros((n, n)))


@pytest.mark.parametrize("rows,n", [(8192, 64), (2048, 32), (5000, 64), (129, 64), (128, 64), (1000, 16), (34277, 64),
                                    (103552, 64),      # = the largest row count the TSQR scratch takes at n = 64 (cap 1216)
                                    (77, 8)])
def test_tsqr_r_matches_householder(rq, orc, rows, n):
    """TSQR tree of 128-row Householder blocks vs the oracle's plain Householder QR of the whole matrix: R with a
    positive diagonal is unique, so the two agree norm-wise to rounding (graded columns: kappa ~ 1e10)."""
    rng = np.random.default_rng(rows + n)
    A = rng.standard_normal((rows, n)) * np.logspace(0, -10, n)
    R = torch.full((n, n), np.nan, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(max(rows, 2 * n * n), n, max(rows, n), 2 * n)
    info = rq.new_info()
    Ad = dev(A)
    rq.tsqr_r(Ad, R, work, info)
    Ro, io = orc.hhqr_r(A)
    assert int(info.item()) == 0 and io == 0
    Rh = host(R)
    assert np.array_equal(host(Ad), A)                      # A is not modified
    assert np.array_equal(np.tril(Rh, -1), np.zeros_like(Rh)) and (np.diag(Rh) > 0).all()
    assert np.linalg.norm(Rh - Ro) <= 1e-13 * np.linalg.norm(Ro)
    assert np.all(np.linalg.norm(Rh - Ro, axis=1) <= 1e-11 * np.linalg.norm(Ro, axis=1) + 1e-300)


# ---- N4: dense Rademacher S2 generated on the fly (reading S21) ----
@pytest.mark.parametrize("s1,s2", [(300, 5), (8192, 128), (129, 7), (40953, 789)])
def test_rademacher_signs_bit_exact(rq, orc, s1, s2):
    So = orc.rademacher_matrix(42, s2, s1)
    for row in sorted({0, 1, s2 // 2, s2 - 1}):
        sg = host(rq.debug_rademacher(42, s1, row, 0, s1))
        assert np.array_equal(sg, np.where(So[row] < 0, -1, 1).astype(np.int8))
    c0 = s1 // 3
    sg = host(rq.debug_rademacher(42, s1, s2 - 1, c0, s1 - c0))        # ragged start inside a 128-bit group
    assert np.array_equal(sg, np.where(So[s2 - 1, c0:] < 0, -1, 1).astype(np.int8))


@pytest.mark.parametrize("s1,n,s2", [(512, 16, 32), (8192, 64, 128), (9940, 70, 140), (300, 5, 7),
                                     (32768, 128, 256), (9984, 200, 401), (40953, 70, 789), (131072, 256, 512)])
def test_rademacher_sketch_parity(rq, orc, s1, n, s2):
    rng = np.random.default_rng(s1 + n)
    W1 = rng.standard_normal((s1, n))
    W = torch.empty(s2, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(s1, n, s1, s2, rq.S2_RADEMACHER)
    rq.gauss_sketch(dev(W1), s2, 42, W, work, rq.S2_RADEMACHER)
    Wo = orc.rademacher_sketch(W1, s2, 42)
    assert np.abs(host(W) - Wo).max() <= 1e-13 * np.abs(Wo).max()


@pytest.mark.parametrize("s1,n,s2", [(5000, 24, 64), (9000, 70, 256), (700, 9, 16)])
def test_rademacher_sketch_exact_on_integers(rq, orc, s1, n, s2):
    """s2 a power of 4: 1/sqrt(s2) is a power of two, so on integer data every +- sum is exact in any order and
    the split-K kernel must agree with the oracle to the last bit (a wrong sign or a dropped column cannot hide)."""
    rng = np.random.default_rng(s1)
    Wi = np.rint(rng.standard_normal((s1, n)) * 16)
    W = torch.empty(s2, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(s1, n, s1, s2, rq.S2_RADEMACHER)
    rq.gauss_sketch(dev(Wi), s2, 42, W, work, rq.S2_RADEMACHER)
    assert np.array_equal(host(W), orc.rademacher_sketch(Wi, s2, 42))


def test_rademacher_workspace_has_no_S2(rq):
    n, m = 256, 1 << 21
    s1, s2 = 2 * n * n, 2 * n
    full = rq.workspace_bytes(m, n, s1, s2, 0)
    lean = rq.workspace_bytes(m, n, s1, s2, rq.S2_RADEMACHER)
    assert full - lean >= 8 * s2 * s1                                  # the 512 MiB of S2 at n = 256
