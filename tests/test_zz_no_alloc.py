"""rqr_trsm_gram_noalloc (include/rqr.h): A4 with its Gram partials in the library's static device array, for callers
that cannot allocate.  Checked against the existing workspace path (rqr_trsm_gram) on two calls in a row, the second
on another shape so that the array still holds the first call's partials.  Collected last on purpose (file name)."""
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


def _pair(rq, V, R0, store):
    """(G, V1) of the workspace path and of the no-alloc path for the same inputs."""
    m, n = V.shape
    work = rq.alloc_workspace(m, n, max(n, 2), 2)
    Ga = torch.empty(n, n, dtype=torch.float64, device="cuda")
    Gb = torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda")
    Xa = torch.empty_like(V) if store else None
    Xb = torch.full_like(V, float("nan")) if store else None
    rq.trsm_gram(V, R0, Ga, Xa, work)
    rq.trsm_gram_noalloc(V, R0, Gb, Xb)
    torch.cuda.synchronize()
    return Ga, Xa, Gb, Xb


def _check(Ga, Xa, Gb, Xb, bitwise):
    # tolerance of tests/test_gpu_steps.py for sums: 1e-13 relative in the Frobenius norm
    assert float(torch.linalg.norm(Gb - Ga)) <= 1e-13 * float(torch.linalg.norm(Ga))
    assert torch.equal(Gb, Gb.T)
    if Xa is not None:
        assert torch.equal(Xa, Xb)          # the substitution is the same kernel, row by row
    if bitwise:
        assert torch.equal(Ga, Gb)          # DMMA path: same kernel, same grid, same reduction order


# (first call, second call): (m, n, with R0, store V1); the second shape differs so stale partials would show
CASES = [
    ((100003, 64, True, True), (4099, 64, True, False)),       # pair kernel, ragged tail; then few CTAs
    ((70001, 32, True, True), (300000, 16, False, False)),     # 4 column blocks; plain Gram with 2
    ((50000, 50, True, False), (9001, 24, True, True)),        # 7 and 3 column blocks (n not a multiple of 8)
    ((20001, 33, True, True), (20001, 63, False, False)),      # odd n: generic kernels, partial count capped at 148
]


@pytest.mark.parametrize("first,second", CASES)
def test_noalloc_matches_workspace_path_on_two_calls_in_a_row(rq, first, second):
    for k, (m, n, with_r0, store) in enumerate((first, second)):
        V = inputs.make_V(m, n, 1e3, 31 + k).cuda()
        R0 = inputs.make_upper(n, 9 + k).cuda() if with_r0 else None
        Ga, Xa, Gb, Xb = _pair(rq, V, R0, store and with_r0)
        _check(Ga, Xa, Gb, Xb, bitwise=(n % 2 == 0))
    # the same call again: the array now holds exactly this call's partials, the result may not move
    Gc = torch.empty_like(Gb)
    rq.trsm_gram_noalloc(V, R0, Gc, None)
    assert torch.equal(Gc, Gb)


def test_noalloc_against_fp64_matmul(rq):
    """Independent of the workspace path: integer data, where the Gram matrix is exact."""
    for m, n in [(65537, 64), (12345, 40)]:
        Vi = inputs.make_integer_V(m, n, 4).cuda()
        G = torch.empty(n, n, dtype=torch.float64, device="cuda")
        rq.trsm_gram_noalloc(Vi, None, G, None)
        assert torch.equal(G, Vi.T @ Vi)


def test_noalloc_in_place_and_strided(rq):
    m, n, ld = 30011, 48, 64
    buf = torch.zeros(m, ld, dtype=torch.float64, device="cuda")
    Vs = buf[:, :n]
    Vs.copy_(inputs.make_V(m, n, 1e3, 5).cuda())
    R0 = inputs.make_upper(n, 3).cuda()
    Vc = Vs.contiguous()
    work = rq.alloc_workspace(m, n, n, 2)
    Ga = torch.empty(n, n, dtype=torch.float64, device="cuda"); Xa = torch.empty_like(Vc)
    rq.trsm_gram(Vc, R0, Ga, Xa, work)
    Gb = torch.empty_like(Ga)
    rq.trsm_gram_noalloc(Vs, R0, Gb, Vs)            # strided input, V1 == V
    assert float(torch.linalg.norm(Gb - Ga)) <= 1e-13 * float(torch.linalg.norm(Ga))
    assert torch.equal(Vs, Xa)
    assert float(buf[:, n:].abs().max()) == 0.0     # nothing written past column n


def test_noalloc_rejects_shapes_beyond_its_scratch(rq):
    V = torch.zeros(128, 66, dtype=torch.float64, device="cuda")
    G = torch.zeros(66, 66, dtype=torch.float64, device="cuda")
    with pytest.raises(rq.RqrError, match="beyond the built-in scratch"):
        rq.trsm_gram_noalloc(V, None, G, None)
    L = rq.lib()
    st = torch.cuda.current_stream().cuda_stream
    # m beyond one chunk of rows: refused from the sizes alone, before anything is read or launched
    assert L.rqr_trsm_gram_noalloc(V.data_ptr(), rq.NOALLOC_MAX_M + 1, 64, 64, None, G.data_ptr(), None, 64, st) \
        == rq.ERR_SCRATCH_LIMIT
    assert L.rqr_trsm_gram_noalloc(V.data_ptr(), 128, rq.NOALLOC_MAX_N + 2, 66, None, G.data_ptr(), None, 66, st) \
        == rq.ERR_SCRATCH_LIMIT
    assert L.rqr_trsm_gram_noalloc(None, 128, 64, 64, None, G.data_ptr(), None, 64, st) == -1
    assert L.rqr_trsm_gram_noalloc(V.data_ptr(), 128, 64, 32, None, G.data_ptr(), None, 64, st) == -4
    assert L.rqr_trsm_gram_noalloc(V.data_ptr(), 128, 64, 64, None, None, None, 64, st) == -6
    torch.cuda.synchronize()


def test_noalloc_at_the_row_limit_allocates_nothing(rq):
    """m = RQR_NOALLOC_MAX_M (2^23 x 16, 1 GiB): accepted; torch's allocator sees no request during the call, and the
    driver's free memory does not move (the library calls no cudaMalloc)."""
    m, n = rq.NOALLOC_MAX_M, 16
    V = inputs.make_graded_V(m, n, 1, 3, device="cuda")
    G = torch.empty(n, n, dtype=torch.float64, device="cuda")
    Ga = torch.empty_like(G)
    work = rq.alloc_workspace(m, n, n, 2)
    rq.trsm_gram_noalloc(V, None, G, None)          # set-up call (symbol address, kernel attributes)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    n0 = torch.cuda.memory_stats()["allocation.all.allocated"]
    rq.trsm_gram_noalloc(V, None, G, None)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == n0
    assert free1 == free0
    rq.trsm_gram(V, None, Ga, None, work)
    assert torch.equal(G, Ga)
