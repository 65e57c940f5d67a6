"""Row-sharded rand_cholQR on the CUDA kernels (SURVEY.md 8(e); PAPER.md:208, :228 footnote 3), on ONE device: the
row shards run one after the other, and the sum over the shards of W and of G is formed on the device in place of the
all-reduce.  What is checked: bucket / sign follow the GLOBAL row index (row0 > 0), the two reductions are the only
exchange, every "rank" ends with the same R, and the stacked Q meets the north_star bars and the oracle's R."""
import numpy as np
import pytest
import torch

from paper_2309_05868_b200 import dist as rdist, inputs

pytestmark = pytest.mark.gpu

ORTH_TOL, RES_TOL, R_TOL = 1e-12, 1e-13, 1e-9


@pytest.fixture(scope="module")
def rq():
    from paper_2309_05868_b200 import binding
    binding.lib()
    assert torch.cuda.is_available()
    return binding


def one_shot(rq, Vd, s1, s2, seed):
    m, n = Vd.shape
    Q = torch.empty_like(Vd)
    R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    work = rq.alloc_workspace(m, n, s1, s2)
    info = rq.new_info()
    rq.rand_cholqr(Vd, s1, s2, seed, Q, R, work, info)
    assert int(info.item()) == 0
    return Q, R


@pytest.mark.parametrize("m,n,kappa,cuts", [(150001, 64, 1e12, (0, 70003, 150001)),
                                            (90000, 32, 1e10, (0, 17, 50000, 90000)),        # a shard with fewer than n rows
                                            (80000, 128, 1e8, (0, 40001, 80000))])
def test_two_row_shards_on_one_device(rq, orc, m, n, kappa, cuts):
    s1, s2 = inputs.sketch_sizes(n)
    seed = 42
    V = inputs.make_V(m, n, kappa, 21)
    Vd = V.cuda()
    shards = [(cuts[i], cuts[i + 1] - cuts[i]) for i in range(len(cuts) - 1)]
    f = dict(dtype=torch.float64, device="cuda")
    # --- pass 1: every shard's local sketch W_k = S2 (S1)_k V_k with its own prepared workspace (row0 = first row)
    st = []
    Wk = []
    for row0, rows in shards:
        bufs = rdist.alloc_bufs(rq, rows, n, s1, s2, "cuda")
        rq.sketch_prepare(rows, n, s1, s2, seed, bufs["work"], 0, row0)
        Vl = Vd[row0: row0 + rows]
        rq.countsketch(Vl, s1, seed, bufs["W1"], bufs["work"], 0, rq.FLAG_PREPARED, row0)
        rq.gauss_sketch(bufs["W1"], s2, seed, bufs["W"], bufs["work"], rq.FLAG_PREPARED)
        Wk.append(bufs["W"].clone())
        st.append((row0, rows, Vl, bufs))
    W = torch.zeros(s2, n, **f)
    for w in Wk:                                # the all-reduce: a sum over the shards in rank order
        W += w
    # the sum of the local sketches is the sketch of the whole matrix (same buckets and signs as the one-shot's)
    Wo = orc.gauss_sketch(orc.countsketch(V.numpy(), s1, seed), s2, seed)
    assert np.abs(W.cpu().numpy() - Wo).max() <= 1e-13 * np.abs(Wo).max()
    # --- pass 2: redundant Householder QR, local trsm + Gram, second reduction
    G = torch.zeros(n, n, **f)
    Gk = []
    Qs = torch.empty_like(Vd)
    for row0, rows, Vl, b in st:
        b["W"].copy_(W)
        rq.small_geqrf(b["W"], b["R0"], b["info"])
        rq.trsm_gram(Vl, b["R0"], b["G"], Qs[row0: row0 + rows], b["work"])
        Gk.append(b["G"].clone())
        G += b["G"]
    Rs = []
    for row0, rows, Vl, b in st:
        rq.chol(G, b["R1"], b["info"])
        Ql = Qs[row0: row0 + rows]
        rq.apply(Ql, None, b["R1"], Ql, b["work"])
        R = torch.empty(n, n, **f)
        rq.triu_mul(b["R1"], b["R0"], R)
        assert int(b["info"].item()) == 0
        Rs.append(R)
    for R in Rs[1:]:
        assert torch.equal(R, Rs[0])            # every rank holds the same R
    R = Rs[0]
    eye = torch.eye(n, **f)
    assert float(torch.linalg.norm(Qs.T @ Qs - eye)) <= ORTH_TOL
    assert float(torch.linalg.norm(Vd - Qs @ R) / torch.linalg.norm(Vd)) <= RES_TOL
    _, Ro, io = orc.rand_cholqr(V.numpy(), s1, s2, seed)
    assert io == 0
    assert np.linalg.norm(R.cpu().numpy() - Ro) <= R_TOL * np.linalg.norm(Ro)
    # against the single-device one-shot: same sketch operator, so R agrees to summation-order rounding
    Q1, R1 = one_shot(rq, Vd, s1, s2, seed)
    assert float(torch.linalg.norm(R - R1) / torch.linalg.norm(R1)) <= 1e-12

    # --- the C-ABI sharded one-shot (rqr_rand_cholqr_sharded), shard by shard.  Its all-reduce callback stands in
    # for the other ranks: it checks that the library hands over THIS shard's W_k / G_k (as computed above with the
    # step entry points) and returns the rank-order sums W and G -- what a real all-reduce gives every rank.
    for k, (row0, rows, Vl, b) in enumerate(st):
        calls = []

        def allreduce(t, k=k):
            mine, total = (Wk[k], W) if not calls else (Gk[k], G)
            calls.append(t.numel())
            assert t.numel() == total.numel()
            assert float(torch.linalg.norm(t - mine.reshape(-1))) <= 1e-14 * float(torch.linalg.norm(mine))
            t.copy_(total.reshape(-1))
        Qk = torch.empty(rows, n, **f)
        Rk = torch.empty(n, n, **f)
        rq.rand_cholqr_sharded(Vl, row0, m, s1, s2, seed, Qk, Rk, b["work"], b["info"], 0, rq.FLAG_PREPARED, allreduce)
        assert int(b["info"].item()) == 0 and calls == [s2 * n, n * n]
        assert float(torch.linalg.norm(Rk - R) / torch.linalg.norm(R)) <= 1e-13
        # same W, same G, same kernels: this shard's rows of Q are those of the step-by-step run (H1: stored or
        # recomputed V1 give the same bits)
        Ql = Qs[row0: row0 + rows]
        assert float((Qk - Ql).abs().max()) <= 1e-14 * float(Ql.abs().max())


def test_sharded_one_rank_equals_the_one_shot(rq):
    """allreduce == NULL, row0 = 0, m_total = m: the sharded entry point is the one-shot, bit for bit, and it is
    CUDA-graph capturable (bench.py --force-sharded times it that way)."""
    m, n = 120000, 64
    s1, s2 = inputs.sketch_sizes(n)
    Vd = inputs.make_V(m, n, 1e12, 8).cuda()
    Q1, R1 = one_shot(rq, Vd, s1, s2, 42)
    Q = torch.empty_like(Vd); R = torch.empty(n, n, dtype=torch.float64, device="cuda")
    bufs = rdist.alloc_bufs(rq, m, n, s1, s2, "cuda")
    rq.sketch_prepare(m, n, s1, s2, 42, bufs["work"])
    rdist.rand_cholqr_sharded(rq, Vd, 0, s1, s2, 42, Q, R, bufs, None, rq.FLAG_PREPARED, 0)
    assert int(bufs["info"].item()) == 0 and torch.equal(Q, Q1) and torch.equal(R, R1)
    Q.zero_(); R.zero_()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            rdist.rand_cholqr_sharded(rq, Vd, 0, s1, s2, 42, Q, R, bufs, None, rq.FLAG_PREPARED, 0)
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(Q, Q1) and torch.equal(R, R1)
    # the step-by-step form of dist.py (what the gloo tests drive with the CPU adapter) on the CUDA kernels
    rdist.rand_cholqr_sharded(rq, Vd, 0, s1, s2, 42, Q, R, bufs, None, rq.FLAG_PREPARED, 0, fused=False)
    # (A7 is its own kernel there, fused into the Cholesky kernel in the one-shot: R may differ in the last bits)
    assert int(bufs["info"].item()) == 0 and torch.equal(Q, Q1)
    assert float(torch.linalg.norm(R - R1) / torch.linalg.norm(R1)) <= 1e-15
