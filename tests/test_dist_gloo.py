"""World-size-2 CPU test (gloo) of the row-sharded driver paper_2309_05868_b200/dist.py
(PAPER.md:228 footnote 3: block rows per process, one reduction for W and one for G; "only
requires two synchronizations").  The step backend is an adapter over the CPU oracle with the binding's
method names, so the host-side sharding logic (row offsets into the global hash, the two all-reduces,
buffer plumbing) runs without a GPU."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2309_05868_b200 import dist as rdist, inputs


class OracleOps:
    """binding.py's step names on CPU tensors, arithmetic by oracle/ (test infrastructure)."""

    def __init__(self):
        from oracle import rqr_oracle
        rqr_oracle.build()
        self.o = rqr_oracle

    def alloc_workspace(self, m, n, s1, s2, variant=0):
        return torch.empty(1, dtype=torch.uint8)

    def new_info(self):
        return torch.zeros(1, dtype=torch.int32)

    def countsketch(self, V, s1, seed, W1, work, variant=0, flags=0, row0=0):
        assert (variant & ~rdist.S2_RADEMACHER) in (0, 1)
        W1.copy_(torch.from_numpy(self.o.countsketch(V.numpy(), s1, seed, row0=row0)))

    def gauss_sketch(self, W1, s2, seed, W, work, flags=0):
        sk = self.o.rademacher_sketch if flags & rdist.S2_RADEMACHER else self.o.gauss_sketch
        W.copy_(torch.from_numpy(sk(W1.numpy(), s2, seed)))

    def small_geqrf(self, W, R0, info=None):
        R, st = self.o.hhqr_r(W.numpy())
        R0.copy_(torch.from_numpy(R))
        if st and info is not None and int(info) == 0:
            info.fill_(st)

    def trsm_gram(self, V, R0, G, V1, work):
        X = self.o.trsm(V.numpy(), R0.numpy()) if R0 is not None else V.numpy()
        G.copy_(torch.from_numpy(self.o.gram(X)))
        if V1 is not None:
            V1.copy_(torch.from_numpy(X))

    def chol(self, G, R1, info=None, shift=0.0):
        R, st = self.o.chol(G.numpy(), shift)
        R1.copy_(torch.from_numpy(R))
        if st and info is not None and int(info) == 0:
            info.fill_(st)

    def apply(self, V, R0, R1, Q, work=None):
        X = V.numpy()
        if R0 is not None:
            X = self.o.trsm(X, R0.numpy())
        Q.copy_(torch.from_numpy(self.o.trsm(X, R1.numpy())))

    def triu_mul(self, R1, R0, R):
        R.copy_(torch.from_numpy(self.o.triu_mul(R1.numpy(), R0.numpy())))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, m, n, kappa, s1, s2, seed, out_dir, variant=0):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.set_num_threads(1)
    ops = OracleOps()
    V = inputs.make_V(m, n, kappa, 77)              # same matrix on every rank, each takes its rows
    row0, rows = rdist.shard_rows(m, world, rank)
    Vl = V[row0:row0 + rows].contiguous()
    Q = torch.empty_like(Vl)
    R = torch.empty(n, n, dtype=torch.float64)
    bufs = rdist.alloc_bufs(ops, rows, n, s1, s2, "cpu", variant)
    rdist.rand_cholqr_sharded(ops, Vl, row0, s1, s2, seed, Q, R, bufs, variant=variant)
    np.save(os.path.join(out_dir, "Q%d.npy" % rank), Q.numpy())
    np.save(os.path.join(out_dir, "R%d.npy" % rank), R.numpy())
    np.save(os.path.join(out_dir, "info%d.npy" % rank), bufs["info"].numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_shard_rows_partition():
    for m, w in [(10, 3), (7, 7), (1 << 20, 8), (5, 2)]:
        blocks = [rdist.shard_rows(m, w, r) for r in range(w)]
        assert blocks[0][0] == 0 and sum(b[1] for b in blocks) == m
        for a, b in zip(blocks, blocks[1:]):
            assert a[0] + a[1] == b[0]
        assert max(b[1] for b in blocks) - min(b[1] for b in blocks) <= 1


@pytest.mark.timeout(300)
@pytest.mark.parametrize("variant", [0, rdist.S2_RADEMACHER])
def test_row_sharded_rand_cholqr_world2(tmp_path, orc, variant):
    m, n, kappa, seed = 6001, 12, 1e9, 42           # odd m: unequal blocks
    s1, s2 = 2 * n * n, 2 * n
    port = _free_port()
    mp.spawn(_worker, args=(2, port, m, n, kappa, s1, s2, seed, str(tmp_path), variant), nprocs=2, join=True)
    R0_, R1_ = np.load(tmp_path / "R0.npy"), np.load(tmp_path / "R1.npy")
    assert np.array_equal(R0_, R1_)                 # all-reduce gives every rank the same W and G
    assert int(np.load(tmp_path / "info0.npy")[0]) == 0
    Q = np.concatenate([np.load(tmp_path / "Q0.npy"), np.load(tmp_path / "Q1.npy")])
    V = inputs.make_V(m, n, kappa, 77).numpy()
    assert np.linalg.norm(Q.T @ Q - np.eye(n)) <= 1e-12
    assert np.linalg.norm(V - Q @ R0_) / np.linalg.norm(V) <= 1e-13
    assert np.all(np.diag(R0_) > 0) and np.array_equal(np.tril(R0_, -1), np.zeros((n, n)))
    # against the single-process oracle on the whole matrix: same hash (global row index), same S2
    _, Rs, info = orc.rand_cholqr(V, s1, s2, seed, rademacher=bool(variant))
    assert info == 0
    assert np.linalg.norm(R0_ - Rs) / np.linalg.norm(Rs) <= 1e-12
