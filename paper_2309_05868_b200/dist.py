"""Row-sharded rand_cholQR over several GPUs (PAPER.md:228 footnote 3).

V and Q are split by block rows, one block per rank; S2 is replicated; S1 is split by the same
rows for free because bucket and sign are a function of the GLOBAL row index.  Exactly two
exchange steps: an all-reduce of W (s2 x n) and an all-reduce of G (n x n) -- "rand_cholQR
only requires two synchronizations total".  Everything else is the single-GPU step kernels.

`ops` is the step backend: the CUDA binding in production; the CPU tests plug an adapter with
the same method names so that the host-side sharding logic runs under gloo without a GPU.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_rows(m_total: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous block rows: returns (row0, rows) of this rank; sizes differ by at most 1."""
    base, rem = divmod(m_total, world)
    rows = base + (1 if rank < rem else 0)
    row0 = rank * base + min(rank, rem)
    return row0, rows


S2_RADEMACHER = 16      # same value as RQR_S2_RADEMACHER in include/rqr.h


def rand_cholqr_sharded(ops, V_local, row0, s1, s2, seed, Q_local, R, bufs, group=None, flags=0,
                        variant=0, m_total=None, fused=True):
    """One factorization step on this rank's block rows.  bufs: dict with W1 (s1 x n), W (s2 x n),
    R0, R1, G (n x n), work, info.  All ranks end with the same R; Q_local holds this rank's rows.
    variant | S2_RADEMACHER: the replicated S2 is the on-the-fly Rademacher sketch (N4): no rank stores it
    (bufs must come from alloc_bufs with the same variant).

    With the CUDA binding (`ops.rand_cholqr_sharded` exists) and fused=True this is ONE library call,
    rqr_rand_cholqr_sharded, with the two all-reduces issued from inside it through a callback on the same stream
    (CUDA-graph capturable); m_total (all ranks' rows) is then required unless there is one rank.  Otherwise the
    step entry points are called one by one (the CPU tests' adapter; fused=False on CUDA)."""
    multi = dist.is_initialized() and dist.get_world_size(group) > 1
    if fused and hasattr(ops, "rand_cholqr_sharded"):
        if m_total is None:
            assert not multi, "m_total is required with more than one rank"
            m_total = row0 + V_local.shape[0]
        ar = (lambda t: dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)) if multi else None
        ops.rand_cholqr_sharded(V_local, row0, m_total, s1, s2, seed, Q_local, R, bufs["work"], bufs["info"],
                                variant, flags, ar)
        return
    rad = variant & S2_RADEMACHER
    ops.countsketch(V_local, s1, seed, bufs["W1"], bufs["work"], variant, flags, row0)
    ops.gauss_sketch(bufs["W1"], s2, seed, bufs["W"], bufs["work"], flags | rad)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(bufs["W"], op=dist.ReduceOp.SUM, group=group)        # reduction 1
    ops.small_geqrf(bufs["W"], bufs["R0"], bufs["info"])
    ops.trsm_gram(V_local, bufs["R0"], bufs["G"], Q_local, bufs["work"])
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(bufs["G"], op=dist.ReduceOp.SUM, group=group)        # reduction 2
    ops.chol(bufs["G"], bufs["R1"], bufs["info"])
    ops.apply(Q_local, None, bufs["R1"], Q_local, bufs["work"])
    ops.triu_mul(bufs["R1"], bufs["R0"], R)


def alloc_bufs(ops, m_local, n, s1, s2, device, variant=0):
    f = dict(dtype=torch.float64, device=device)
    return {"W1": torch.empty(s1, n, **f), "W": torch.empty(s2, n, **f), "R0": torch.empty(n, n, **f),
            "R1": torch.empty(n, n, **f), "G": torch.empty(n, n, **f),
            "work": ops.alloc_workspace(m_local, n, s1, s2, variant), "info": ops.new_info()}
