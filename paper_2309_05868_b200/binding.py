"""Thin Python binding of librqr (include/rqr.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch supplies device memory and the
current stream.  There is no CPU fallback: if librqr.so is missing or a tensor is not on a CUDA
device the call raises.  Names match the C ABI without the rqr_ prefix.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librqr.so")

OK = 0
INFO_NOT_SPD = 1000
INFO_SINGULAR = 2000
VARIANT_SORTED = 0
VARIANT_SCATTER = 1
VARIANT_STREAM = 2
FLAG_PREPARED = 1
FLAG_RECOMPUTE_V1 = 2
FLAG_STORE_V1 = 4
S2_RADEMACHER = 16          # OR into `variant` (workspace, prepare, countsketch, rand_cholqr) / `flags` (gauss_sketch)
MAX_N = 256                 # argument limits of include/rqr.h
MAX_S2 = 1024
ERR_SCRATCH_LIMIT = -1002   # rqr_trsm_gram_noalloc: shape beyond its built-in scratch
NOALLOC_MAX_N = 64
NOALLOC_MAX_M = 1 << 23

_i64, _u64, _u32, _int, _dbl, _vp, _sz = (ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int,
                                          ctypes.c_double, ctypes.c_void_p, ctypes.c_size_t)

# name -> (restype, argtypes); mirrors include/rqr.h
SIGNATURES = {
    "rqr_workspace_bytes": (_sz, [_i64, _int, _i64, _int, _int]),
    "rqr_sketch_prepare": (_int, [_i64, _int, _i64, _i64, _int, _u64, _int, _vp, _vp]),
    "rqr_countsketch": (_int, [_vp, _i64, _int, _i64, _i64, _i64, _u64, _vp, _vp, _int, _int, _vp]),
    "rqr_gauss_sketch": (_int, [_vp, _i64, _int, _int, _u64, _vp, _vp, _int, _vp]),
    "rqr_small_geqrf": (_int, [_vp, _int, _int, _vp, _vp, _vp]),
    "rqr_trsm_gram": (_int, [_vp, _i64, _int, _i64, _vp, _vp, _vp, _i64, _vp, _vp]),
    "rqr_trsm_gram_noalloc": (_int, [_vp, _i64, _int, _i64, _vp, _vp, _vp, _i64, _vp]),
    "rqr_chol": (_int, [_vp, _int, _dbl, _vp, _vp, _vp]),
    "rqr_apply": (_int, [_vp, _i64, _int, _i64, _vp, _vp, _vp, _i64, _vp, _vp]),
    "rqr_triu_mul": (_int, [_vp, _vp, _int, _vp, _vp]),
    "rqr_rand_cholqr": (_int, [_vp, _i64, _int, _i64, _int, _u64, _vp, _vp, _vp, _vp, _int, _int, _vp]),
    "rqr_rand_cholqr_sharded": (_int, [_vp, _i64, _i64, _i64, _int, _i64, _int, _u64, _vp, _vp, _vp, _vp, _int, _int, _vp,
                                       _vp, _vp]),
    "rqr_rand_cholqr_batched": (_int, [_vp, _i64, _int, _int, _i64, _i64, _int, _u64, _vp, _i64, _vp, _vp, _vp, _int, _int,
                                       _vp]),
    "rqr_cholqr2": (_int, [_vp, _i64, _int, _vp, _vp, _vp, _vp, _vp]),
    "rqr_scholqr3": (_int, [_vp, _i64, _int, _vp, _vp, _vp, _vp, _vp]),
    "rqr_gauss_randcholqr": (_int, [_vp, _i64, _int, _int, _u64, _vp, _vp, _vp, _vp, _vp]),
    "rqr_count_randcholqr": (_int, [_vp, _i64, _int, _i64, _u64, _vp, _vp, _vp, _vp, _int, _int, _vp]),
    "rqr_tsqr_r": (_int, [_vp, _i64, _int, _vp, _vp, _vp, _vp]),
    "rqr_dense_gauss_sketch": (_int, [_vp, _i64, _int, _i64, _i64, _i64, _int, _u64, _vp, _vp, _vp]),
    "rqr_debug_dense_gauss_draw_only": (_int, [_i64, _int, _int, _u64, _vp, _vp]),
    "rqr_debug_hash_sign": (_int, [_u64, _i64, _i64, _i64, _vp, _vp, _vp]),
    "rqr_debug_gauss": (_int, [_u64, _u32, _u64, _i64, _vp, _vp]),
    "rqr_workspace_S2": (_vp, [_vp, _int, _i64]),
    "rqr_workspace_rows": (_int, [_vp, _i64, _int, _i64, _int, _vp, _vp]),
    "rqr_workspace_scholqr3_shift": (_vp, [_vp]),
    "rqr_debug_rademacher": (_int, [_u64, _i64, _int, _i64, _i64, _vp, _vp]),
    "rqr_debug_trsm_gram_generic": (_int, [_vp, _i64, _int, _i64, _vp, _vp, _vp, _i64, _vp, _vp]),
    "rqr_debug_apply_generic": (_int, [_vp, _i64, _int, _i64, _vp, _vp, _vp, _i64, _vp, _vp]),
    "rqr_version": (ctypes.c_char_p, []),
}

_lib = None


def lib():
    """Loads librqr.so; raises loudly if it is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("librqr.so not built: run __graft_entry__.build() "
                               "(python -m paper_2309_05868_b200.build); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


class RqrError(RuntimeError):
    pass


def _chk(rc, name):
    if rc != OK:
        raise RqrError("%s returned %d (%s)" % (name, rc, "argument %d invalid" % -rc if rc > -1000 else "launch failed"))


def _ptr(t):
    if t is None:
        return None
    if not t.is_cuda:
        raise RqrError("librqr needs CUDA tensors (no CPU fallback)")
    return t.data_ptr()


def _f64(t, name):
    if t.dtype != torch.float64 or not t.is_cuda:
        raise RqrError("%s must be a CUDA float64 tensor" % name)
    return t


def _stream():
    return torch.cuda.current_stream().cuda_stream


def version() -> str:
    return lib().rqr_version().decode()


def workspace_bytes(m, n, s1, s2, variant=VARIANT_SORTED) -> int:
    b = int(lib().rqr_workspace_bytes(m, n, s1, s2, variant))
    if b == 0:
        raise RqrError("rqr_workspace_bytes: invalid shape")
    return b


def alloc_workspace(m, n, s1, s2, variant=VARIANT_SORTED, device="cuda"):
    return torch.empty(workspace_bytes(m, n, s1, s2, variant), dtype=torch.uint8, device=device)


def new_info(device="cuda"):
    return torch.zeros(1, dtype=torch.int32, device=device)


def sketch_prepare(m, n, s1, s2, seed, work, variant=VARIANT_SORTED, row0=0):
    _chk(lib().rqr_sketch_prepare(m, n, row0, s1, s2, seed, variant, _ptr(work), _stream()), "rqr_sketch_prepare")


def countsketch(V, s1, seed, W1, work, variant=VARIANT_SORTED, flags=0, row0=0):
    _f64(V, "V"); _f64(W1, "W1")
    m, n = V.shape
    _chk(lib().rqr_countsketch(_ptr(V), m, n, V.stride(0), row0, s1, seed, _ptr(W1), _ptr(work), variant,
                               flags, _stream()), "rqr_countsketch")


def gauss_sketch(W1, s2, seed, W, work, flags=0):
    _f64(W1, "W1"); _f64(W, "W")
    s1, n = W1.shape
    _chk(lib().rqr_gauss_sketch(_ptr(W1), s1, n, s2, seed, _ptr(W), _ptr(work), flags, _stream()), "rqr_gauss_sketch")


def small_geqrf(W, R0, info=None):
    _f64(W, "W"); _f64(R0, "R0")
    s2, n = W.shape
    _chk(lib().rqr_small_geqrf(_ptr(W), s2, n, _ptr(R0), _ptr(info), _stream()), "rqr_small_geqrf")


def trsm_gram(V, R0, G, V1, work):
    _f64(V, "V"); _f64(G, "G")
    m, n = V.shape
    ldq = V1.stride(0) if V1 is not None else n
    f = lib().rqr_debug_trsm_gram_generic if _force_generic else lib().rqr_trsm_gram
    _chk(f(_ptr(V), m, n, V.stride(0), _ptr(R0), _ptr(G), _ptr(V1), ldq, _ptr(work), _stream()), "rqr_trsm_gram")


def trsm_gram_noalloc(V, R0, G, V1):
    """rqr_trsm_gram without a workspace: the Gram partials live in the library's own static device array
    (n <= 64, m <= 2^23; calls that overlap on the GPU race on it).  Allocates nothing."""
    _f64(V, "V"); _f64(G, "G")
    m, n = V.shape
    ldq = V1.stride(0) if V1 is not None else n
    rc = lib().rqr_trsm_gram_noalloc(_ptr(V), m, n, V.stride(0), _ptr(R0), _ptr(G), _ptr(V1), ldq, _stream())
    if rc == ERR_SCRATCH_LIMIT:
        raise RqrError("rqr_trsm_gram_noalloc: shape %d x %d is beyond the built-in scratch (n <= %d, m <= %d); "
                       "use rqr_trsm_gram with a workspace" % (m, n, NOALLOC_MAX_N, NOALLOC_MAX_M))
    _chk(rc, "rqr_trsm_gram_noalloc")


def chol(G, R1, info=None, shift=0.0):
    _f64(G, "G"); _f64(R1, "R1")
    _chk(lib().rqr_chol(_ptr(G), G.shape[0], float(shift), _ptr(R1), _ptr(info), _stream()), "rqr_chol")


def apply(V, R0, R1, Q, work=None):
    _f64(V, "V"); _f64(Q, "Q")
    m, n = V.shape
    f = lib().rqr_debug_apply_generic if _force_generic else lib().rqr_apply
    _chk(f(_ptr(V), m, n, V.stride(0), _ptr(R0), _ptr(R1), _ptr(Q), Q.stride(0), _ptr(work), _stream()), "rqr_apply")


def triu_mul(R1, R0, R):
    _chk(lib().rqr_triu_mul(_ptr(R1), _ptr(R0), R1.shape[0], _ptr(R), _stream()), "rqr_triu_mul")


def rand_cholqr(V, s1, s2, seed, Q, R, work, info, variant=VARIANT_SORTED, flags=0):
    _f64(V, "V"); _f64(Q, "Q"); _f64(R, "R")
    m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous()
    _chk(lib().rqr_rand_cholqr(_ptr(V), m, n, s1, s2, seed, _ptr(Q), _ptr(R), _ptr(work), _ptr(info), variant, flags,
                               _stream()), "rqr_rand_cholqr")


ALLREDUCE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p)


def rand_cholqr_sharded(V, row0, m_total, s1, s2, seed, Q, R, work, info, variant=VARIANT_SORTED, flags=0,
                        allreduce=None):
    """Row-sharded one-shot on this rank's rows.  `allreduce(t)` sums the float64 device tensor t in place over the
    ranks on torch's current stream (e.g. torch.distributed.all_reduce); the library hands it W (s2 x n) and G
    (n x n), both views into `work`.  None: one rank."""
    _f64(V, "V"); _f64(Q, "Q"); _f64(R, "R")
    m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous()
    base = work.data_ptr()
    err = []

    def _cb(ctx, buf, count, stream):
        try:
            off = buf - base
            allreduce(work[off: off + 8 * count].view(torch.float64))
            return 0
        except BaseException as e:              # an exception must not unwind through the C frames
            err.append(e)
            return 1
    cb = ALLREDUCE_FN(_cb) if allreduce is not None else None
    rc = lib().rqr_rand_cholqr_sharded(_ptr(V), m, row0, m_total, n, s1, s2, seed, _ptr(Q), _ptr(R), _ptr(work),
                                       _ptr(info), variant, flags, cb, None, _stream())
    if err:
        raise err[0]
    _chk(rc, "rqr_rand_cholqr_sharded")


def rand_cholqr_batched(V, s1, s2, seed, Q, R, work, info, variant=VARIANT_SORTED, flags=0):
    """V, Q: (batch, m, n) contiguous; R: (batch, n, n); info: (batch,) int32."""
    _f64(V, "V"); _f64(Q, "Q"); _f64(R, "R")
    batch, m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous() and R.is_contiguous() and info.numel() >= batch
    _chk(lib().rqr_rand_cholqr_batched(_ptr(V), m, n, batch, m * n, s1, s2, seed, _ptr(Q), m * n, _ptr(R), _ptr(work),
                                       _ptr(info), variant, flags, _stream()), "rqr_rand_cholqr_batched")


def cholqr2(V, Q, R, work, info):
    m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous()
    _chk(lib().rqr_cholqr2(_ptr(_f64(V, "V")), m, n, _ptr(Q), _ptr(R), _ptr(work), _ptr(info), _stream()), "rqr_cholqr2")


def scholqr3(V, Q, R, work, info):
    m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous()
    _chk(lib().rqr_scholqr3(_ptr(_f64(V, "V")), m, n, _ptr(Q), _ptr(R), _ptr(work), _ptr(info), _stream()), "rqr_scholqr3")


def gauss_randcholqr(V, s, seed, Q, R, work, info):
    m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous()
    _chk(lib().rqr_gauss_randcholqr(_ptr(_f64(V, "V")), m, n, s, seed, _ptr(Q), _ptr(R), _ptr(work), _ptr(info),
                                    _stream()), "rqr_gauss_randcholqr")


def count_randcholqr(V, s1, seed, Q, R, work, info, variant=VARIANT_SORTED, flags=0):
    m, n = V.shape
    assert V.is_contiguous() and Q.is_contiguous()
    _chk(lib().rqr_count_randcholqr(_ptr(_f64(V, "V")), m, n, s1, seed, _ptr(Q), _ptr(R), _ptr(work), _ptr(info),
                                    variant, flags, _stream()), "rqr_count_randcholqr")


def tsqr_r(A, R, work, info=None):
    rows, n = A.shape
    assert A.is_contiguous()
    _chk(lib().rqr_tsqr_r(_ptr(_f64(A, "A")), rows, n, _ptr(R), _ptr(work), _ptr(info), _stream()), "rqr_tsqr_r")


def dense_gauss_sketch(V, s, seed, W, work, row0=0, m_total=None):
    m, n = V.shape
    _chk(lib().rqr_dense_gauss_sketch(_ptr(_f64(V, "V")), m, n, V.stride(0), row0, m if m_total is None else m_total,
                                      s, seed, _ptr(W), _ptr(work), _stream()), "rqr_dense_gauss_sketch")


def debug_dense_gauss_draw_only(m, n, s, seed, work):
    _chk(lib().rqr_debug_dense_gauss_draw_only(m, n, s, seed, _ptr(work), _stream()), "rqr_debug_dense_gauss_draw_only")


def debug_hash_sign(seed, row0, count, s1, device="cuda"):
    b = torch.empty(count, dtype=torch.int32, device=device)      # holds uint32 bit patterns (< 2^31)
    s = torch.empty(count, dtype=torch.int8, device=device)
    _chk(lib().rqr_debug_hash_sign(seed, row0, count, s1, _ptr(b), _ptr(s), _stream()), "rqr_debug_hash_sign")
    return b, s


def debug_gauss(seed, stream_id, first, count, device="cuda"):
    z = torch.empty(count, dtype=torch.float64, device=device)
    _chk(lib().rqr_debug_gauss(seed, stream_id, first, count, _ptr(z), _stream()), "rqr_debug_gauss")
    return z


def debug_rademacher(seed, s1, row, c0, count, device="cuda"):
    sg = torch.empty(count, dtype=torch.int8, device=device)
    _chk(lib().rqr_debug_rademacher(seed, s1, row, c0, count, _ptr(sg), _stream()), "rqr_debug_rademacher")
    return sg


def workspace_S2(work, n, s1, s2):
    """View of S2 (s2 x s1) inside a prepared workspace."""
    base = lib().rqr_workspace_S2(_ptr(work), n, s1)
    off = base - work.data_ptr()
    ld = (s1 + 15) & ~15                  # rows are padded with zeros to a multiple of 16 doubles
    return work[off: off + s2 * ld * 8].view(torch.float64).view(s2, ld)[:, :s1]


def workspace_rows(work, m, n, s1, variant=VARIANT_SORTED):
    """Views of the bucket offsets (s1 + 1, int32 bit patterns) and the sorted row list (m, int32 bit patterns of
    uint32 row | sign << 31) inside a prepared workspace."""
    po, pe = ctypes.c_void_p(0), ctypes.c_void_p(0)
    _chk(lib().rqr_workspace_rows(_ptr(work), m, n, s1, variant, ctypes.byref(po), ctypes.byref(pe)), "rqr_workspace_rows")
    o0, e0 = po.value - work.data_ptr(), pe.value - work.data_ptr()
    return work[o0: o0 + 4 * (s1 + 1)].view(torch.int32), work[e0: e0 + 4 * m].view(torch.int32)


def workspace_scholqr3_shift(work):
    off = lib().rqr_workspace_scholqr3_shift(_ptr(work)) - work.data_ptr()
    return work[off: off + 8].view(torch.float64)


_force_generic = False


def force_generic(on: bool):
    """Test hook (binding-side switch, no state in the library): trsm_gram / apply call the library's
    rqr_debug_*_generic entry points, which run the generic (non-DMMA) kernels."""
    global _force_generic
    _force_generic = bool(on)
