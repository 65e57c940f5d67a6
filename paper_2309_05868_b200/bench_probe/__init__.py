"""Bench-only FP64 peak probe (librqr_probe.so): register-resident DFMA / DMMA chains timed by the caller with CUDA
events.  Used by bench.py and the sweep scripts for the roofline denominator; the library (librqr.so) does not
contain it and nothing in the library or the tests' parity path depends on it."""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(os.path.dirname(_HERE), "librqr_probe.so")
DFMA, DMMA, MIX = 0, 1, 2
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("librqr_probe.so not built: run __graft_entry__.build()")
        L = ctypes.CDLL(LIB_PATH)
        L.rqr_probe_fp64.restype = ctypes.c_int
        L.rqr_probe_fp64.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                     ctypes.c_void_p]
        _lib = L
    return _lib


def probe_fp64(kind, iters, blocks, sink):
    """Launches one probe kernel on torch's current stream; returns the flop count of the launch."""
    import torch
    fl = ctypes.c_double(0.0)
    rc = lib().rqr_probe_fp64(kind, iters, blocks, sink.data_ptr(), ctypes.addressof(fl),
                              torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError("rqr_probe_fp64 returned %d" % rc)
    return fl.value
