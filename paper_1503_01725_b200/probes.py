"""Measurement probes (libpslmc_probe.so, csrc/probes/mem_probe.cu): the random-access ceilings bench.py and profiles/
compare the transport kernels with.  Not part of the product ABI; nothing in the hot path calls this."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libpslmc_probe.so")
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libpslmc_probe.so not built: run `python -m paper_1503_01725_b200.build`")
        L = C.CDLL(LIB_PATH)
        for f in (L.probe_red64, L.probe_gather32):
            f.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
        _lib = L
    return _lib


def _rate(fn, buf, n: int, n_ops: int, seed: int) -> float:
    out = np.zeros(2, np.float32)
    rc = fn(buf.data_ptr(), n, n_ops, seed, out.ctypes.data_as(C.c_void_p))
    if rc != 0:
        raise RuntimeError("probe failed: %d" % rc)
    return float(out[1]) / (float(out[0]) * 1e-3)


def red64_rate(nvox: int, n_ops: int = 1 << 28, seed: int = 1) -> float:
    """int64 scoring atomics per second on pseudo-random voxels of an nvox grid."""
    import torch
    return _rate(lib().probe_red64, torch.zeros(nvox, dtype=torch.int64, device="cuda"), nvox, n_ops, seed)


def gather32_rate(n_words: int, n_ops: int = 1 << 28, seed: int = 1) -> float:
    """random 4-byte gathers per second from a table of n_words words."""
    import torch
    return _rate(lib().probe_gather32, torch.ones(n_words, dtype=torch.int32, device="cuda"), n_words, n_ops, seed)
