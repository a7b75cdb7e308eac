"""Measurement aids that are not part of the product ABI: ``libmstar_benchaux.so`` (built beside
``libmstar_attn.so`` by ``paper_2606_12688_b200.build``) holds the read-only HBM streaming probe that
``bench.py`` times as the practical read ceiling.  Nothing in the hot path loads it."""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libmstar_benchaux.so")
_lib = None


def load_library() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("%s not found: build it with `python -m paper_2606_12688_b200.build`" % LIB_PATH)
        lib = ctypes.CDLL(LIB_PATH)
        lib.mstar_benchaux_hbm_read_probe.restype = ctypes.c_int
        lib.mstar_benchaux_hbm_read_probe.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p,
                                                      ctypes.c_void_p]
        _lib = lib
    return _lib


def hbm_read_probe(buf: torch.Tensor, nbytes: int, sum_out: Optional[torch.Tensor] = None) -> None:
    """Stream the first ``nbytes`` bytes of ``buf`` through 16-byte read-only loads; adds the wrapping sum of its
    32-bit words to ``sum_out`` (int64 [1], device) when given."""
    if not buf.is_cuda:
        raise RuntimeError("buf must be a CUDA tensor")
    if sum_out is not None and (not sum_out.is_cuda or sum_out.dtype != torch.int64):
        raise RuntimeError("sum_out must be a CUDA int64 tensor")
    rc = load_library().mstar_benchaux_hbm_read_probe(
        ctypes.c_void_p(buf.data_ptr()), int(nbytes), ctypes.c_void_p(0 if sum_out is None else sum_out.data_ptr()),
        ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != 0:
        raise RuntimeError("mstar_benchaux_hbm_read_probe failed (%d)" % rc)
