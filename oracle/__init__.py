"""ctypes front end of the CPU oracle (``mstar_oracle.c``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2606_12688_b200`` and the product never imports it.

Arrays are numpy; bf16 tensors travel as ``uint16`` bit patterns.  Pools are
``[num_pages, Hkv, page_size, D]`` (a *compact store* with a remapped block table is a valid
pool: the definition depends on physical page ids only through the data they hold).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mstar_oracle.c")
_LIB = os.path.join(_HERE, "libmstar_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over independent rows, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
        for name in ("oracle_paged_decode", "oracle_decode_probs", "oracle_paged_prefill_rows",
                     "oracle_decode_partition"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def _geom(k_pool):
    assert k_pool.ndim == 4
    _, Hkv, p, D = k_pool.shape
    return int(Hkv), int(p), int(D)


def kv_append(k_pool, v_pool, k_new, v_new, slot_mapping):
    """APPEND in place on ``k_pool`` / ``v_pool`` (uint16, C-contiguous)."""
    lib = _load()
    assert k_pool.dtype == np.uint16 and v_pool.dtype == np.uint16
    assert k_pool.flags.c_contiguous and v_pool.flags.c_contiguous
    Hkv, p, D = _geom(k_pool)
    k_new, v_new = _c(k_new, np.uint16), _c(v_new, np.uint16)
    slot = _c(slot_mapping, np.int64)
    T = slot.shape[0]
    assert k_new.shape == (T, Hkv, D) and v_new.shape == (T, Hkv, D)
    lib.oracle_kv_append(_p(k_pool), _p(v_pool), ctypes.c_int32(Hkv), ctypes.c_int32(p),
                         ctypes.c_int32(D), _p(k_new), _p(v_new), _p(slot), ctypes.c_int64(T))


def kv_gather(k_pool, v_pool, block_table, seq_lens):
    """GATHER.  -> (k uint16 [sum L, Hkv, D], v the same, cu int32 [S+1])."""
    lib = _load()
    Hkv, p, D = _geom(k_pool)
    k_pool, v_pool = _c(k_pool, np.uint16), _c(v_pool, np.uint16)
    bt, sl = _c(block_table, np.int32), _c(seq_lens, np.int32)
    S = sl.shape[0]
    cu = np.zeros(S + 1, dtype=np.int32)
    cu[1:] = np.cumsum(sl)
    k_out = np.zeros((int(cu[-1]), Hkv, D), dtype=np.uint16)
    v_out = np.zeros_like(k_out)
    lib.oracle_kv_gather(_p(k_out), _p(v_out), _p(k_pool), _p(v_pool), _p(bt),
                         ctypes.c_int64(bt.shape[1] if bt.ndim == 2 else 0), _p(sl), _p(cu), ctypes.c_int32(S),
                         ctypes.c_int32(Hkv), ctypes.c_int32(p), ctypes.c_int32(D))
    return k_out, v_out, cu


def kv_copy_pages(k_dst, v_dst, k_src, v_src, dst_pages, src_pages):
    """COPY_PAGES in place on ``k_dst`` / ``v_dst`` (uint16, C-contiguous)."""
    lib = _load()
    assert k_dst.dtype == np.uint16 and k_dst.flags.c_contiguous and v_dst.flags.c_contiguous
    Hkv, p, D = _geom(k_dst)
    assert _geom(k_src) == (Hkv, p, D)
    k_src, v_src = _c(k_src, np.uint16), _c(v_src, np.uint16)
    dp, sp = _c(dst_pages, np.int64), _c(src_pages, np.int64)
    assert dp.shape == sp.shape
    lib.oracle_kv_copy_pages(_p(k_dst), _p(v_dst), _p(k_src), _p(v_src), _p(dp), _p(sp),
                             ctypes.c_int64(dp.shape[0]), ctypes.c_int32(Hkv), ctypes.c_int32(p), ctypes.c_int32(D))


def paged_decode(q, k_pool, v_pool, block_table, seq_lens, scale):
    """DECODE.  q uint16 [S,Hq,D] -> (out fp64 [S,Hq,D], lse fp64 [S,Hq])."""
    lib = _load()
    Hkv, p, D = _geom(k_pool)
    q = _c(q, np.uint16)
    S, Hq, _ = q.shape
    k_pool, v_pool = _c(k_pool, np.uint16), _c(v_pool, np.uint16)
    bt, sl = _c(block_table, np.int32), _c(seq_lens, np.int32)
    out = np.zeros((S, Hq, D), dtype=np.float64)
    lse = np.zeros((S, Hq), dtype=np.float64)
    rc = lib.oracle_paged_decode(_p(out), _p(lse), _p(q), _p(k_pool), _p(v_pool), _p(bt),
                                 ctypes.c_int64(bt.shape[1] if bt.ndim == 2 else 0), _p(sl),
                                 ctypes.c_int32(S), ctypes.c_int32(Hq), ctypes.c_int32(Hkv),
                                 ctypes.c_int32(D), ctypes.c_int32(p), ctypes.c_double(float(scale)))
    if rc != 0:
        raise ValueError("oracle_paged_decode: bad geometry (%d)" % rc)
    return out, lse


def decode_probs(q, k_pool, v_pool, block_table, seq_lens, scale, s, h):
    """Row of the attention matrix P for decode row (s, h): fp64 [L_s]."""
    lib = _load()
    Hkv, p, D = _geom(k_pool)
    q = _c(q, np.uint16)
    _, Hq, _ = q.shape
    k_pool, v_pool = _c(k_pool, np.uint16), _c(v_pool, np.uint16)
    bt, sl = _c(block_table, np.int32), _c(seq_lens, np.int32)
    probs = np.zeros(int(sl[s]), dtype=np.float64)
    rc = lib.oracle_decode_probs(_p(probs), _p(q), _p(k_pool), _p(v_pool), _p(bt),
                                 ctypes.c_int64(bt.shape[1]), _p(sl), ctypes.c_int32(s),
                                 ctypes.c_int32(h), ctypes.c_int32(Hq), ctypes.c_int32(Hkv),
                                 ctypes.c_int32(D), ctypes.c_int32(p), ctypes.c_double(float(scale)))
    if rc != 0:
        raise ValueError("oracle_decode_probs: bad geometry (%d)" % rc)
    return probs


def paged_prefill(q, cu_seqlens_q, k_pool, v_pool, block_table, seq_lens, scale, causal=True, rows=None):
    """PREFILL.  q uint16 [T,Hq,D]; rows = ascending global row indices (default all).

    Returns (out fp64 [n_rows,Hq,D], lse fp64 [n_rows,Hq]).
    """
    lib = _load()
    Hkv, p, D = _geom(k_pool)
    q = _c(q, np.uint16)
    T, Hq, _ = q.shape
    cu = _c(cu_seqlens_q, np.int32)
    S = cu.shape[0] - 1
    k_pool, v_pool = _c(k_pool, np.uint16), _c(v_pool, np.uint16)
    bt, sl = _c(block_table, np.int32), _c(seq_lens, np.int32)
    rows = np.arange(T, dtype=np.int32) if rows is None else _c(rows, np.int32)
    assert np.all(np.diff(rows) > 0) if rows.size > 1 else True
    n = rows.shape[0]
    out = np.zeros((n, Hq, D), dtype=np.float64)
    lse = np.zeros((n, Hq), dtype=np.float64)
    rc = lib.oracle_paged_prefill_rows(_p(out), _p(lse), _p(q), _p(cu), _p(k_pool), _p(v_pool), _p(bt),
                                       ctypes.c_int64(bt.shape[1] if bt.ndim == 2 else 0), _p(sl),
                                       ctypes.c_int32(S), ctypes.c_int32(Hq), ctypes.c_int32(Hkv),
                                       ctypes.c_int32(D), ctypes.c_int32(p),
                                       ctypes.c_double(float(scale)), ctypes.c_int32(1 if causal else 0),
                                       _p(rows), ctypes.c_int64(n))
    if rc != 0:
        raise ValueError("oracle_paged_prefill_rows: bad geometry (%d)" % rc)
    return out, lse


def decode_partition(q, k_pool, v_pool, block_table, seq_lens, scale, s, h, j0, j1):
    """One split-K partition [j0, j1) of decode row (s, h): (m, l, O fp64 [D]) unnormalised."""
    lib = _load()
    Hkv, p, D = _geom(k_pool)
    q = _c(q, np.uint16)
    _, Hq, _ = q.shape
    k_pool, v_pool = _c(k_pool, np.uint16), _c(v_pool, np.uint16)
    bt, sl = _c(block_table, np.int32), _c(seq_lens, np.int32)
    m, l = ctypes.c_double(0.0), ctypes.c_double(0.0)
    O = np.zeros(D, dtype=np.float64)
    rc = lib.oracle_decode_partition(ctypes.byref(m), ctypes.byref(l), _p(O), _p(q), _p(k_pool),
                                     _p(v_pool), _p(bt), ctypes.c_int64(bt.shape[1]), _p(sl),
                                     ctypes.c_int32(s), ctypes.c_int32(h), ctypes.c_int32(Hq),
                                     ctypes.c_int32(Hkv), ctypes.c_int32(D), ctypes.c_int32(p),
                                     ctypes.c_double(float(scale)), ctypes.c_int32(j0), ctypes.c_int32(j1))
    if rc != 0:
        raise ValueError("oracle_decode_partition: bad geometry (%d)" % rc)
    return m.value, l.value, O


def lse_combine(m, l, O):
    """COMBINE: m, l fp64 [n]; O fp64 [n, D] -> (out fp64 [D], lse)."""
    lib = _load()
    m, l, O = _c(m, np.float64), _c(l, np.float64), _c(O, np.float64)
    n, D = O.shape
    out = np.zeros(D, dtype=np.float64)
    lse = ctypes.c_double(0.0)
    lib.oracle_lse_combine(_p(out), ctypes.byref(lse), _p(m), _p(l), _p(O), ctypes.c_int32(n),
                           ctypes.c_int32(D))
    return out, lse.value
