"""Test helpers: format conversion, a numpy brute force and the parity gates.

The brute force is an independent restatement of softmax(Q K^T scale) V on explicitly gathered dense
K/V with library matmuls; it shares no code with ``oracle/`` (C loops) or with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from workloads import BF16_NAN, PagedBatch, bf16_bits_from_f32, f64_from_bf16_bits  # noqa: F401

# Parity gates of BASELINE.json north_star as read in DESIGN.md R11:
#   (i) max elementwise |gpu - oracle| <= 2e-2
#   (ii) per output row (one (token, head) D-vector)  max|gpu - oracle| / max|oracle| <= 1e-2
MAX_ABS = 2e-2
MAX_ROW_REL = 1e-2


def numpy_scatter(batch: PagedBatch, k_pool: np.ndarray, v_pool: np.ndarray, slot=None):
    """Brute-force APPEND with numpy fancy indexing (in place)."""
    p = batch.page_size
    slot = batch.slot_mapping if slot is None else slot
    ok = slot >= 0
    k_pool[slot[ok] // p, :, slot[ok] % p, :] = batch.k_new[ok]
    v_pool[slot[ok] // p, :, slot[ok] % p, :] = batch.v_new[ok]


def compact_pool_after_append(batch: PagedBatch):
    """The compact store with the step's new rows written (numpy scatter), as a pool."""
    k, v = batch.k_store.copy(), batch.v_store.copy()
    numpy_scatter(batch, k, v, batch.compact_slot_mapping)
    return k, v


def decode_q(batch: PagedBatch) -> np.ndarray:
    """One query row per sequence for decode: the sequence's new token, zeros where it has none (L = 0)."""
    assert int(batch.q_lens.max(initial=0)) <= 1
    q = np.zeros((batch.num_seqs, batch.num_q_heads, batch.head_dim), dtype=np.uint16)
    has = batch.q_lens > 0
    q[has] = batch.q[batch.cu_seqlens_q[:-1][has]]
    return q


def dense_kv(batch: PagedBatch, k_pool, v_pool, block_table, s):
    """Gather sequence s to dense fp64 K, V [L, Hkv, D] with numpy indexing."""
    p = batch.page_size
    L = int(batch.seq_lens[s])
    j = np.arange(L)
    pages = block_table[s, j // p].astype(np.int64)
    K = f64_from_bf16_bits(k_pool[pages, :, j % p, :])
    V = f64_from_bf16_bits(v_pool[pages, :, j % p, :])
    return K, V


def brute_force_attention(batch: PagedBatch, k_pool, v_pool, block_table, causal=True):
    """softmax(Q K^T scale) V per sequence with an explicit [n, L] mask matrix.

    Returns (out [T,Hq,D] fp64, lse [T,Hq] fp64).  K/V repeat-interleaved to Hq heads.
    """
    Hq, Hkv, D = batch.num_q_heads, batch.num_kv_heads, batch.head_dim
    G = Hq // Hkv
    T = batch.total_q
    out = np.zeros((T, Hq, D))
    lse = np.full((T, Hq), -np.inf)
    scale = float(batch.scale)
    for s in range(batch.num_seqs):
        r0, r1 = int(batch.cu_seqlens_q[s]), int(batch.cu_seqlens_q[s + 1])
        n, L = r1 - r0, int(batch.seq_lens[s])
        if n == 0 or L == 0:
            continue
        K, V = dense_kv(batch, k_pool, v_pool, block_table, s)
        K = np.repeat(K, G, axis=1)  # [L, Hq, D]
        V = np.repeat(V, G, axis=1)
        Q = f64_from_bf16_bits(batch.q[r0:r1])  # [n, Hq, D]
        X = np.einsum("nhd,lhd->hnl", Q, K) * scale
        if causal:
            i = np.arange(n)[:, None]
            j = np.arange(L)[None, :]
            X = np.where(j <= (L - n) + i, X, -np.inf)
        M = X.max(axis=2, keepdims=True)
        W = np.exp(X - M)
        Z = W.sum(axis=2, keepdims=True)
        Pm = W / Z
        out[r0:r1] = np.einsum("hnl,lhd->nhd", Pm, V)
        lse[r0:r1] = (M[..., 0] + np.log(Z[..., 0])).T
    return out, lse


def check_parity(got: np.ndarray, want: np.ndarray, what: str = ""):
    """Apply both gates; returns (max_abs, max_row_rel) for reporting."""
    got = np.asarray(got, dtype=np.float64).reshape(-1, want.shape[-1])
    want = np.asarray(want, dtype=np.float64).reshape(-1, want.shape[-1])
    assert got.shape == want.shape, (got.shape, want.shape)
    assert np.all(np.isfinite(got)), "%s: non-finite values in the GPU output" % what
    err = np.abs(got - want)
    max_abs = float(err.max()) if err.size else 0.0
    row_ref = np.abs(want).max(axis=1)
    row_err = err.max(axis=1)
    nz = row_ref > 0
    max_rel = float((row_err[nz] / row_ref[nz]).max()) if nz.any() else 0.0
    # rows whose oracle value is identically zero (L = 0) must be reproduced exactly
    assert np.all(row_err[~nz] == 0), "%s: non-zero output where the oracle is exactly 0" % what
    assert max_abs <= MAX_ABS, "%s: max-abs %.3e > %.1e" % (what, max_abs, MAX_ABS)
    assert max_rel <= MAX_ROW_REL, "%s: max row-rel %.3e > %.1e" % (what, max_rel, MAX_ROW_REL)
    return max_abs, max_rel
