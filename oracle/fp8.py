"""CPU oracle of the quantised (fp8 e4m3) K/V pool: SURVEY 8(f) rank 4, "fp8 K/V pages with per-page scales"
(PAPER.md:134 lists the KV-cache state the runtime owns; the paper gives no numerical detail, the reading is
DESIGN.md sec. 2, R24-R26).  TEST INFRASTRUCTURE ONLY: plain numpy, fp64 unless the definition fixes fp32; shares
no code with the CUDA path.

Format (OCP 8-bit floating point, E4M3 "fn" variant): bit 7 sign, bits 6..3 exponent e (bias 7), bits 2..0
mantissa m.  e = 0: value = (-1)^s * 2^-6 * m/8 (subnormal, includes +-0); 1 <= e <= 15: (-1)^s * 2^(e-7) * (1+m/8),
except e = 15, m = 7 which is NaN.  No infinities; largest finite magnitude 448.

Definitions
  DEQUANT        value(page, h, slot, d) = e4m3(code) * scale[page][h]           (exact in fp64)
  APPEND_FP8     y = fp32(x) / scale[page][h] in IEEE fp32 (round to nearest even), code = RNE(y) to e4m3 with
                 saturation to +-448 ("satfinite"); NaN -> 0x7F.  The quantised code is an integer decided by
                 floating point, so both sides take the decision in the kernel's precision (fp32).
  DECODE_FP8     ORACLE_DECODE on the dequantised K and V.
  PREFILL_FP8    ORACLE_PREFILL on the dequantised K and V: query row i of sequence s (n_s rows) sees
                 positions j <= (L_s - n_s) + i when causal (R6), all L_s positions otherwise.
Pools are uint8 ``[num_pages, Hkv, page_size, D]``; scales fp32 ``[num_pages, Hkv]`` (inputs, caller-owned).
"""
from __future__ import annotations

import numpy as np


def e4m3_decode_table() -> np.ndarray:
    """fp64[256]: the value of every code, written out from the format definition."""
    t = np.zeros(256, dtype=np.float64)
    for code in range(256):
        s = -1.0 if code & 0x80 else 1.0
        e = (code >> 3) & 0xF
        m = code & 0x7
        if e == 15 and m == 7:
            v = np.nan
        elif e == 0:
            v = s * 2.0 ** -6 * (m / 8.0)
        else:
            v = s * 2.0 ** (e - 7) * (1.0 + m / 8.0)
        t[code] = v
    return t


_TABLE = e4m3_decode_table()
_POS = _TABLE[:0x7F].copy()  # magnitudes of codes 0x00..0x7E, strictly increasing, 0 .. 448


def e4m3_encode(y) -> np.ndarray:
    """fp32 array -> uint8 codes: round to nearest, ties to the even code, saturate to +-448, NaN -> 0x7F."""
    y = np.asarray(y, dtype=np.float32)
    a = np.abs(y).astype(np.float64)
    sign = np.signbit(y).astype(np.uint8) << 7
    a_c = np.minimum(a, 448.0)  # satfinite (also maps +-inf to 448)
    hi = np.searchsorted(_POS, a_c, side="left")  # first magnitude >= a
    hi = np.clip(hi, 0, 0x7E)
    lo = np.maximum(hi - 1, 0)
    d_hi = _POS[hi] - a_c
    d_lo = a_c - _POS[lo]
    take_lo = (d_lo < d_hi) | ((d_lo == d_hi) & ((lo & 1) == 0))
    mag = np.where(take_lo, lo, hi).astype(np.uint8)
    code = (mag | sign).astype(np.uint8)
    return np.where(np.isnan(y), np.uint8(0x7F), code).astype(np.uint8)


def bf16_bits_to_f32(u16) -> np.ndarray:
    u = np.ascontiguousarray(u16, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32)


def kv_append_fp8(k_pool8, v_pool8, k_scale, v_scale, k_new, v_new, slot_mapping):
    """APPEND_FP8 in place.  k_new / v_new: bf16 bit patterns uint16 [T, Hkv, D]; slot < 0 = skip."""
    assert k_pool8.dtype == np.uint8 and v_pool8.dtype == np.uint8
    _, Hkv, p, D = k_pool8.shape
    kf, vf = bf16_bits_to_f32(k_new), bf16_bits_to_f32(v_new)
    ks, vs = np.asarray(k_scale, dtype=np.float32), np.asarray(v_scale, dtype=np.float32)
    slot = np.asarray(slot_mapping, dtype=np.int64)
    ok = slot >= 0
    # R19: two rows naming one slot in a call is a caller error; the bf16 oracle's sequential loop gives "last writer
    # wins", numpy fancy assignment gives no stated order, so this vectorised form refuses duplicates outright
    assert np.unique(slot[ok]).size == int(ok.sum()), "duplicate slots in one append (undefined, R19)"
    page, off = slot[ok] // p, slot[ok] % p
    # fp32 / fp32 -> fp32, IEEE round to nearest even, element by element (the scale of the row's page and head)
    yk = kf[ok] / ks[page][:, :, None]
    yv = vf[ok] / vs[page][:, :, None]
    assert yk.dtype == np.float32 and yv.dtype == np.float32
    k_pool8[page, :, off, :] = e4m3_encode(yk)  # slots are unique within a call (duplicates: caller error, R19)
    v_pool8[page, :, off, :] = e4m3_encode(yv)


def dequant_gather(pool8, scale, block_table_row, L):
    """GATHER + DEQUANT of one sequence: fp64 [L, Hkv, D]."""
    _, Hkv, p, D = pool8.shape
    out = np.zeros((L, Hkv, D), dtype=np.float64)
    for j in range(L):
        page, off = int(block_table_row[j // p]), j % p
        out[j] = _TABLE[pool8[page, :, off, :]] * np.asarray(scale[page], dtype=np.float64)[:, None]
    return out


def paged_decode_fp8(q, k_pool8, v_pool8, k_scale, v_scale, block_table, seq_lens, scale):
    """DECODE_FP8.  q bf16 bits uint16 [S, Hq, D] -> (out fp64 [S, Hq, D], lse fp64 [S, Hq])."""
    qf = bf16_bits_to_f32(q).astype(np.float64)
    S, Hq, D = qf.shape
    Hkv = k_pool8.shape[1]
    G = Hq // Hkv
    sc = float(np.float32(scale))
    out = np.zeros((S, Hq, D), dtype=np.float64)
    lse = np.full((S, Hq), -np.inf, dtype=np.float64)
    for s in range(S):
        L = int(seq_lens[s])
        if L == 0:
            continue
        K = dequant_gather(k_pool8, k_scale, block_table[s], L)
        V = dequant_gather(v_pool8, v_scale, block_table[s], L)
        for h in range(Hq):
            g = h // G
            x = sc * (K[:, g, :] @ qf[s, h])
            M = x.max()
            w = np.exp(x - M)
            Z = w.sum()
            out[s, h] = (w @ V[:, g, :]) / Z
            lse[s, h] = M + np.log(Z)
    return out, lse


def paged_prefill_fp8(q, cu_seqlens_q, k_pool8, v_pool8, k_scale, v_scale, block_table, seq_lens, scale, causal=True,
                      rows=None):
    """PREFILL_FP8.  q bf16 bits uint16 [T, Hq, D], ragged by cu_seqlens_q; rows = ascending global row indices
    (default all) -> (out fp64 [n_rows, Hq, D], lse fp64 [n_rows, Hq]).  Written out row by row: gather and dequantise
    the sequence, logits over the visible positions, max, exp, sum, weighted sum."""
    qf = bf16_bits_to_f32(q).astype(np.float64)
    T, Hq, D = qf.shape
    Hkv = k_pool8.shape[1]
    G = Hq // Hkv
    sc = float(np.float32(scale))
    cu = np.asarray(cu_seqlens_q, dtype=np.int64)
    rows = np.arange(T, dtype=np.int64) if rows is None else np.asarray(rows, dtype=np.int64)
    out = np.zeros((len(rows), Hq, D), dtype=np.float64)
    lse = np.full((len(rows), Hq), -np.inf, dtype=np.float64)
    cache_s, K, V = -1, None, None
    for idx, r in enumerate(rows):
        s = int(np.searchsorted(cu, r, side="right") - 1)
        n, L = int(cu[s + 1] - cu[s]), int(seq_lens[s])
        i = int(r - cu[s])
        if s != cache_s:
            K = dequant_gather(k_pool8, k_scale, block_table[s], L)
            V = dequant_gather(v_pool8, v_scale, block_table[s], L)
            cache_s = s
        vis = (L - n) + i + 1 if causal else L   # number of visible positions
        if vis <= 0:
            continue
        for h in range(Hq):
            g = h // G
            x = sc * (K[:vis, g, :] @ qf[r, h])
            M = x.max()
            w = np.exp(x - M)
            Z = w.sum()
            out[idx, h] = (w @ V[:vis, g, :]) / Z
            lse[idx, h] = M + np.log(Z)
    return out, lse
