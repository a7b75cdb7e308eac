"""Pins of the fp8 (e4m3) K/V-pool oracle (oracle/fp8.py) against things other than itself: values the format
definition fixes, brute-force nearest-value search, torch's float8_e4m3fn cast (a library routine), and the
pinned bf16 oracle on pools whose dequantised values are exactly bf16-representable.  CPU only."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle
from oracle import fp8
from workloads import bf16_bits_from_f32


def test_e4m3_decode_table_values_fixed_by_the_format():
    t = fp8.e4m3_decode_table()
    fixed = {0x00: 0.0, 0x01: 2.0 ** -9, 0x07: 7 * 2.0 ** -9, 0x08: 2.0 ** -6, 0x0F: 2.0 ** -6 * 1.875,
             0x38: 1.0, 0x39: 1.125, 0x3A: 1.25, 0x40: 2.0, 0x77: 240.0, 0x78: 256.0, 0x7E: 448.0,
             0xB8: -1.0, 0xFE: -448.0}
    for code, v in fixed.items():
        assert t[code] == v, hex(code)
    assert np.isnan(t[0x7F]) and np.isnan(t[0xFF])
    assert np.isfinite(t).sum() == 254
    assert np.signbit(t[0x80]) and t[0x80] == 0.0
    assert np.all(np.diff(t[:0x7F]) > 0)          # magnitudes strictly increasing with the code
    assert np.all(t[0x80:0xFF] == -t[0x00:0x7F])  # sign bit only flips the sign


def test_e4m3_encode_cases_fixed_by_round_to_nearest_even_and_saturation():
    cases = [(1.0, 0x38), (1.0625, 0x38),   # tie 1.0 | 1.125 -> even code 0x38
             (1.1875, 0x3A),                # tie 1.125 (0x39) | 1.25 (0x3A) -> even
             (1.07, 0x39), (448.0, 0x7E), (464.0, 0x7E), (1e6, 0x7E), (np.inf, 0x7E), (-1e6, 0xFE),
             (2.0 ** -9, 0x01), (2.0 ** -10, 0x00),  # tie 0 | 2^-9 -> even code 0
             (1.5 * 2.0 ** -9, 0x02),                # tie 0x01 | 0x02 -> even
             (0.0, 0x00), (-0.0, 0x80), (-1.0, 0xB8), (np.nan, 0x7F), (2.0 ** -6, 0x08), (0.3, 0x2A)]
    y = np.array([c[0] for c in cases], dtype=np.float32)
    want = np.array([c[1] for c in cases], dtype=np.uint8)
    got = fp8.e4m3_encode(y)
    assert got.tolist() == want.tolist(), [(c, hex(g)) for c, g in zip(cases, got)]


def test_e4m3_encode_round_trip_and_brute_force_nearest():
    t = fp8.e4m3_decode_table()
    finite = np.array([c for c in range(256) if np.isfinite(t[c])], dtype=np.uint8)
    assert fp8.e4m3_encode(t[finite].astype(np.float32)).tolist() == finite.tolist()
    rng = np.random.default_rng(7)
    y = np.concatenate([rng.normal(0, 1, 4000), rng.normal(0, 100, 2000), rng.uniform(-2.0 ** -6, 2.0 ** -6, 2000)]
                       ).astype(np.float32)
    got = fp8.e4m3_encode(y)
    vals = t[finite]
    for yi, ci in zip(y.astype(np.float64), got):
        yc = min(max(yi, -448.0), 448.0)
        d = np.abs(vals - yc)
        assert abs(t[ci] - yc) == d.min()
        near = finite[d == d.min()]
        if len(near) > 1 and not (yc == 0.0):  # an exact tie: the even code wins
            assert ci & 1 == 0


def test_e4m3_encode_matches_torch_cast_in_range():
    rng = np.random.default_rng(11)
    y = np.concatenate([rng.normal(0, 1, 20000), rng.normal(0, 60, 20000), rng.uniform(-0.02, 0.02, 20000)]
                       ).astype(np.float32)
    y = y[np.abs(y) <= 448.0]
    ref = torch.from_numpy(y).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(fp8.e4m3_encode(y), ref)


def _exact_case(seed=3, S=3, Hq=8, Hkv=2, D=64, p=16, num_pages=24):
    rng = np.random.default_rng(seed)
    seq_lens = np.array([1, 37, 64][:S], dtype=np.int32)
    perm = rng.permutation(num_pages)
    maxp = 6
    bt = np.full((S, maxp), -1, dtype=np.int32)
    cur = 0
    for s in range(S):
        n = (int(seq_lens[s]) + p - 1) // p
        bt[s, :n] = perm[cur:cur + n]
        cur += n
    finite = np.array([c for c in range(256) if c not in (0x7F, 0xFF)], dtype=np.uint8)
    k8 = finite[rng.integers(0, 254, (num_pages, Hkv, p, D))]
    v8 = finite[rng.integers(0, 254, (num_pages, Hkv, p, D))]
    # power-of-two scales, different for every (page, head): dequantised values stay exactly bf16-representable
    ks = (2.0 ** rng.integers(-6, 3, (num_pages, Hkv))).astype(np.float32)
    vs = (2.0 ** rng.integers(-6, 3, (num_pages, Hkv))).astype(np.float32)
    q = bf16_bits_from_f32(rng.normal(0, 0.05, (S, Hq, D)).astype(np.float32))
    return seq_lens, bt, k8, v8, ks, vs, q


def test_decode_fp8_equals_pinned_bf16_oracle_on_the_dequantised_pool():
    seq_lens, bt, k8, v8, ks, vs, q = _exact_case()
    t = fp8.e4m3_decode_table()
    kd = (t[k8] * ks.astype(np.float64)[:, :, None, None]).astype(np.float32)
    vd = (t[v8] * vs.astype(np.float64)[:, :, None, None]).astype(np.float32)
    kb, vb = bf16_bits_from_f32(kd), bf16_bits_from_f32(vd)
    # exactness of the detour through bf16 (e4m3 has 4 significant bits, the scale is a power of two)
    assert np.array_equal((kb.astype(np.uint32) << 16).view(np.float32), kd)
    scale = np.float32(1 / 8)
    want, want_lse = oracle.paged_decode(q, kb, vb, bt, seq_lens, scale)
    got, got_lse = fp8.paged_decode_fp8(q, k8, v8, ks, vs, bt, seq_lens, scale)
    assert np.abs(got - want).max() <= 1e-12 * max(1.0, np.abs(want).max())
    assert np.abs(got_lse - want_lse).max() <= 1e-12 * max(1.0, np.abs(want_lse).max())


def test_decode_fp8_len0_and_len1_closed_forms():
    seq_lens, bt, k8, v8, ks, vs, q = _exact_case()
    seq_lens = np.array([0, 1, 64], dtype=np.int32)
    out, lse = fp8.paged_decode_fp8(q, k8, v8, ks, vs, bt, seq_lens, np.float32(0.125))
    assert np.all(out[0] == 0) and np.all(np.isneginf(lse[0]))
    t = fp8.e4m3_decode_table()
    page = int(bt[1, 0])
    for h in range(q.shape[1]):
        g = h // (q.shape[1] // k8.shape[1])
        assert np.array_equal(out[1, h], t[v8[page, g, 0]] * float(vs[page, g]))  # L = 1: the V row itself


def test_append_fp8_round_trip_skip_and_untouched_slots():
    rng = np.random.default_rng(5)
    num_pages, Hkv, p, D, T = 6, 2, 16, 64, 40
    t = fp8.e4m3_decode_table()
    finite = np.array([c for c in range(256) if c not in (0x7F, 0xFF, 0x80)], dtype=np.uint8)
    ks = (2.0 ** rng.integers(-4, 3, (num_pages, Hkv))).astype(np.float32)
    vs = (2.0 ** rng.integers(-4, 3, (num_pages, Hkv))).astype(np.float32)
    slots = rng.permutation(num_pages * p)[:T].astype(np.int64)
    slots[::7] = -1
    ck = finite[rng.integers(0, len(finite), (T, Hkv, D))]
    cv = finite[rng.integers(0, len(finite), (T, Hkv, D))]
    page = np.where(slots >= 0, slots // p, 0)
    # rows whose exact value is code * scale (power-of-two scale: representable in bf16): the append must return the code
    k_new = bf16_bits_from_f32((t[ck] * ks[page].astype(np.float64)[:, :, None]).astype(np.float32))
    v_new = bf16_bits_from_f32((t[cv] * vs[page].astype(np.float64)[:, :, None]).astype(np.float32))
    k8 = np.full((num_pages, Hkv, p, D), 0x7F, dtype=np.uint8)
    v8 = np.full((num_pages, Hkv, p, D), 0x7F, dtype=np.uint8)
    fp8.kv_append_fp8(k8, v8, ks, vs, k_new, v_new, slots)
    written = np.zeros((num_pages, p), dtype=bool)
    for i, s in enumerate(slots):
        if s < 0:
            continue
        written[s // p, s % p] = True
        assert np.array_equal(k8[s // p, :, s % p, :], ck[i])
        assert np.array_equal(v8[s // p, :, s % p, :], cv[i])
    assert np.all(k8.transpose(0, 2, 1, 3)[~written] == 0x7F) and np.all(v8.transpose(0, 2, 1, 3)[~written] == 0x7F)


def test_append_fp8_quantisation_error_bound_and_saturation():
    rng = np.random.default_rng(9)
    num_pages, Hkv, p, D = 2, 1, 16, 128
    x = rng.normal(0, 1, (p, Hkv, D)).astype(np.float32)
    x[0, 0, :4] = [1e4, -1e4, 0.0, 3e-4]
    xb = bf16_bits_from_f32(x)
    xf = (xb.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    sc = np.full((num_pages, Hkv), 0.01, dtype=np.float32)
    k8 = np.zeros((num_pages, Hkv, p, D), dtype=np.uint8)
    v8 = np.zeros_like(k8)
    fp8.kv_append_fp8(k8, v8, sc, sc, xb, xb, np.arange(p, dtype=np.int64))
    deq = fp8.e4m3_decode_table()[k8[0, 0]] * float(sc[0, 0])
    y = xf[:, 0, :] / float(sc[0, 0])
    inr = np.abs(y) <= 448
    # relative error of a normal e4m3 value <= 2^-4; absolute error of a subnormal <= 2^-10 (in units of the scale)
    assert np.all(np.abs(deq - xf[:, 0, :])[inr] <= np.maximum(np.abs(xf[:, 0, :])[inr] * 2.0 ** -4, 2.0 ** -10 * 0.01) * 1.0001)
    assert k8[0, 0, 0, 0] == 0x7E and k8[0, 0, 0, 1] == 0xFE and k8[0, 0, 0, 2] == 0x00
    assert np.array_equal(k8, v8)


def _prefill_case(seed=13, Hq=8, Hkv=2, D=64, p=16, num_pages=40):
    """Ragged prefill batch on an exactly representable quantised pool: (cu, seq_lens, bt, k8, v8, ks, vs, q)."""
    rng = np.random.default_rng(seed)
    q_lens = np.array([5, 1, 0, 33], dtype=np.int32)
    prefix = np.array([20, 0, 7, 16], dtype=np.int32)
    seq_lens = (prefix + q_lens).astype(np.int32)
    S = len(q_lens)
    cu = np.zeros(S + 1, dtype=np.int32)
    cu[1:] = np.cumsum(q_lens)
    perm = rng.permutation(num_pages)
    bt = np.full((S, 6), -1, dtype=np.int32)
    cur = 0
    for s in range(S):
        n = (int(seq_lens[s]) + p - 1) // p
        bt[s, :n] = perm[cur:cur + n]
        cur += n
    finite = np.array([c for c in range(256) if c not in (0x7F, 0xFF)], dtype=np.uint8)
    k8 = finite[rng.integers(0, 254, (num_pages, Hkv, p, D))]
    v8 = finite[rng.integers(0, 254, (num_pages, Hkv, p, D))]
    ks = (2.0 ** rng.integers(-6, 3, (num_pages, Hkv))).astype(np.float32)
    vs = (2.0 ** rng.integers(-6, 3, (num_pages, Hkv))).astype(np.float32)
    q = bf16_bits_from_f32(rng.normal(0, 0.05, (int(cu[-1]), Hq, D)).astype(np.float32))
    return cu, seq_lens, bt, k8, v8, ks, vs, q


@pytest.mark.parametrize("causal", [True, False])
def test_prefill_fp8_equals_pinned_bf16_prefill_oracle_on_the_dequantised_pool(causal):
    """PREFILL_FP8 against the pinned C prefill oracle (tests/test_oracle_pins.py) on a pool whose dequantised
    values are exactly bf16 (power-of-two scales that differ per (page, head))."""
    cu, seq_lens, bt, k8, v8, ks, vs, q = _prefill_case()
    t = fp8.e4m3_decode_table()
    kb = bf16_bits_from_f32((t[k8] * ks.astype(np.float64)[:, :, None, None]).astype(np.float32))
    vb = bf16_bits_from_f32((t[v8] * vs.astype(np.float64)[:, :, None, None]).astype(np.float32))
    scale = np.float32(1 / 8)
    want, want_lse = oracle.paged_prefill(q, cu, kb, vb, bt, seq_lens, scale, causal=causal)
    got, got_lse = fp8.paged_prefill_fp8(q, cu, k8, v8, ks, vs, bt, seq_lens, scale, causal=causal)
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 1e-12 * max(1.0, np.abs(want).max())
    assert np.abs(got_lse - want_lse).max() <= 1e-12 * max(1.0, np.abs(want_lse).max())


def test_prefill_fp8_one_row_is_decode_last_row_sees_everything_and_row_subset():
    cu, seq_lens, bt, k8, v8, ks, vs, q = _prefill_case()
    scale = np.float32(0.125)
    full, full_lse = fp8.paged_prefill_fp8(q, cu, k8, v8, ks, vs, bt, seq_lens, scale)
    # the last row of every sequence with rows = DECODE_FP8 with that row as the query
    last = [int(cu[s + 1]) - 1 for s in range(len(seq_lens)) if cu[s + 1] > cu[s]]
    seqs = [s for s in range(len(seq_lens)) if cu[s + 1] > cu[s]]
    dec, dec_lse = fp8.paged_decode_fp8(q[last], k8, v8, ks, vs, bt[seqs], seq_lens[seqs], scale)
    assert np.abs(full[last] - dec).max() < 1e-13 and np.abs(full_lse[last] - dec_lse).max() < 1e-13
    # a subset of rows = the same rows of the full result
    rows = np.array([0, 4, 5, 6, 20, 38])
    sub, sub_lse = fp8.paged_prefill_fp8(q, cu, k8, v8, ks, vs, bt, seq_lens, scale, rows=rows)
    assert np.array_equal(sub, full[rows]) and np.array_equal(sub_lse, full_lse[rows])
    # first row of a sequence without prefix: the dequantised V row 0
    t = fp8.e4m3_decode_table()
    r = int(cu[1])   # sequence 1: prefix 0, one row
    page = int(bt[1, 0])
    for h in range(q.shape[1]):
        g = h // (q.shape[1] // k8.shape[1])
        assert np.array_equal(full[r, h], t[v8[page, g, 0]] * float(vs[page, g]))


def test_prefill_fp8_causality_under_saturated_future_codes():
    """Overwriting every position a row must not see with +-448 codes leaves that row unchanged (R6)."""
    cu, seq_lens, bt, k8, v8, ks, vs, q = _prefill_case()
    scale = np.float32(0.125)
    s, p = 3, 16
    n, L = int(cu[s + 1] - cu[s]), int(seq_lens[s])
    i = 10
    r = int(cu[s]) + i
    base, _ = fp8.paged_prefill_fp8(q, cu, k8, v8, ks, vs, bt, seq_lens, scale, rows=[r])
    k2, v2 = k8.copy(), v8.copy()
    for j in range((L - n) + i + 1, L):
        k2[bt[s, j // p], :, j % p, :] = 0x7E
        v2[bt[s, j // p], :, j % p, :] = 0xFE
    pois, _ = fp8.paged_prefill_fp8(q, cu, k2, v2, ks, vs, bt, seq_lens, scale, rows=[r])
    assert np.array_equal(base, pois)
    # and it is not a no-op: the non-causal result does change
    a, _ = fp8.paged_prefill_fp8(q, cu, k8, v8, ks, vs, bt, seq_lens, scale, causal=False, rows=[r])
    b, _ = fp8.paged_prefill_fp8(q, cu, k2, v2, ks, vs, bt, seq_lens, scale, causal=False, rows=[r])
    assert np.abs(a - b).max() > 1e-3
