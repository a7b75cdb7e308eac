"""Pins of the CPU oracle against things other than itself (no GPU needed).

Each test names the SURVEY.md 8(c) pin it implements.  A plausible mistake anywhere in
``oracle/mstar_oracle.c`` (dropped scale, wrong GQA map, transposed operand, off-by-one in the causal
bound, wrong page/offset split, missing max subtraction, wrong combine weight) fails at least one.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from tests.util import (brute_force_attention, compact_pool_after_append, decode_q, dense_kv,
                        f64_from_bf16_bits, bf16_bits_from_f32, numpy_scatter)

TOL = 1e-12


def small_batch(seed, lens, q_lens=None, Hq=8, Hkv=2, D=64, p=16, pool=None, **kw):
    rng = np.random.default_rng(seed)
    q_lens = [1] * len(lens) if q_lens is None else q_lens
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(rng, "t", lens, q_lens, Hq, Hkv, D, p, pool or max(2 * pages, 4), **kw)


def decode_on(batch, k=None, v=None, bt=None):
    if k is None:
        k, v = compact_pool_after_append(batch)
    bt = batch.compact_block_table if bt is None else bt
    return oracle.paged_decode(batch.q, k, v, bt, batch.seq_lens, batch.scale)


# ----------------------------------------------------------------------------- append

def test_append_matches_numpy_scatter_whole_pool_and_roundtrip():
    """Append pins (i)-(iii): whole-pool bit equality, untouched slots keep their bits, gather roundtrip."""
    b = small_batch(1, [1, 17, 33, 100], q_lens=[1, 5, 33, 40], Hq=4, Hkv=2, D=64, p=16)
    k0, v0 = b.full_pool()
    k1, v1 = k0.copy(), v0.copy()
    oracle.kv_append(k1, v1, b.k_new, b.v_new, b.slot_mapping)
    k2, v2 = k0.copy(), v0.copy()
    numpy_scatter(b, k2, v2)
    assert np.array_equal(k1, k2) and np.array_equal(v1, v2)
    # exactly T * Hkv * D words changed from NaN poison to data, nothing else moved
    changed = (k1 != k0)
    assert changed.sum() <= b.total_q * b.num_kv_heads * b.head_dim
    assert np.all(k0[changed] == W.BF16_NAN)
    # roundtrip: the new rows read back through the block table are the rows that were appended
    for s in range(b.num_seqs):
        n, L = int(b.q_lens[s]), int(b.seq_lens[s])
        j = np.arange(L - n, L)
        pages = b.block_table[s, j // b.page_size]
        t0 = int(b.cu_seqlens_q[s])
        assert np.array_equal(k1[pages, :, j % b.page_size, :], b.k_new[t0:t0 + n])
        assert np.array_equal(v1[pages, :, j % b.page_size, :], b.v_new[t0:t0 + n])


def test_gather_and_copy_pages_pins():
    """GATHER == numpy fancy indexing through the block table; GATHER(APPEND(x)) returns x for the new rows;
    COPY_PAGES == numpy page assignment, other pages keep their bits, negative ids skipped; copying a sequence's
    pages to fresh ids and pointing the block table at them leaves GATHER (and decode) bit-identical."""
    b = small_batch(3, [1, 17, 33, 100, 0], q_lens=[1, 5, 33, 40, 0], Hq=4, Hkv=2, D=64, p=16)
    k, v = b.full_pool()
    oracle.kv_append(k, v, b.k_new, b.v_new, b.slot_mapping)
    kg, vg, cu = oracle.kv_gather(k, v, b.block_table, b.seq_lens)
    assert cu.tolist() == [0, 1, 18, 51, 151, 151]
    for s in range(b.num_seqs):
        L, n = int(b.seq_lens[s]), int(b.q_lens[s])
        j = np.arange(L)
        pages = b.block_table[s, j // b.page_size]
        assert np.array_equal(kg[cu[s]:cu[s + 1]], k[pages, :, j % b.page_size, :])
        assert np.array_equal(vg[cu[s]:cu[s + 1]], v[pages, :, j % b.page_size, :])
        t0 = int(b.cu_seqlens_q[s])
        assert np.array_equal(kg[cu[s + 1] - n:cu[s + 1]], b.k_new[t0:t0 + n])
    # copy pages: sequence 3's pages to unused ids (in reverse order), one skipped pair
    used = set(b.used_pages.tolist())
    free = [pg for pg in range(b.num_pages) if pg not in used]
    src = b.block_table[3, :7].astype(np.int64)
    dst = np.array(free[:7][::-1], dtype=np.int64)
    src_s, dst_s = np.append(src, [5, -1]), np.append(dst, [-1, 5])
    k2, v2 = k.copy(), v.copy()
    oracle.kv_copy_pages(k2, v2, k, v, dst_s, src_s)
    k3, v3 = k.copy(), v.copy()
    k3[dst] = k[src]
    v3[dst] = v[src]
    assert np.array_equal(k2, k3) and np.array_equal(v2, v3)
    bt2 = b.block_table.copy()
    bt2[3, :7] = dst
    kg2, vg2, _ = oracle.kv_gather(k2, v2, bt2, b.seq_lens)
    assert np.array_equal(kg2, kg) and np.array_equal(vg2, vg)
    q = np.ascontiguousarray(b.q[:b.num_seqs])   # any S query rows
    o1, l1 = oracle.paged_decode(q, k, v, b.block_table, b.seq_lens, b.scale)
    o2, l2 = oracle.paged_decode(q, k2, v2, bt2, b.seq_lens, b.scale)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_cascade_identity_stacked_prefix_plus_suffix_merge():
    """SURVEY 8(f) rank 3 in fp64: decode over the shared prefix with the branches' queries stacked as grouped
    heads gives each branch's prefix state; merged with its private-suffix state by COMBINE (l = 1) it equals the
    plain decode over the whole sequence."""
    B, shared, p = 2, 32, 16
    lens = [40, 40, 33, 33, 100, 100]
    rng = np.random.default_rng(77)
    b = W.make_batch(rng, "cfg", lens, [1] * 6, 4, 2, 64, p, 64, share_with=[-1, 0, -1, 2, -1, 4],
                     shared_tokens=shared)
    k, v = compact_pool_after_append(b)
    q = decode_q(b)
    full, full_lse = oracle.paged_decode(q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    S, Hq, Hkv, D = 6, 4, 2, 64
    G, R = Hq // Hkv, S // B
    qa = np.zeros((R, Hq * B, D), dtype=np.uint16)
    for r in range(R):
        for kvh in range(Hkv):
            for br in range(B):
                for g in range(G):
                    qa[r, kvh * B * G + br * G + g] = q[r * B + br, kvh * G + g]
    pa, pa_lse = oracle.paged_decode(qa, k, v, b.compact_block_table[::B], np.full(R, shared, np.int32), b.scale)
    sb, sb_lse = oracle.paged_decode(q, k, v, np.ascontiguousarray(b.compact_block_table[:, shared // p:]),
                                     b.seq_lens - shared, b.scale)
    for s in range(S):
        for h in range(Hq):
            r, br, kvh, g = s // B, s % B, h // G, h % G
            ra = kvh * B * G + br * G + g
            out, lse = oracle.lse_combine(np.array([pa_lse[r, ra], sb_lse[s, h]]), np.ones(2),
                                          np.stack([pa[r, ra], sb[s, h]]))
            assert np.abs(out - full[s, h]).max() < 1e-12 and abs(lse - full_lse[s, h]) < 1e-12


def test_cascade_identity_three_branches_ragged_shared_lens_split_pieces():
    """The work split of mstar_paged_attn_decode_cascade in fp64: per request a prefix state over its shared_lens[r]
    tokens (ragged over requests, 0 allowed; branches grouped two + one as the 16 MMA rows allow at G = 7), cut in
    pieces, plus per-branch suffix states cut in pieces, all merged by COMBINE, equals the plain decode over the
    whole sequence, for three CFG labels."""
    B, p = 3, 16
    shared_r = [48, 0, 112]
    sfx = [[5, 40, 1], [33, 17, 64], [1, 90, 16]]   # a suffix of one token is only the step's new token
    lens = [shared_r[r] + sfx[r][b] for r in range(3) for b in range(B)]
    share = [-1 if b == 0 else r * B for r in range(3) for b in range(B)]
    shared = [shared_r[r] for r in range(3) for b in range(B)]
    rng = np.random.default_rng(78)
    b = W.make_batch(rng, "cfg3", lens, [1] * 9, 14, 2, 64, p, 96, share_with=share, shared_tokens=shared)
    k, v = compact_pool_after_append(b)
    q = decode_q(b)
    full, full_lse = oracle.paged_decode(q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    S, Hq = 9, 14
    chunk = 32   # pieces of 32 tokens
    for s in range(S):
        r = s // B
        for h in range(Hq):
            ms, ls, os_ = [], [], []
            # prefix pieces: computed once per request from any branch's block-table row, with this row's query
            for a in range(0, shared_r[r], chunk):
                m, l, o = oracle.decode_partition(q[s:s + 1], k, v, b.compact_block_table[r * B:r * B + 1],
                                                  np.array([shared_r[r]], np.int32), b.scale, 0, h, a,
                                                  min(a + chunk, shared_r[r]))
                ms.append(m); ls.append(l); os_.append(o)
            for a in range(shared_r[r], int(b.seq_lens[s]), chunk):
                m, l, o = oracle.decode_partition(q[s:s + 1], k, v, b.compact_block_table[s:s + 1],
                                                  b.seq_lens[s:s + 1], b.scale, 0, h, a,
                                                  min(a + chunk, int(b.seq_lens[s])))
                ms.append(m); ls.append(l); os_.append(o)
            out, lse = oracle.lse_combine(np.array(ms), np.array(ls), np.stack(os_))
            assert np.abs(out - full[s, h]).max() < 1e-12 and abs(lse - full_lse[s, h]) < 1e-12


def test_append_negative_slot_skipped():
    b = small_batch(2, [20, 9], q_lens=[3, 2], Hq=2, Hkv=1, D=64)
    k0, v0 = b.full_pool()
    slot = b.slot_mapping.copy()
    slot[1] = -1
    slot[4] = -7
    k1, v1 = k0.copy(), v0.copy()
    oracle.kv_append(k1, v1, b.k_new, b.v_new, slot)
    k2, v2 = k0.copy(), v0.copy()
    numpy_scatter(b, k2, v2, slot)
    assert np.array_equal(k1, k2) and np.array_equal(v1, v2)
    pg, off = b.slot_mapping[1] // 16, b.slot_mapping[1] % 16
    assert np.all(k1[pg, :, off, :] == W.BF16_NAN)


# ----------------------------------------------------------------------------- decode

@pytest.mark.parametrize("Hq,Hkv,D,p", [(8, 2, 64, 16), (7, 1, 128, 16), (4, 4, 64, 32), (6, 3, 128, 32)])
def test_decode_matches_brute_force(Hq, Hkv, D, p):
    """Decode pin (i): numpy brute force on dense gathered K/V, K/V repeat-interleaved to Hq heads."""
    b = small_batch(3, [1, p - 1, p, p + 1, 2 * p + 3, 100], Hq=Hq, Hkv=Hkv, D=D, p=p)
    k, v = compact_pool_after_append(b)
    out, lse = oracle.paged_decode(b.q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    ref, ref_lse = brute_force_attention(b, k, v, b.compact_block_table)
    assert np.abs(out - ref).max() < TOL
    assert np.abs(lse - ref_lse).max() < TOL


def test_decode_full_pool_equals_compact_store():
    """The physical-id pool and the compact store are the same problem (basis of the config-5 protocol)."""
    b = W.config1_tiny_decode()
    kf, vf = b.full_pool()
    numpy_scatter(b, kf, vf)
    o1, l1 = oracle.paged_decode(b.q, kf, vf, b.block_table, b.seq_lens, b.scale)
    o2, l2 = decode_on(b)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_decode_len1_is_v_row():
    """Decode pin (ii): L = 1 => out = V row 0 of head h div G, exactly."""
    b = small_batch(4, [1, 1, 1], Hq=8, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    out, lse = decode_on(b, k, v)
    for s in range(3):
        K, V = dense_kv(b, k, v, b.compact_block_table, s)
        for h in range(8):
            assert np.array_equal(out[s, h], V[0, h // 4])
            x = float(b.scale) * np.dot(f64_from_bf16_bits(b.q[s, h]), K[0, h // 4])
            assert abs(lse[s, h] - x) < TOL


def test_decode_two_key_logistic():
    """Closed form: two keys with logits 0 and x => out = v0 + sigmoid(x) (v1 - v0); lse = log(1 + e^x)."""
    b = small_batch(5, [2], Hq=1, Hkv=1, D=64, p=16)
    k, v = compact_pool_after_append(b)
    u0 = int(b.compact_block_table[0, 0])
    qv = np.zeros(64, np.float32); qv[3] = 2.0
    k0 = np.zeros(64, np.float32)
    k1 = np.zeros(64, np.float32); k1[3] = 1.5; k1[7] = 9.0   # q.k1 = 3, scale 1/8 -> x = 0.375
    b.q[0, 0] = bf16_bits_from_f32(qv)
    k[u0, 0, 0] = bf16_bits_from_f32(k0)
    k[u0, 0, 1] = bf16_bits_from_f32(k1)
    out, lse = decode_on(b, k, v)
    x = 0.375
    sig = 1.0 / (1.0 + math.exp(-x))
    v0 = f64_from_bf16_bits(v[u0, 0, 0]); v1 = f64_from_bf16_bits(v[u0, 0, 1])
    assert np.abs(out[0, 0] - (v0 + sig * (v1 - v0))).max() < TOL
    assert abs(lse[0, 0] - math.log1p(math.exp(x))) < TOL


def test_decode_zero_query_is_mean_and_position_code():
    """Decode pins (iii) + (v): q = 0 => arithmetic mean of the V rows; V[j][.][0] = j => (L-1)/2."""
    lens = [1, 15, 16, 17, 47, 100]
    b = small_batch(6, lens, Hq=4, Hkv=2, D=64)
    b.q[:] = 0
    k, v = compact_pool_after_append(b)
    for s, L in enumerate(lens):   # position code in element 0 of every kv head
        j = np.arange(L)
        v[b.compact_block_table[s, j // 16], :, j % 16, 0] = bf16_bits_from_f32(j.astype(np.float32))[:, None]
    out, lse = decode_on(b, k, v)
    for s, L in enumerate(lens):
        _, V = dense_kv(b, k, v, b.compact_block_table, s)
        for h in range(4):
            assert np.abs(out[s, h] - V[:, h // 2].mean(axis=0)).max() < TOL
            assert abs(out[s, h, 0] - (L - 1) / 2.0) < TOL
            assert abs(lse[s, h] - math.log(L)) < TOL


def test_decode_unit_values_and_convex_hull():
    """Decode pins (iv) + (xi): V == 1 => out == 1; min_j V <= out <= max_j V."""
    b = small_batch(7, [33, 64, 5], Hq=8, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    out, _ = decode_on(b, k, v)
    for s in range(3):
        _, V = dense_kv(b, k, v, b.compact_block_table, s)
        for h in range(8):
            assert np.all(out[s, h] <= V[:, h // 4].max(axis=0) + TOL)
            assert np.all(out[s, h] >= V[:, h // 4].min(axis=0) - TOL)
    v1 = np.where(v == W.BF16_NAN, v, np.uint16(0x3F80))  # 1.0 wherever a token lives
    out, _ = decode_on(b, k, v1)
    assert np.abs(out - 1.0).max() < TOL


def test_decode_dominant_key():
    """Decode pin (vi): q = 8 k_j* => out ~= V[j*]."""
    b = small_batch(8, [40], Hq=2, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    K, V = dense_kv(b, k, v, b.compact_block_table, 0)
    jstar = 23
    for h in range(2):
        b.q[0, h] = bf16_bits_from_f32((8.0 * K[jstar, h]).astype(np.float32))
    out, _ = decode_on(b, k, v)
    for h in range(2):
        assert np.abs(out[0, h] - V[jstar, h]).max() < 1e-6


def test_probs_rows_sum_to_one_and_reproduce_output():
    """Decode pin (vii): rows of P sum to 1; out = P V."""
    b = small_batch(9, [17, 100], Hq=8, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    out, _ = decode_on(b, k, v)
    for s in range(2):
        _, V = dense_kv(b, k, v, b.compact_block_table, s)
        for h in (0, 3, 4, 7):
            P = oracle.decode_probs(b.q, k, v, b.compact_block_table, b.seq_lens, b.scale, s, h)
            assert abs(P.sum() - 1.0) < TOL and np.all(P > 0)
            assert np.abs(P @ V[:, h // 4] - out[s, h]).max() < TOL


def test_page_permutation_invariance():
    """Decode pin (viii): relabel physical pages (moving the data) => bit-identical output."""
    b = W.config1_tiny_decode()
    kf, vf = b.full_pool()
    numpy_scatter(b, kf, vf)
    o1, l1 = oracle.paged_decode(b.q, kf, vf, b.block_table, b.seq_lens, b.scale)
    perm = np.random.default_rng(10).permutation(b.num_pages)   # new id of old page i is perm[i]
    k2, v2 = np.empty_like(kf), np.empty_like(vf)
    k2[perm], v2[perm] = kf, vf
    bt2 = np.where(b.block_table >= 0, perm[np.maximum(b.block_table, 0)], -1).astype(np.int32)
    o2, l2 = oracle.paged_decode(b.q, k2, v2, bt2, b.seq_lens, b.scale)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_shared_prefix_equals_duplicated_prefix():
    """Decode pin (ix): two block-table rows naming the same pages == each owning a copy."""
    lens = [80, 80, 50, 50]
    b = small_batch(11, lens, Hq=4, Hkv=2, D=64, p=16, share_with=[-1, 0, -1, 2], shared_tokens=32, pool=64)
    assert np.array_equal(b.block_table[0, :2], b.block_table[1, :2])
    kf, vf = b.full_pool()
    numpy_scatter(b, kf, vf)
    o1, _ = oracle.paged_decode(b.q, kf, vf, b.block_table, b.seq_lens, b.scale)
    # duplicate: give sequences 1 and 3 private copies of the shared pages in unused pool pages
    free = [pg for pg in range(b.num_pages) if pg not in set(b.used_pages.tolist())]
    bt2 = b.block_table.copy()
    for s in (1, 3):
        for i in range(2):
            new = free.pop()
            kf[new], vf[new] = kf[bt2[s, i]], vf[bt2[s, i]]
            bt2[s, i] = new
    o2, _ = oracle.paged_decode(b.q, kf, vf, bt2, b.seq_lens, b.scale)
    assert np.array_equal(o1, o2)


def test_shift_invariance():
    """Decode pin (x): k_j <- k_j + c for all j leaves out unchanged (pins the max subtraction)."""
    b = small_batch(12, [37], Hq=2, Hkv=1, D=64)
    rng = np.random.default_rng(12)
    k, v = compact_pool_after_append(b)
    ki = rng.integers(-3, 4, size=k.shape).astype(np.float32)      # small integers: exact in bf16
    c = rng.integers(-2, 3, size=(64,)).astype(np.float32)
    b.q[:] = bf16_bits_from_f32(rng.integers(-2, 3, size=b.q.shape).astype(np.float32))
    o1, l1 = decode_on(b, bf16_bits_from_f32(ki), v)
    o2, l2 = decode_on(b, bf16_bits_from_f32(ki + c), v)
    assert np.abs(o1 - o2).max() < TOL
    shift = float(b.scale) * (f64_from_bf16_bits(b.q[0]) @ c.astype(np.float64))
    assert np.abs((l2 - l1)[0] - shift).max() < 1e-10


def test_gqa_equals_repeat_interleaved_mha():
    """GQA map kv = h div G: running with K/V heads repeat-interleaved to Hq gives the same result."""
    b = small_batch(13, [29, 64], Hq=6, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    o1, _ = decode_on(b, k, v)
    o2, _ = oracle.paged_decode(b.q, np.repeat(k, 3, axis=1), np.repeat(v, 3, axis=1),
                                b.compact_block_table, b.seq_lens, b.scale)
    assert np.array_equal(o1, o2)


def test_empty_sequence():
    """Reading R8: L = 0 => out = 0, lse = -inf."""
    b = small_batch(14, [0, 5], q_lens=[0, 1], Hq=2, Hkv=1, D=64)
    q = np.concatenate([b.q[:1], b.q], axis=0)      # decode wants one q row per sequence
    k, v = compact_pool_after_append(b)
    out, lse = oracle.paged_decode(q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    assert np.all(out[0] == 0) and np.all(np.isneginf(lse[0]))
    assert np.all(np.isfinite(out[1])) and np.all(np.isfinite(lse[1]))


@pytest.mark.parametrize("parts", [1, 2, 3, 16])
def test_split_merge_identity(parts):
    """Decode pin (xii): per-partition oracle merged with the (a3) formula == unsplit, incl. empty partitions."""
    b = small_batch(15, [100, 7], Hq=4, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    out, lse = decode_on(b, k, v)
    for s, L in enumerate([100, 7]):
        chunk = -(-max(L, 1) // parts)
        chunk = -(-chunk // 16) * 16          # page-aligned partitions, so some are empty
        for h in range(4):
            ms, ls, Os = [], [], []
            for i in range(parts):
                m, l, O = oracle.decode_partition(b.q, k, v, b.compact_block_table, b.seq_lens, b.scale,
                                                  s, h, i * chunk, (i + 1) * chunk)
                ms.append(m); ls.append(l); Os.append(O)
            if parts * chunk >= L:
                o, e = oracle.lse_combine(ms, ls, np.stack(Os))
                assert np.abs(o - out[s, h]).max() < TOL and abs(e - lse[s, h]) < TOL


def test_combine_closed_form():
    """COMBINE on hand-made partials: weights e^{m_i - M} written out."""
    m = np.array([0.0, math.log(3.0), -np.inf])
    l = np.array([2.0, 1.0, 0.0])
    O = np.array([[2.0, 4.0], [3.0, -3.0], [0.0, 0.0]])
    out, lse = oracle.lse_combine(m, l, O)
    # in units of e^{-M}, M = ln 3: weights 1/3, 1, 0 -> Z = 2/3 + 1, numerators 2/3+3, 4/3-3
    assert np.abs(out - np.array([(2 / 3 + 3) / (5 / 3), (4 / 3 - 3) / (5 / 3)])).max() < TOL
    assert abs(lse - math.log(2.0 + 3.0)) < TOL
    out, lse = oracle.lse_combine([-np.inf, -np.inf], [0.0, 0.0], np.zeros((2, 2)))
    assert np.all(out == 0) and np.isneginf(lse)


# ----------------------------------------------------------------------------- prefill

def prefill_on(batch, k, v, rows=None, causal=True):
    return oracle.paged_prefill(batch.q, batch.cu_seqlens_q, k, v, batch.compact_block_table,
                                batch.seq_lens, batch.scale, causal=causal, rows=rows)


@pytest.mark.parametrize("Hq,Hkv,D,p", [(4, 2, 64, 16), (7, 1, 128, 16), (4, 1, 64, 32)])
def test_prefill_matches_brute_force_with_explicit_mask(Hq, Hkv, D, p):
    """Prefill pin (i): explicit [n x L] mask matrix, bottom-right aligned (R6)."""
    lens = [40, 17, 33, 5, 64]
    qls = [40, 1, 16, 5, 3]          # prefix 0 / 16 / 17 / 0 / 61
    b = small_batch(20, lens, q_lens=qls, Hq=Hq, Hkv=Hkv, D=D, p=p)
    k, v = compact_pool_after_append(b)
    out, lse = prefill_on(b, k, v)
    ref, ref_lse = brute_force_attention(b, k, v, b.compact_block_table, causal=True)
    assert np.abs(out - ref).max() < TOL and np.abs(lse - ref_lse).max() < TOL
    out, lse = prefill_on(b, k, v, causal=False)
    ref, ref_lse = brute_force_attention(b, k, v, b.compact_block_table, causal=False)
    assert np.abs(out - ref).max() < TOL and np.abs(lse - ref_lse).max() < TOL


def test_prefill_row_subset_equals_full():
    b = small_batch(21, [50, 30], q_lens=[20, 30], Hq=4, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    full, full_lse = prefill_on(b, k, v)
    rows = np.array([0, 3, 19, 20, 49], dtype=np.int32)
    sub, sub_lse = prefill_on(b, k, v, rows=rows)
    assert np.array_equal(sub, full[rows]) and np.array_equal(sub_lse, full_lse[rows])


def test_prefill_one_token_equals_decode_and_last_row_equals_decode():
    """Prefill pins (ii) + (iii)."""
    b = small_batch(22, [1, 17, 33, 100], Hq=8, Hkv=2, D=64)          # n_s = 1 everywhere
    k, v = compact_pool_after_append(b)
    o_p, l_p = prefill_on(b, k, v)
    o_d, l_d = decode_on(b, k, v)
    assert np.array_equal(o_p, o_d) and np.array_equal(l_p, l_d)
    b2 = small_batch(23, [40, 70], q_lens=[25, 70], Hq=4, Hkv=2, D=64)
    k, v = compact_pool_after_append(b2)
    o_p, l_p = prefill_on(b2, k, v)
    last = b2.cu_seqlens_q[1:] - 1
    o_d, l_d = oracle.paged_decode(b2.q[last], k, v, b2.compact_block_table, b2.seq_lens, b2.scale)
    assert np.array_equal(o_p[last], o_d) and np.array_equal(l_p[last], l_d)


def test_prefill_first_row_without_prefix_is_v_row():
    """Prefill pin (iv): P = 0, i = 0 => V row 0."""
    b = small_batch(24, [30], q_lens=[30], Hq=4, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    out, _ = prefill_on(b, k, v, rows=np.array([0], np.int32))
    _, V = dense_kv(b, k, v, b.compact_block_table, 0)
    for h in range(4):
        assert np.array_equal(out[0, h], V[0, h // 2])


def test_prefill_causality_under_poisoned_future():
    """Prefill pin (v): +-1e30 in K/V at positions > P + i leaves row i unchanged."""
    b = small_batch(25, [60], q_lens=[20], Hq=2, Hkv=1, D=64)
    k, v = compact_pool_after_append(b)
    out, _ = prefill_on(b, k, v)
    big = bf16_bits_from_f32(np.array([1e30, -1e30], np.float32))
    for i in (0, 7, 18):
        k2, v2 = k.copy(), v.copy()
        j = np.arange(40 + i + 1, 60)
        k2[b.compact_block_table[0, j // 16], :, j % 16, :] = big[0]
        v2[b.compact_block_table[0, j // 16], :, j % 16, :] = big[1]
        o2, _ = prefill_on(b, k2, v2, rows=np.array([i], np.int32))
        assert np.array_equal(o2[0], out[i])


def test_chunked_prefill_identity():
    """Prefill pin (vii): prefill(n) == prefill(first half) then prefill(second half over prefix P + n/2)."""
    b = small_batch(26, [48], q_lens=[32], Hq=4, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    full, _ = prefill_on(b, k, v)
    # first half: sequence truncated to L = 16 + 16
    o1, _ = oracle.paged_prefill(b.q[:16], np.array([0, 16], np.int32), k, v, b.compact_block_table,
                                 np.array([32], np.int32), b.scale)
    o2, _ = oracle.paged_prefill(b.q[16:], np.array([0, 16], np.int32), k, v, b.compact_block_table,
                                 np.array([48], np.int32), b.scale)
    assert np.array_equal(full[:16], o1) and np.array_equal(full[16:], o2)


def test_bad_geometry_rejected():
    b = small_batch(27, [5], Hq=3, Hkv=2, D=64)
    k, v = compact_pool_after_append(b)
    with pytest.raises(ValueError):
        decode_on(b, k, v)


# ----------------------------------------------------------------------------- workloads

def test_workload_check_values():
    """The draws SURVEY.md 8(d) lists for numpy 2.3 (recipe restated in DESIGN.md)."""
    b2 = W.config2_bagel_cfg_decode()
    assert b2.num_seqs == 64 and b2.seq_lens[::2][:5].tolist() == [1584, 3308, 1409, 1936, 3386]
    assert int(b2.seq_lens[::2].sum()) == 76766
    assert np.array_equal(b2.block_table[0, :16], b2.block_table[1, :16])
    assert not np.intersect1d(b2.block_table[0, 16:99], b2.block_table[1, 16:99]).size
    assert b2.kv_bytes_logical() == 314433536 and b2.kv_bytes_unique() == 297656320
    b3 = W.config3_prefill()
    assert (b3.seq_lens - 1024).tolist() == [1965, 484, 381, 75, 282, 1019, 742, 704]
    b4 = W.config4_thinker()
    assert b4.seq_lens[:5].tolist() == [6018, 6754, 5165, 735, 590] and int(b4.seq_lens.sum()) == 147330
    b4t = W.config4_talker()
    assert b4t.seq_lens[:5].tolist() == [568, 77, 860, 75, 997] and int(b4t.seq_lens.sum()) == 67290
    b1 = W.config1_tiny_decode()
    assert b1.kv_bytes_logical() == 77312 and len(b1.used_pages) == 13


def test_bf16_rounding_is_rne():
    x = np.array([1.0, 1.00390625, 1.01171875, -2.5, 3.0e38, 1e-40], np.float32)
    # 1 + 2^-8 is a tie -> even (1.0); 1 + 3*2^-8 is a tie -> even (1 + 2^-6)
    bits = bf16_bits_from_f32(x)
    assert bits[0] == 0x3F80 and bits[1] == 0x3F80 and bits[2] == 0x3F82 and bits[3] == 0xC020
    assert np.array_equal(bf16_bits_from_f32(f64_from_bf16_bits(bits).astype(np.float32)), bits)
