"""Property tests (hypothesis) over small random geometries: page sizes {16, 32}, head_dim {64, 128},
group sizes {1, 4, 7, 8}, lengths that straddle page / tile / partition boundaries, seq_len 0 and 1, NaN-poisoned unused
slots (the generator poisons them).  CPU part: the oracle against the independent numpy brute force and its invariants.
GPU part: decode (fixed partitions and balanced), cascade decode, prefill (both kernels, causal and not) and the fp8
pool against the oracle, gates R11.  Derandomised: the same examples on every run."""
import numpy as np
import pytest
from hypothesis import HealthCheck, given, settings, strategies as st

import oracle
import workloads as W
from tests.util import brute_force_attention, check_parity, compact_pool_after_append, decode_q

EDGE = [0, 1, 2, 15, 16, 17, 31, 32, 33, 63, 64, 65, 127, 128, 129, 200, 257]
geometry = st.tuples(st.sampled_from([16, 32]), st.sampled_from([64, 128]), st.sampled_from([1, 4, 7, 8]),
                     st.sampled_from([1, 2, 3]))
lens = st.lists(st.sampled_from(EDGE), min_size=1, max_size=6)
# soak runs (profiles/r2_sanitizer.md): MSTAR_SOAK=k multiplies the number of examples of every property below;
# MSTAR_SOAK_RANDOM=1 lifts the derandomisation, so that `pytest --hypothesis-seed=N` draws other examples
import os as _os
_SOAK = max(1, int(_os.environ.get("MSTAR_SOAK", "1")))
SET = dict(deadline=None, derandomize=not _os.environ.get("MSTAR_SOAK_RANDOM"), database=None,
           suppress_health_check=list(HealthCheck))
_settings = settings


def settings(max_examples=100, **kw):   # noqa: F811 -- the decorator below, scaled
    return _settings(max_examples=max_examples * _SOAK, **kw)


def decode_batch(seed, geo, L):
    p, D, G, Hkv = geo
    pages = sum((l + p - 1) // p for l in L)
    return W.make_batch(np.random.default_rng(seed), "prop", L, [min(1, l) for l in L], G * Hkv, Hkv, D, p,
                        2 * pages + 3)


def prefill_batch(seed, geo, L, frac):
    p, D, G, Hkv = geo
    n = [int(round(l * f)) for l, f in zip(L, frac)]
    n = [min(max(x, 1 if l > 0 else 0), l) for x, l in zip(n, L)]
    pages = sum((l + p - 1) // p for l in L)
    return W.make_batch(np.random.default_rng(seed), "prop", L, n, G * Hkv, Hkv, D, p, 2 * pages + 3)


# ----------------------------------------------------------------------------- CPU: the oracle

@settings(max_examples=25, **SET)
@given(seed=st.integers(0, 2 ** 20), geo=geometry, L=lens)
def test_oracle_decode_equals_brute_force_and_is_page_relabelling_invariant(seed, geo, L):
    b = decode_batch(seed, geo, L)
    k, v = compact_pool_after_append(b)
    got, lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    want, want_lse = brute_force_attention(b, k, v, b.compact_block_table, causal=True)
    has = b.q_lens > 0
    assert np.abs(got[has] - want).max(initial=0.0) < 1e-12
    assert np.abs(lse[has] - want_lse).max(initial=0.0) < 1e-12
    assert not got[~has].any() and np.all(np.isneginf(lse[~has]))
    # relabel the physical pages: bit-identical
    U = k.shape[0]
    if U == 0:
        return
    perm = np.random.default_rng(seed + 1).permutation(U)
    inv = np.argsort(perm)
    bt = np.where(b.compact_block_table >= 0, inv[np.maximum(b.compact_block_table, 0)], -1).astype(np.int32)
    got2, lse2 = oracle.paged_decode(decode_q(b), k[perm], v[perm], bt, b.seq_lens, b.scale)
    assert np.array_equal(got, got2) and np.array_equal(lse, lse2)


@settings(max_examples=20, **SET)
@given(seed=st.integers(0, 2 ** 20), geo=geometry, L=lens, causal=st.booleans(),
       frac=st.lists(st.sampled_from([0.0, 0.1, 0.5, 1.0]), min_size=6, max_size=6))
def test_oracle_prefill_equals_brute_force(seed, geo, L, causal, frac):
    b = prefill_batch(seed, geo, L, frac)
    k, v = compact_pool_after_append(b)
    got, lse = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale, causal=causal)
    want, want_lse = brute_force_attention(b, k, v, b.compact_block_table, causal=causal)
    assert np.abs(got - want).max(initial=0.0) < 1e-12 and np.abs(lse - want_lse).max(initial=0.0) < 1e-12


@settings(max_examples=20, **SET)
@given(seed=st.integers(0, 2 ** 20), geo=geometry, L=st.sampled_from([1, 17, 64, 129, 257]),
       parts=st.sampled_from([1, 2, 3, 16]))
def test_oracle_split_then_combine_is_unsplit(seed, geo, L, parts):
    b = decode_batch(seed, geo, [L])
    k, v = compact_pool_after_append(b)
    q = decode_q(b)
    full, full_lse = oracle.paged_decode(q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    chunk = (L + parts - 1) // parts
    for h in range(b.num_q_heads):
        m, l, o = [], [], []
        for i in range(parts):
            a, e = i * chunk, min(L, (i + 1) * chunk)
            mi, li, oi = oracle.decode_partition(q, k, v, b.compact_block_table, b.seq_lens, b.scale, 0, h, a, max(a, e))
            m.append(mi); l.append(li); o.append(oi)
        out, lse = oracle.lse_combine(np.array(m), np.array(l), np.stack(o))
        assert np.abs(out - full[0, h]).max() < 1e-12 and abs(lse - full_lse[0, h]) < 1e-12


# ----------------------------------------------------------------------------- GPU: the CUDA path against the oracle

@pytest.mark.gpu
@settings(max_examples=30, **SET)
@given(seed=st.integers(0, 2 ** 20), geo=geometry, L=lens, parts=st.sampled_from([0, 1, 2, 3, 16]))
def test_gpu_decode_random_geometry(seed, geo, L, parts):
    from tests.gpu_util import DeviceBatch, f64_of
    b = decode_batch(seed, geo, L)
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    db = DeviceBatch(b)
    db.append()
    out, lse = db.decode(num_partitions=parts)
    check_parity(f64_of(out), want, "decode %s %s parts=%d" % (geo, L, parts))
    got_lse = f64_of(lse)
    fin = np.isfinite(want_lse)
    assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse))
    assert np.abs(got_lse[fin] - want_lse[fin]).max(initial=0.0) < 2e-3


@pytest.mark.gpu
@settings(max_examples=20, **SET)
@given(seed=st.integers(0, 2 ** 20), geo=geometry, B=st.sampled_from([2, 3]),
       shared=st.lists(st.sampled_from([0, 1, 2, 5]), min_size=1, max_size=3),
       sfx=st.lists(st.sampled_from([1, 2, 15, 16, 17, 63, 64, 65, 130]), min_size=9, max_size=9))
def test_gpu_cascade_decode_random_geometry(seed, geo, B, shared, sfx):
    from tests.gpu_util import DeviceBatch, f64_of
    from tests.test_gpu_cascade import cfg_batch
    p, D, G, Hkv = geo
    shared_r = [s * p for s in shared]
    sf = [[sfx[(r * B + j) % 9] for j in range(B)] for r in range(len(shared_r))]
    b = cfg_batch(seed, shared_r, sf, B, G * Hkv, Hkv, D, p)
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    db = DeviceBatch(b)
    db.append()
    out, lse = db.decode_cascade(B, shared_r)
    check_parity(f64_of(out), want, "cascade %s" % (geo,))
    assert np.abs(f64_of(lse) - want_lse).max() < 2e-3


@pytest.mark.gpu
@settings(max_examples=30, **SET)
@given(seed=st.integers(0, 2 ** 20), geo=geometry, L=lens, causal=st.booleans(), mma_sync=st.booleans(),
       frac=st.lists(st.sampled_from([0.0, 0.1, 0.5, 1.0]), min_size=6, max_size=6))
def test_gpu_prefill_random_geometry(seed, geo, L, causal, mma_sync, frac):
    from tests.gpu_util import DeviceBatch, f64_of
    b = prefill_batch(seed, geo, L, frac)
    if b.total_q == 0:
        return
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale,
                                          causal=causal)
    db = DeviceBatch(b)
    db.append()
    out, lse = db.prefill(causal=causal, mma_sync=mma_sync)
    check_parity(f64_of(out), want, "prefill %s %s causal=%d mma_sync=%d" % (geo, L, causal, mma_sync))
    assert np.abs(f64_of(lse) - want_lse).max(initial=0.0) < 2e-3


@pytest.mark.gpu
@settings(max_examples=15, **SET)
@given(seed=st.integers(0, 2 ** 20), p=st.sampled_from([16, 32]), G=st.sampled_from([1, 4, 7, 8]), L=lens,
       causal=st.booleans(), frac=st.lists(st.sampled_from([0.0, 0.1, 0.5, 1.0]), min_size=6, max_size=6))
def test_gpu_fp8_pool_random_geometry(seed, p, G, L, causal, frac):
    """Quantised pool: codes bit-exact, decode and prefill within the gates."""
    from oracle import fp8 as ofp8
    from tests.gpu_util import DeviceBatchFp8, f64_of
    from tests.test_gpu_fp8 import oracle_pool
    geo = (p, 128, G, 2)
    for kind in ("decode", "prefill"):
        b = decode_batch(seed, geo, L) if kind == "decode" else prefill_batch(seed, geo, L, frac)
        if b.total_q == 0:
            continue
        ks, vs = W.fp8_page_scales(seed % 97, b.num_pages, b.num_kv_heads)
        db = DeviceBatchFp8(b, ks, vs)
        db.quantise_store()
        db.append()
        k8, v8, cks, cvs = oracle_pool(b, ks, vs)
        gk, gv = db.store_codes()
        assert np.array_equal(gk, k8) and np.array_equal(gv, v8)
        if kind == "decode":
            want, _ = ofp8.paged_decode_fp8(decode_q(b), k8, v8, cks, cvs, b.compact_block_table, b.seq_lens, b.scale)
            out, _ = db.decode(num_partitions=0)
        else:
            want, _ = ofp8.paged_prefill_fp8(b.q, b.cu_seqlens_q, k8, v8, cks, cvs, b.compact_block_table, b.seq_lens,
                                             b.scale, causal=causal)
            out, _ = db.prefill(causal=causal)
        check_parity(f64_of(out), want, "fp8 %s p=%d G=%d %s" % (kind, p, G, L))


@pytest.mark.gpu
@settings(max_examples=25, **SET)
@given(seed=st.integers(0, 2 ** 20), V=st.sampled_from([1, 2, 3, 31, 32, 33, 257, 1000, 4096, 4097, 8193, 16385, 20011]),
       sigma=st.sampled_from([0.0, 0.5, 2.0, 6.0]), bf16=st.booleans(), step=st.sampled_from([0, 1, 2 ** 32 + 3]))
def test_gpu_sampling_random_rows(seed, V, sigma, bf16, step):
    """Sampling (R28): every token valid against the oracle's fp64 interval, and the cluster kernel (1, 2, 4 or 8
    CTAs per row by V) equal to the one-CTA kernel, on random rows with random filters."""
    import torch
    from tests.test_gpu_sampling import check_rows, run, unambiguous
    rng = np.random.default_rng(seed)
    B = 12
    dtype = torch.bfloat16 if bf16 else torch.float32
    lg = np.float32(rng.normal(0, 1, (B, V)) * sigma)
    T = np.float32(rng.choice([0.0, 0.4, 1.0, 1.9], B))
    K = rng.choice([0, 1, 3, 40, V], B).astype(np.int32)
    P = np.float32(rng.choice([1.0, 0.97, 0.6, 0.1], B))
    seeds = rng.integers(0, 2 ** 62, B)
    a, lg64, _ = run(lg, T, K, P, seeds, step, dtype=dtype)
    b, _, _ = run(lg, T, K, P, seeds, step, dtype=dtype, one_cta=True)
    assert np.array_equal(a, b)
    ok = np.array([T[r] == 0 or unambiguous(lg64[r], float(T[r]), int(K[r]) if K[r] < V else 0, float(P[r]))
                   for r in range(B)])
    if ok.any():   # rows whose top-k / top-p cut is within rounding have several valid supports: not checked
        check_rows(a[ok], lg64[ok], T[ok], K[ok], P[ok], seeds[ok], step, rows=np.flatnonzero(ok))


BIG_LENS = st.lists(st.integers(0, 5000), min_size=2, max_size=8)


@pytest.mark.gpu
@settings(max_examples=6, **SET)
@given(seed=st.integers(0, 2 ** 20), p=st.sampled_from([16, 32]), D=st.sampled_from([64, 128]),
       G=st.sampled_from([1, 2, 4, 7, 8, 12, 16]), Hkv=st.sampled_from([1, 2, 4]), L=BIG_LENS,
       parts=st.sampled_from([0, 0, 1, 2, 5, 16]), causal=st.booleans(),
       frac=st.lists(st.sampled_from([0.0, 0.02, 0.3, 1.0]), min_size=8, max_size=8))
def test_gpu_large_random_geometry(seed, p, D, G, Hkv, L, parts, causal, frac):
    """Lengths up to 5000 (tens of KV stages and work units per sequence, ragged across the batch), every group
    size and both head dims: decode on all rows, prefill (tcgen05 kernel) on sampled rows of every sequence."""
    from tests.gpu_util import DeviceBatch, f64_of
    geo = (p, D, G, Hkv)
    what = "large %s %s" % (geo, L)
    # decode
    b = decode_batch(seed, geo, L)
    if b.total_q:
        k, v = compact_pool_after_append(b)
        want, want_lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
        db = DeviceBatch(b)
        db.append()
        out, lse = db.decode(num_partitions=parts)
        check_parity(f64_of(out), want, "decode " + what)
        got_lse = f64_of(lse)
        fin = np.isfinite(want_lse)
        assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse))
        assert np.abs(got_lse[fin] - want_lse[fin]).max(initial=0.0) < 2e-3
    # prefill
    b = prefill_batch(seed + 1, geo, L, frac)
    if b.total_q:
        k, v = compact_pool_after_append(b)
        rng = np.random.default_rng(seed)
        rows = np.unique(np.concatenate([rng.integers(0, b.total_q, 48), b.cu_seqlens_q[:-1][b.q_lens > 0],
                                         (b.cu_seqlens_q[1:] - 1)[b.q_lens > 0]]))
        want, want_lse = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale,
                                              causal=causal, rows=rows)
        db = DeviceBatch(b)
        db.append()
        out, lse = db.prefill(causal=causal)
        check_parity(f64_of(out)[rows], want, "prefill " + what)
        assert np.abs(f64_of(lse)[rows] - want_lse).max(initial=0.0) < 2e-3


@pytest.mark.gpu
@settings(max_examples=5, **SET)
@given(seed=st.integers(0, 2 ** 20), p=st.sampled_from([16, 32]), G=st.sampled_from([1, 4, 7, 8, 12, 16]),
       Hkv=st.sampled_from([1, 2, 4]), L=st.lists(st.integers(0, 3000), min_size=2, max_size=7),
       long_one=st.sampled_from([0, 0, 8300, 12000]), parts=st.sampled_from([0, 0, 1, 3, 16]), causal=st.booleans(),
       frac=st.lists(st.sampled_from([0.0, 0.02, 0.3, 1.0]), min_size=8, max_size=8))
def test_gpu_fp8_large_random_geometry(seed, p, G, Hkv, L, long_one, parts, causal, frac):
    """The quantised pool on long ragged batches: a sequence past 8192 tokens selects the 12-warp decode kernel
    (G <= 8); decode on all rows, the fp8 prefill on sampled rows."""
    from oracle import fp8 as ofp8
    from tests.gpu_util import DeviceBatchFp8, f64_of
    from tests.test_gpu_fp8 import oracle_pool
    geo = (p, 128, G, Hkv)
    L = list(L) + ([long_one] if long_one else [])
    what = "fp8 large %s %s" % (geo, L)
    b = decode_batch(seed, geo, L)
    if b.total_q:
        ks, vs = W.fp8_page_scales(seed % 89, b.num_pages, b.num_kv_heads)
        db = DeviceBatchFp8(b, ks, vs)
        db.quantise_store()
        db.append()
        k8, v8, cks, cvs = oracle_pool(b, ks, vs)
        want, want_lse = ofp8.paged_decode_fp8(decode_q(b), k8, v8, cks, cvs, b.compact_block_table, b.seq_lens, b.scale)
        out, lse = db.decode(num_partitions=parts)
        check_parity(f64_of(out), want, "decode " + what)
        fin = np.isfinite(want_lse)
        assert np.abs(f64_of(lse)[fin] - want_lse[fin]).max(initial=0.0) < 2e-3
        del db
    Ls = [min(l, 3000) for l in L]
    b = prefill_batch(seed + 1, geo, Ls, frac)
    if b.total_q:
        ks, vs = W.fp8_page_scales(seed % 83, b.num_pages, b.num_kv_heads)
        db = DeviceBatchFp8(b, ks, vs)
        db.quantise_store()
        db.append()
        k8, v8, cks, cvs = oracle_pool(b, ks, vs)
        rng = np.random.default_rng(seed)
        rows = np.unique(np.concatenate([rng.integers(0, b.total_q, 32), b.cu_seqlens_q[:-1][b.q_lens > 0],
                                         (b.cu_seqlens_q[1:] - 1)[b.q_lens > 0]]))
        want, _ = ofp8.paged_prefill_fp8(b.q, b.cu_seqlens_q, k8, v8, cks, cvs, b.compact_block_table, b.seq_lens,
                                         b.scale, causal=causal, rows=rows)
        out, _ = db.prefill(causal=causal)
        check_parity(f64_of(out)[rows], want, "prefill " + what)


@pytest.mark.gpu
@settings(max_examples=6, **SET)
@given(seed=st.integers(0, 2 ** 20), p=st.sampled_from([16, 32]), D=st.sampled_from([64, 128]),
       G=st.sampled_from([1, 4, 7, 8, 12]), B=st.sampled_from([2, 3, 4]),
       shared=st.lists(st.integers(0, 200), min_size=1, max_size=5),
       sfx=st.lists(st.integers(1, 700), min_size=20, max_size=20))
def test_gpu_cascade_large_random_geometry(seed, p, D, G, B, shared, sfx):
    """Cascade decode with shared contexts up to 200 pages and private suffixes up to 700 tokens, 2 to 4 branches."""
    from tests.gpu_util import DeviceBatch, f64_of
    from tests.test_gpu_cascade import cfg_batch
    shared_r = [s * p for s in shared]
    sf = [[sfx[(r * B + j) % 20] for j in range(B)] for r in range(len(shared_r))]
    b = cfg_batch(seed, shared_r, sf, B, G * 2, 2, D, p)
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    db = DeviceBatch(b)
    db.append()
    out, lse = db.decode_cascade(B, shared_r)
    check_parity(f64_of(out), want, "cascade large p=%d D=%d G=%d B=%d" % (p, D, G, B))
    assert np.abs(f64_of(lse) - want_lse).max() < 2e-3


@pytest.mark.gpu
@settings(max_examples=8, **SET)
@given(seed=st.integers(0, 2 ** 20), kind=st.sampled_from(list(W.ADVERSARIAL_KINDS)), p=st.sampled_from([16, 32]),
       D=st.sampled_from([64, 128]), G=st.sampled_from([1, 4, 7, 8, 16]),
       L=st.lists(st.integers(1, 1500), min_size=1, max_size=5), parts=st.sampled_from([0, 1, 3, 16]),
       causal=st.booleans(), frac=st.lists(st.sampled_from([0.02, 0.3, 1.0]), min_size=5, max_size=5))
def test_gpu_adversarial_values_random_geometry(seed, kind, p, D, G, L, parts, causal, frac):
    """The adversarial value patterns (dominant keys, the ramp that forces the lazy rescale, huge logits, zero
    queries, constant keys) on random geometries: decode and both prefill kernels against the oracle."""
    from tests.gpu_util import DeviceBatch, f64_of
    geo = (p, D, G, 2)
    what = "%s %s %s" % (kind, geo, L)
    b = W.make_adversarial(decode_batch(seed, geo, L), kind, stage=64, seed=seed)
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    db = DeviceBatch(b)
    db.append()
    out, lse = db.decode(num_partitions=parts)
    check_parity(f64_of(out), want, "decode " + what)
    assert np.abs(f64_of(lse) - want_lse).max(initial=0.0) < 2e-3
    b = W.make_adversarial(prefill_batch(seed + 1, geo, L, frac), kind, stage=128, seed=seed)
    k, v = compact_pool_after_append(b)
    want, _ = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale, causal=causal)
    db = DeviceBatch(b)
    db.append()
    for mma_sync in (False, True):
        out, _ = db.prefill(causal=causal, mma_sync=mma_sync)
        check_parity(f64_of(out), want, "prefill %s mma_sync=%d" % (what, mma_sync))
