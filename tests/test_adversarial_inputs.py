"""CPU checks of the adversarial value patterns (workloads/adversarial.py) and of the oracle on them: the properties
the GPU tests rely on hold BY CONSTRUCTION (the ramp moves the stage maximum by more than 8 log2 units at every stage;
a dominant key carries all the weight), checked here with plain numpy on the fp64 logits, and the oracle reproduces
the closed forms those patterns have (SURVEY 8(c) pins (iii), (vi))."""
import numpy as np
import pytest

import oracle
import workloads as W
from tests.util import compact_pool_after_append, f64_from_bf16_bits

LOG2E = 1.4426950408889634


def batch(kind, lens, q_lens, seed=1, Hq=14, Hkv=2, p=16, stage=128):
    rng = np.random.default_rng(seed)
    pages = sum((l + p - 1) // p for l in lens)
    b = W.make_batch(rng, "adv", lens, q_lens, Hq, Hkv, 128, p, 2 * pages)
    return W.make_adversarial(b, kind, stage=stage, seed=seed)


def logits(b, s, i, h):
    """fp64 logits of query row i (within sequence s), head h over all L positions (no mask)."""
    k, _ = W.logical_kv(b, s)
    G = b.num_q_heads // b.num_kv_heads
    q = f64_from_bf16_bits(b.q[int(b.cu_seqlens_q[s]) + i, h])
    return float(b.scale) * (f64_from_bf16_bits(k[:, h // G, :]) @ q)


def test_logical_kv_roundtrip_and_store_split():
    b = batch("q_zero", [100, 40], [30, 40])
    k, v = compact_pool_after_append(b)
    for s in range(2):
        kb, vb = W.logical_kv(b, s)
        L = int(b.seq_lens[s])
        j = np.arange(L)
        pg = b.compact_block_table[s, j // 16]
        assert np.array_equal(kb, k[pg, :, j % 16, :]) and np.array_equal(vb, v[pg, :, j % 16, :])


@pytest.mark.parametrize("stage", [64, 128])
def test_ramp_moves_the_stage_maximum_past_the_lazy_rescale_threshold(stage):
    b = batch("ramp", [1200, 700], [400, 1], stage=stage)
    for s, i, h in ((0, 399, 0), (0, 399, 2), (1, 0, 4)):
        x = logits(b, s, i, h) * LOG2E
        L = x.shape[0]
        mx = np.array([x[a:a + stage].max() for a in range(0, L, stage)])
        assert np.all(np.diff(mx) > 8.0), "even heads: every stage must raise the running max by > 2^8"
        assert np.all(np.diff(mx) < 16.0)
    x = logits(b, 0, 399, 1) * LOG2E   # odd heads: falling, the first stage holds the maximum for good
    mx = np.array([x[a:a + stage].max() for a in range(0, x.shape[0], stage)])
    assert np.all(np.diff(mx) < -8.0)


@pytest.mark.parametrize("kind,f", [("dominant_first", 0.0), ("dominant_mid", 0.5), ("dominant_last", 1.0)])
def test_dominant_key_pins_the_oracle_to_its_v_row(kind, f):
    """SURVEY 8(c) pin (vi): q = 8 k_j* => out = V[j*] to ~1e-12 (weights of the other keys < e^-40)."""
    b = batch(kind, [600, 300, 129], [200, 1, 129])
    k, v = compact_pool_after_append(b)
    out, _ = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    for s in range(3):
        _, vb = W.logical_kv(b, s)
        L, n = int(b.seq_lens[s]), int(b.q_lens[s])
        for i in (0, n // 2, n - 1):
            jstar = int(np.floor(f * (L - n + i)))
            x = logits(b, s, i, 3)[:L - n + i + 1]
            assert np.argmax(x) == jstar and (len(x) < 2 or x[jstar] - np.partition(x, -2)[-2] > 30.0)
            for h in (0, 3, 13):
                want = f64_from_bf16_bits(vb[jstar, h // 7])
                assert np.abs(out[int(b.cu_seqlens_q[s]) + i, h] - want).max() < 1e-9


def test_equal_logits_give_the_mean_of_v():
    for kind in ("q_zero", "k_const"):
        b = batch(kind, [333, 64], [1, 1])
        k, v = compact_pool_after_append(b)
        q = b.q[b.cu_seqlens_q[:-1]]
        out, lse = oracle.paged_decode(q, k, v, b.compact_block_table, b.seq_lens, b.scale)
        for s in range(2):
            _, vb = W.logical_kv(b, s)
            mean = f64_from_bf16_bits(vb).mean(axis=0)   # [Hkv, D]
            for h in (0, 8):
                assert np.abs(out[s, h] - mean[h // 7]).max() < 1e-12
            x0 = logits(b, s, 0, 0)
            assert np.ptp(x0) == 0.0 and abs(lse[s, 0] - (x0[0] + np.log(len(x0)))) < 1e-12


def test_huge_logits_reach_the_advertised_range():
    b = batch("huge", [3000], [1])
    x = logits(b, 0, 0, 0)
    assert 45.0 < x.max() < 110.0 and -110.0 < x.min() < -45.0
