"""Adversarial value patterns for the parity tests (inputs only, no attention arithmetic).

The five BASELINE configs draw Q, K, V ~ N(0,1), so every logit is ~N(0,1) and the online-softmax machinery of
the kernels (running-max updates, lazy rescale of O, exp2 underflow, split-K combine weights that differ by many
orders of magnitude) is barely exercised.  The functions here take a seeded ``PagedBatch`` and overwrite Q and/or
the K rows of its sequences with structured values (pin (vi) "one dominant key (q = 8 k_j*)"
and the edge cases VERDICT r1 lists): copies and scalings of rows, nothing of the method's arithmetic.  The same
16-bit words then go to the oracle and to the device, as for every other batch.

A sequence's logical token j lives in the compact store (j < L - n, the cached prefix) or in ``k_new`` / ``v_new``
(the step's n new rows); ``logical_kv`` / ``overwrite_k`` hide that split.
"""
from __future__ import annotations

import numpy as np

from .generators import PagedBatch, bf16_bits_from_f32, f64_from_bf16_bits

KINDS = ("dominant_first", "dominant_mid", "dominant_last", "ramp", "huge", "q_zero", "k_const")


def _f32(bits: np.ndarray) -> np.ndarray:
    return f64_from_bf16_bits(bits).astype(np.float32)


def logical_kv(b: PagedBatch, s: int):
    """K, V bit patterns uint16 [L, Hkv, D] of sequence s in token order (prefix from the store, then the new rows)."""
    p = b.page_size
    L, n = int(b.seq_lens[s]), int(b.q_lens[s])
    P = L - n
    j = np.arange(P, dtype=np.int64)
    u = b.compact_block_table[s, j // p].astype(np.int64)
    t0 = int(b.cu_seqlens_q[s])
    k = np.concatenate([b.k_store[u, :, j % p, :], b.k_new[t0:t0 + n]], axis=0)
    v = np.concatenate([b.v_store[u, :, j % p, :], b.v_new[t0:t0 + n]], axis=0)
    return k, v


def overwrite_k(b: PagedBatch, s: int, k_bits: np.ndarray) -> None:
    """Write K rows uint16 [L, Hkv, D] of sequence s back (prefix rows to the store, the last n rows to k_new)."""
    _overwrite(b, s, k_bits, b.k_store, b.k_new)


def overwrite_v(b: PagedBatch, s: int, v_bits: np.ndarray) -> None:
    """The same for V."""
    _overwrite(b, s, v_bits, b.v_store, b.v_new)


def _overwrite(b: PagedBatch, s: int, bits: np.ndarray, store: np.ndarray, new: np.ndarray) -> None:
    p = b.page_size
    L, n = int(b.seq_lens[s]), int(b.q_lens[s])
    P = L - n
    assert bits.shape[0] == L
    j = np.arange(P, dtype=np.int64)
    u = b.compact_block_table[s, j // p].astype(np.int64)
    store[u, :, j % p, :] = bits[:P]
    t0 = int(b.cu_seqlens_q[s])
    new[t0:t0 + n] = bits[P:]


def make_adversarial(b: PagedBatch, kind: str, stage: int = 128, seed: int = 0) -> PagedBatch:
    """Overwrite Q (and for some kinds K) of ``b`` in place and return it.

    dominant_first / _mid / _last
        q[row, h] = 8 * k[j*, h div G] with j* = floor(f * (last visible position of the row)), f = 0, 0.5, 1:
        one key carries essentially all the weight; it sits in the first KV stage, a middle one, or is the very
        last visible key (the masked diagonal stage of a causal prefill, the last partition of a decode).
    ramp
        k_j = t_j * u + 0.1 * noise with u in {-1, +1}^D per kv head and t_j = 0.25 * (1 + j div stage);
        q[row, h] = +-2.828125 * u (sign + for even h, - for odd h).  With scale = 1/sqrt(D), D = 128 the logits of
        even heads grow by 8.0 nats = 11.5 log2 units from each ``stage`` tokens to the next (the running max moves at
        every stage, by more than any lazy-rescale threshold of 8), those of odd heads fall by as much (everything
        after the first stage underflows).  Keep L <= 32 * stage so that t_j stays exactly representable.
    huge
        q *= 20: logits ~ N(0, 20^2), maxima near +-70.  V *= 0.5 (exact): a row's weight then sits on one or two keys,
        so outputs are as large as single V elements, and N(0,1) rows reach |v| > 4 where half an ulp of a bf16 OUTPUT
        alone is 1.56e-2 -- no bf16-output kernel can meet the 2e-2 max-abs gate there (the oracle-exact result
        rounded to bf16 already sits at 1.56e-2).  Halving V keeps outputs inside (-4, 4), where the gate is reachable.
    q_zero
        q = 0: all logits equal (0), the output is the plain mean of the visible V rows.
    k_const
        every K row of a sequence equals its first row: all logits of a (row, head) equal, but not zero.
    """
    assert kind in KINDS, kind
    G = b.num_q_heads // b.num_kv_heads
    D = b.head_dim
    rng = np.random.default_rng(9000 + seed)
    for s in range(b.num_seqs):
        L, n = int(b.seq_lens[s]), int(b.q_lens[s])
        if L == 0 or n == 0:
            continue
        t0 = int(b.cu_seqlens_q[s])
        k_bits, v_bits = logical_kv(b, s)
        if kind.startswith("dominant"):
            f = {"dominant_first": 0.0, "dominant_mid": 0.5, "dominant_last": 1.0}[kind]
            kf = _f32(k_bits)                                   # [L, Hkv, D]
            last_visible = (L - n) + np.arange(n)               # decode (n = 1): L - 1
            jstar = np.floor(f * last_visible).astype(np.int64)
            q = np.float32(8.0) * np.repeat(kf[jstar], G, axis=1)   # [n, Hq, D]; times 8 is exact in bf16
            b.q[t0:t0 + n] = bf16_bits_from_f32(q)
        elif kind == "ramp":
            assert L <= 32 * stage, "ramp: t_j must stay exactly representable in bf16"
            u = rng.choice(np.array([-1.0, 1.0], dtype=np.float32), size=(b.num_kv_heads, D))
            t = (0.25 * (1 + np.arange(L) // stage)).astype(np.float32)
            noise = rng.standard_normal((L, b.num_kv_heads, D), dtype=np.float32) * np.float32(0.1)
            overwrite_k(b, s, bf16_bits_from_f32(t[:, None, None] * u[None] + noise))
            sign = np.where(np.arange(b.num_q_heads) % 2 == 0, 1.0, -1.0).astype(np.float32)
            q = np.float32(2.828125) * sign[None, :, None] * np.repeat(u, G, axis=0)[None]
            b.q[t0:t0 + n] = bf16_bits_from_f32(np.broadcast_to(q, (n, b.num_q_heads, D)))
        elif kind == "huge":
            b.q[t0:t0 + n] = bf16_bits_from_f32(_f32(b.q[t0:t0 + n]) * np.float32(20.0))
            overwrite_v(b, s, bf16_bits_from_f32(_f32(v_bits) * np.float32(0.5)))
        elif kind == "q_zero":
            b.q[t0:t0 + n] = 0
        elif kind == "k_const":
            overwrite_k(b, s, np.broadcast_to(k_bits[:1], k_bits.shape).copy())
    b.name = "%s[%s]" % (b.name, kind)
    return b
