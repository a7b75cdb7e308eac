"""CPU oracle of CUDA-graph-compatible token sampling: SURVEY 8(f) rank 4, last clause ("then CUDA-graph-compatible
sampling"); PAPER.md:134 names "a cuda-graph-compatible sampling plugin" of the KVCacheEngine and PAPER.md:230 credits
"cuda-graph-compatible sampling" for part of the Orpheus gain, without giving a definition.  The reading is DESIGN.md
R28.  TEST INFRASTRUCTURE ONLY: plain numpy / Python integers, fp64; shares no code with the CUDA path (both sides
implement the same published counter-based generator, Philox4x32-10, as the task's rules allow).

Definitions (one row = one sequence's logits over the vocabulary)
  UNIFORM(seed, step, row)   x = word 0 of Philox4x32-10 with counter (step mod 2^32, step div 2^32, row, 0) and key
                             (seed mod 2^32, seed div 2^32);  u = (x + 1/2) / 2^32, so 0 < u < 1.
  SUPPORT(logits, T, k, p)   z = logits / T.  top-k (0 < k < V): keep the tokens with z >= the k-th largest z (ties at
                             that value are all kept).  Probabilities q = softmax(z) over the kept tokens.  top-p
                             (0 < p < 1): order the kept tokens by q descending; take the shortest prefix whose mass is
                             >= p; keep the tokens with q >= the smallest q of that prefix (ties kept).
  SAMPLE                     T == 0: the argmax of the logits (lowest index among equals).  Otherwise, with the kept
                             tokens in INDEX order and c_i the running sum of their q: the first kept token with
                             c_i > u * (total mass of the kept tokens).
No state lives on the host: the same (seed, step) gives the same token, a replayed CUDA graph whose step counter is
device memory draws fresh numbers.
"""
from __future__ import annotations

import numpy as np

_M0, _M1 = 0xD2511F53, 0xCD9E8D57
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = 0xFFFFFFFF


def philox4x32_10(counter, key):
    """Philox4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3", SC'11),
    written out with Python integers.  counter: 4 words, key: 2 words -> 4 words."""
    c0, c1, c2, c3 = (int(x) & _MASK for x in counter)
    k0, k1 = (int(x) & _MASK for x in key)
    for r in range(10):
        if r:
            k0 = (k0 + _W0) & _MASK
            k1 = (k1 + _W1) & _MASK
        p0 = _M0 * c0
        p1 = _M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & _MASK, p1 & _MASK, ((p0 >> 32) ^ c3 ^ k1) & _MASK, p0 & _MASK
    return c0, c1, c2, c3


def uniform(seed: int, step: int, row: int) -> float:
    """UNIFORM: fp64 in (0, 1), exact."""
    x = philox4x32_10((step & _MASK, (step >> 32) & _MASK, row & _MASK, 0), (seed & _MASK, (seed >> 32) & _MASK))[0]
    return (x + 0.5) / 4294967296.0


def support(logits, temperature: float, top_k: int = 0, top_p: float = 1.0):
    """SUPPORT: (kept bool [V], q fp64 [V] = probabilities over the kept tokens, 0 elsewhere)."""
    z = np.asarray(logits, dtype=np.float64) / float(temperature)
    V = z.shape[0]
    kept = np.ones(V, dtype=bool)
    if 0 < top_k < V:
        kth = np.sort(z)[V - top_k]
        kept = z >= kth
    w = np.where(kept, np.exp(z - z[kept].max()), 0.0)
    q = w / w.sum()
    if 0.0 < top_p < 1.0:
        order = np.argsort(-q, kind="stable")
        cum = np.cumsum(q[order])
        n = int(np.searchsorted(cum, top_p, side="left")) + 1   # shortest prefix with mass >= top_p
        n = min(n, int(kept.sum()))
        thr = q[order[n - 1]]
        kept = kept & (q >= thr)
        w = np.where(kept, w, 0.0)
        q = w / w.sum()
    return kept, q


def sample(logits, temperature: float, top_k: int, top_p: float, u: float) -> int:
    """SAMPLE with a given uniform number u in (0, 1)."""
    logits = np.asarray(logits, dtype=np.float64)
    if temperature == 0.0:
        return int(np.argmax(logits))
    kept, q = support(logits, temperature, top_k, top_p)
    c = np.cumsum(q)                      # index order; q is 0 outside the support
    idx = np.flatnonzero(kept & (c > u * c[-1]))
    return int(idx[0]) if idx.size else int(np.flatnonzero(kept)[-1])


def sample_tokens(logits, temperature, top_k, top_p, seeds, step: int):
    """One token per row: logits [B, V]; temperature / top_k / top_p / seeds [B]; step = the shared counter."""
    logits = np.asarray(logits, dtype=np.float64)
    B = logits.shape[0]
    return np.array([sample(logits[r], float(temperature[r]), int(top_k[r]), float(top_p[r]),
                            uniform(int(seeds[r]), int(step), r)) for r in range(B)], dtype=np.int32)


def cdf_interval(logits, temperature: float, top_k: int, top_p: float, token: int):
    """(in support?, c_lo, c_hi): the slice of [0, 1) that maps to `token` (normalised running sums, index order)."""
    kept, q = support(logits, temperature, top_k, top_p)
    c = np.cumsum(q) / q.sum()
    return bool(kept[token]), float(c[token] - q[token] / q.sum()), float(c[token])
