"""Seeded generators for paged-KV batches (inputs only, no attention arithmetic).

Layout conventions (the ones ``include/mstar_attn.h`` documents):

* pool          ``[num_pages, Hkv, page_size, D]`` bf16 ("HND"), K and V separate
* block_table   ``[S, max_pages]`` int32, row s lists the physical page of logical
                page 0, 1, ...; entries past ceil(L_s / page_size) are -1
* seq_lens      ``[S]`` int32, KV length L_s *including* this step's new tokens
* q             ``[T, Hq, D]`` bf16, ragged over sequences by ``cu_seqlens_q``
* k_new, v_new  ``[T, Hkv, D]`` bf16, the step's new rows (the last n_s tokens of s)
* slot_mapping  ``[T]`` int64, page * page_size + offset of every new row

bf16 values travel as uint16 bit patterns (numpy has no bf16 dtype).  Every
slot of a used page that holds no token yet (tail of the last page, and the
slots the step's append will fill) and every unused page is NaN poison
(0x7FC0): results must not depend on them.

To keep the 60 GiB pool of config 5 off the host, the K/V data live in a
*compact store* holding only the pages some sequence references, with
``used_pages[u]`` the physical page id of store row u and ``compact_*`` copies
of the block table / slot mapping indexing the store instead of the pool.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np

BF16_NAN = np.uint16(0x7FC0)
CONFIG_SEED_BASE = 202606120  # rng seed of config c is CONFIG_SEED_BASE + c


def bf16_bits_from_f32(x: np.ndarray) -> np.ndarray:
    """Round float32 to bf16 (round-to-nearest-even), return the uint16 bit patterns."""
    b = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rnd = ((b >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((b + rnd) >> np.uint32(16)).astype(np.uint16)


def f64_from_bf16_bits(bits: np.ndarray) -> np.ndarray:
    """Widen bf16 bit patterns to float64 (exact).  Format conversion only."""
    u = np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(np.float64)


def _normal_bf16(rng: np.random.Generator, shape, chunk_elems: int = 1 << 26) -> np.ndarray:
    """N(0,1) float32 draws rounded to bf16 bits, drawn in flat order in bounded chunks."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    pos = 0
    while pos < n:
        m = min(chunk_elems, n - pos)
        out[pos:pos + m] = bf16_bits_from_f32(rng.standard_normal(m, dtype=np.float32))
        pos += m
    return out.reshape(shape)


@dataclasses.dataclass
class PagedBatch:
    name: str
    num_seqs: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    page_size: int
    num_pages: int
    scale: np.float32
    seq_lens: np.ndarray          # int32 [S]
    q_lens: np.ndarray            # int32 [S]
    cu_seqlens_q: np.ndarray      # int32 [S+1]
    block_table: np.ndarray       # int32 [S, max_pages], physical page ids, -1 tail
    q: np.ndarray                 # uint16 [T, Hq, D]
    k_new: np.ndarray             # uint16 [T, Hkv, D]
    v_new: np.ndarray             # uint16 [T, Hkv, D]
    slot_mapping: np.ndarray      # int64 [T]
    used_pages: np.ndarray        # int64 [U]
    k_store: np.ndarray           # uint16 [U, Hkv, p, D], state BEFORE the append
    v_store: np.ndarray           # uint16 [U, Hkv, p, D]
    compact_block_table: np.ndarray   # int32 [S, max_pages], store rows, -1 tail
    compact_slot_mapping: np.ndarray  # int64 [T]

    @property
    def total_q(self) -> int:
        return int(self.cu_seqlens_q[-1])

    @property
    def max_seq_len(self) -> int:
        return int(self.seq_lens.max()) if self.num_seqs else 0

    @property
    def max_q_len(self) -> int:
        return int(self.q_lens.max()) if self.num_seqs else 0

    def full_pool(self):
        """Materialise the whole pool on the host (small configs only): NaN poison + store rows."""
        shape = (self.num_pages, self.num_kv_heads, self.page_size, self.head_dim)
        k = np.full(shape, BF16_NAN, dtype=np.uint16)
        v = np.full(shape, BF16_NAN, dtype=np.uint16)
        k[self.used_pages] = self.k_store
        v[self.used_pages] = self.v_store
        return k, v

    def kv_bytes_logical(self) -> int:
        """sum_s L_s * 2 * Hkv * D * 2 B -- the algorithmic K/V read of one attention call."""
        return int(self.seq_lens.astype(np.int64).sum()) * 2 * self.num_kv_heads * self.head_dim * 2

    def kv_bytes_unique(self) -> int:
        """Same, counting a physical (page, slot) shared by several sequences once."""
        p = self.page_size
        best = {}
        for s in range(self.num_seqs):
            L = int(self.seq_lens[s])
            for i in range((L + p - 1) // p):
                pg = int(self.block_table[s, i])
                best[pg] = max(best.get(pg, 0), min(p, L - i * p))
        return sum(best.values()) * 2 * self.num_kv_heads * self.head_dim * 2


def make_batch(
    rng: np.random.Generator,
    name: str,
    seq_lens: Sequence[int],
    q_lens: Sequence[int],
    num_q_heads: int,
    num_kv_heads: int,
    head_dim: int,
    page_size: int,
    num_pages: int,
    share_with: Optional[Sequence[int]] = None,
    shared_tokens=0,
    table_width: Optional[int] = None,
) -> PagedBatch:
    """Draw one batch.  Draw order: page permutation, Q, K store, V store.

    ``share_with[s] = r`` (r < s) makes sequence s reuse the physical pages of the
    first ``shared_tokens`` tokens of sequence r (``shared_tokens`` must be a
    multiple of ``page_size`` and <= both lengths minus their new tokens; an int for
    the whole batch or one value per sequence).
    """
    S = len(seq_lens)
    p, D, Hq, Hkv = page_size, head_dim, num_q_heads, num_kv_heads
    seq_lens = np.asarray(seq_lens, dtype=np.int32).reshape(S)
    q_lens = np.asarray(q_lens, dtype=np.int32).reshape(S)
    assert np.all(q_lens <= seq_lens) and np.all(q_lens >= 0)
    n_pages_seq = (seq_lens.astype(np.int64) + p - 1) // p
    max_pages = int(n_pages_seq.max()) if S else 0
    width = max(max_pages, 1) if table_width is None else int(table_width)
    assert width >= max_pages

    if share_with is None:
        share_with = [-1] * S
    shared_arr = np.broadcast_to(np.asarray(shared_tokens, dtype=np.int64), (S,)) if S else np.zeros(0, np.int64)
    assert np.all(shared_arr % p == 0)

    perm = rng.permutation(num_pages).astype(np.int64)
    block_table = np.full((S, width), -1, dtype=np.int32)
    used_list = []
    cursor = 0
    for s in range(S):
        n = int(n_pages_seq[s])
        r = share_with[s]
        first_private = 0
        if r is not None and r >= 0:
            sh = int(shared_arr[s])
            assert r < s and sh <= int(seq_lens[s]) - int(q_lens[s])
            assert sh <= int(seq_lens[r]) - int(q_lens[r])
            block_table[s, :sh // p] = block_table[r, :sh // p]
            first_private = sh // p
        m = n - first_private
        assert cursor + m <= num_pages, "pool too small"
        ids = perm[cursor:cursor + m]
        cursor += m
        block_table[s, first_private:n] = ids
        used_list.append(ids)
    used_pages = np.concatenate(used_list) if used_list else np.zeros(0, np.int64)
    U = used_pages.shape[0]
    store_row = {int(pg): u for u, pg in enumerate(used_pages)}
    compact_bt = np.full_like(block_table, -1)
    for s in range(S):
        n = int(n_pages_seq[s])
        compact_bt[s, :n] = [store_row[int(pg)] for pg in block_table[s, :n]]

    cu = np.zeros(S + 1, dtype=np.int32)
    cu[1:] = np.cumsum(q_lens)
    T = int(cu[-1])

    q = _normal_bf16(rng, (T, Hq, D))
    k_store = _normal_bf16(rng, (U, Hkv, p, D))
    v_store = _normal_bf16(rng, (U, Hkv, p, D))

    # poison the slots past the end of each sequence's last page
    for s in range(S):
        L = int(seq_lens[s])
        if L % p:
            u = int(compact_bt[s, L // p])
            k_store[u, :, L % p:, :] = BF16_NAN
            v_store[u, :, L % p:, :] = BF16_NAN

    # lift the step's new rows out of the store (state before the append) and poison their slots
    k_new = np.empty((T, Hkv, D), dtype=np.uint16)
    v_new = np.empty((T, Hkv, D), dtype=np.uint16)
    slot = np.empty(T, dtype=np.int64)
    cslot = np.empty(T, dtype=np.int64)
    for s in range(S):
        L, n = int(seq_lens[s]), int(q_lens[s])
        if n == 0:
            continue
        j = np.arange(L - n, L, dtype=np.int64)
        u = compact_bt[s, j // p].astype(np.int64)
        off = j % p
        t0 = int(cu[s])
        k_new[t0:t0 + n] = k_store[u, :, off, :]
        v_new[t0:t0 + n] = v_store[u, :, off, :]
        k_store[u, :, off, :] = BF16_NAN
        v_store[u, :, off, :] = BF16_NAN
        slot[t0:t0 + n] = block_table[s, j // p].astype(np.int64) * p + off
        cslot[t0:t0 + n] = u * p + off

    return PagedBatch(
        name=name, num_seqs=S, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=p,
        num_pages=int(num_pages), scale=np.float32(1.0 / math.sqrt(D)),
        seq_lens=seq_lens, q_lens=q_lens, cu_seqlens_q=cu, block_table=block_table,
        q=q, k_new=k_new, v_new=v_new, slot_mapping=slot,
        used_pages=used_pages, k_store=k_store, v_store=v_store,
        compact_block_table=compact_bt, compact_slot_mapping=cslot,
    )


def _rng(c: int) -> np.random.Generator:
    return np.random.default_rng(CONFIG_SEED_BASE + c)


def _pages(lens, p):
    return int(((np.asarray(lens, dtype=np.int64) + p - 1) // p).sum())


def config1_tiny_decode() -> PagedBatch:
    """BASELINE.json configs[0]: 4 seqs {1,17,33,100}, 8q/2kv, D 64, page 16, 64-page pool."""
    lens = [1, 17, 33, 100]
    return make_batch(_rng(1), "cfg1_tiny_decode", lens, [1] * 4, 8, 2, 64, 16, 64)


def config2_bagel_cfg_decode(num_requests: int = 32, n_branches: int = 2) -> PagedBatch:
    """configs[1]: BAGEL-like T2I decode, 32 requests x CFG pair sharing the first 256 tokens' pages."""
    rng = _rng(2)
    L = rng.integers(512, 4097, num_requests)
    lens, share = [], []
    for r in range(num_requests):
        for b in range(n_branches):
            lens.append(int(L[r]))
            share.append(-1 if b == 0 else r * n_branches)
    return make_batch(rng, "cfg2_bagel_cfg_decode", lens, [1] * len(lens), 28, 4, 128, 16,
                      2 * _pages(lens, 16), share_with=share, shared_tokens=256)


def config3_prefill(num_seqs: int = 8, n_new: int = 1024, max_prefix: int = 2048) -> PagedBatch:
    """configs[2]: causal prefill over cached prefix U[0,2048] + 1024 new tokens, 28q/4kv, D 128, page 16."""
    rng = _rng(3)
    P = rng.integers(0, max_prefix + 1, num_seqs)
    lens = [int(x) + n_new for x in P]
    return make_batch(rng, "cfg3_prefill", lens, [n_new] * num_seqs, 28, 4, 128, 16, 2 * _pages(lens, 16))


def _config4_lengths():
    rng = _rng(4)
    thinker = np.floor(np.minimum(8192.0, np.exp(rng.normal(math.log(1500.0), 0.8, 64))))
    thinker = np.maximum(thinker, 1).astype(np.int64)
    talker = rng.integers(64, 1025, 128)
    return rng, thinker, talker


def config4_thinker() -> PagedBatch:
    """configs[3], Thinker stream: 64 seqs, 32q/4kv, D 128, lognormal(median 1500, sigma 0.8) cap 8192."""
    rng, thinker, _ = _config4_lengths()
    lens = [int(x) for x in thinker]
    return make_batch(rng, "cfg4_thinker", lens, [1] * 64, 32, 4, 128, 16, 2 * _pages(lens, 16))


def config4_talker() -> PagedBatch:
    """configs[3], Talker stream: 128 seqs, 16q/2kv, D 128, U[64,1024].  Own pool, own value stream."""
    _, _, talker = _config4_lengths()
    lens = [int(x) for x in talker]
    rng = np.random.default_rng(CONFIG_SEED_BASE + 40)
    return make_batch(rng, "cfg4_talker", lens, [1] * 128, 16, 2, 128, 16, 2 * _pages(lens, 16))


def config5_long_context(num_seqs: int = 16, seq_len: int = 32768, num_pages: int = 491520) -> PagedBatch:
    """configs[4]: 16 x 32768, 32q/8kv, D 128, page 32, pages scattered over a 60 GiB pool (491520 pages)."""
    return make_batch(_rng(5), "cfg5_long_context", [seq_len] * num_seqs, [1] * num_seqs,
                      32, 8, 128, 32, num_pages)


def flow_step_bagel(num_requests: int = 4, n_latent: int = 4096, n_labels: int = 3) -> PagedBatch:
    """SURVEY 8(f) rank 1, the denoise ("flow") step of BAGEL-like text-to-image: every
    request has ``n_labels`` CFG labels (cond, cfg_text, cfg_img); each label is one sequence whose ``n_latent``
    new latent-image tokens attend bidirectionally among themselves and to the label's cached context
    (``causal = 0`` over seq_len = context + n_latent).  The paper gives no lengths: context of the cond label
    U{64..512} prompt tokens, cfg_text label 1 token (no text), cfg_img label = the cond context, by reference
    (same physical pages for its first 64 tokens).  n_latent = 4096 is a 1024 x 1024 image at 16 x 16 pixels per
    latent token.  28 q / 4 kv heads, head_dim 128, page 16 (the BAGEL-like geometry of configs[1])."""
    rng = np.random.default_rng(CONFIG_SEED_BASE + 61)
    ctx = rng.integers(64, 513, num_requests)
    lens, share = [], []
    for r in range(num_requests):
        for lab in range(n_labels):
            c = 1 if lab == 1 else int(ctx[r])
            lens.append(c + n_latent)
            share.append(r * n_labels if lab == 2 else -1)
    if n_labels < 3:
        share = [-1] * len(lens)
    return make_batch(rng, "flow_step_bagel", lens, [n_latent] * len(lens), 28, 4, 128, 16,
                      2 * _pages(lens, 16), share_with=share, shared_tokens=64 if n_labels >= 3 else 0)


def cfg_cascade_decode(num_requests: int = 16, n_branches: int = 3, num_q_heads: int = 28, num_kv_heads: int = 4,
                       page_size: int = 16, ctx_lo: int = 2048, ctx_hi: int = 6144, sfx_lo: int = 16,
                       sfx_hi: int = 512, seed: int = 71):
    """SURVEY 8(f) rank 3, a decode step in which sharing dominates ("three labels over a single paged
    KV pool ... reading page tables in place"; :104-106, the three CFG contexts): ``num_requests`` requests x
    ``n_branches`` CFG labels, request-major; the labels of a request reference the same physical pages for a
    context of U{ctx_lo..ctx_hi} tokens rounded down to whole pages (ragged across requests) and each label adds a
    private suffix of U{sfx_lo..sfx_hi} tokens (the part of the context the label keeps to itself plus what it has
    generated).  The paper gives no lengths; with the defaults about 90 % of the logical K/V bytes are shared.
    BAGEL-like geometry of configs[1] (28 q / 4 kv heads, head_dim 128, page 16).  Returns (batch, shared_lens[R])."""
    rng = np.random.default_rng(CONFIG_SEED_BASE + seed)
    p = page_size
    ctx = (rng.integers(ctx_lo, ctx_hi + 1, num_requests) // p) * p
    lens, share, shared = [], [], []
    for r in range(num_requests):
        for b in range(n_branches):
            lens.append(int(ctx[r]) + int(rng.integers(sfx_lo, sfx_hi + 1)))
            share.append(-1 if b == 0 else r * n_branches)
            shared.append(int(ctx[r]))
    b = make_batch(rng, "cfg_cascade_decode", lens, [1] * len(lens), num_q_heads, num_kv_heads, 128, p,
                   2 * _pages(lens, p), share_with=share, shared_tokens=shared)
    return b, ctx.astype(np.int32)


def fp8_page_scales(seed: int, num_pages: int, num_kv_heads: int, lo: float = 0.006, hi: float = 0.02):
    """Caller-owned scales of a quantised pool: fp32 [num_pages, Hkv] for K and for V, uniform
    in [lo, hi).  With N(0,1) rows the quotient x / scale spans subnormal codes, the normal range and, at the low
    end of the interval (448 * 0.006 = 2.7 sigma), saturation.  Inputs only: no arithmetic of the method."""
    rng = np.random.default_rng(seed)
    k = rng.uniform(lo, hi, (num_pages, num_kv_heads)).astype(np.float32)
    v = rng.uniform(lo, hi, (num_pages, num_kv_heads)).astype(np.float32)
    return k, v
