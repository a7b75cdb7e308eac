"""Out-of-bounds WRITE check of every entry point without a sanitizer (compute-sanitizer is closed on this pool,
profiles/r2_sanitizer.md): every buffer a call may write -- outputs, LSE, workspaces, pools -- is carved out of a larger
allocation with 64 KiB guard bands of a known pattern on both sides; after the call (small ragged cases that span
several tiles, partial pages, empty sequences, split-K cuts) the bands must be untouched.  Values are checked by the
parity tests; this file only looks at the bands."""
import numpy as np
import pytest
import torch

import paper_2606_12688_b200 as mstar
import workloads as W
from tests.gpu_util import DeviceBatch, DeviceBatchFp8, bf16_tensor

pytestmark = pytest.mark.gpu
GUARD = 64 << 10
PATTERN = 0xA5


class Guarded:
    """A tensor of ``shape``/``dtype`` inside a byte buffer with GUARD bytes of PATTERN before and after it."""

    def __init__(self, shape, dtype, fill=None):
        n = int(np.prod(shape)) * torch.empty(0, dtype=dtype).element_size()
        self.pad = (-n) % 256
        self.raw = torch.full((GUARD + n + self.pad + GUARD,), PATTERN, dtype=torch.uint8, device="cuda")
        self.t = self.raw[GUARD:GUARD + n].view(dtype).view(*shape)
        if fill is not None:
            self.t.copy_(fill)

    def check(self, what):
        n = self.raw.numel()
        lo, hi = self.raw[:GUARD], self.raw[n - GUARD - self.pad:]
        assert bool((lo == PATTERN).all()), "%s: bytes BEFORE the buffer were written" % what
        assert bool((hi == PATTERN).all()), "%s: bytes AFTER the buffer were written" % what


def guarded_batch(b, cls=DeviceBatch, **kw):
    """Device batch whose K/V pools sit between guard bands."""
    d = cls(b, **kw)
    gk = Guarded(tuple(d.k_pool.shape), d.k_pool.dtype, fill=d.k_pool)
    gv = Guarded(tuple(d.v_pool.shape), d.v_pool.dtype, fill=d.v_pool)
    d.k_pool, d.v_pool = gk.t, gv.t
    d.pool = mstar.KVPool(gk.t, gv.t) if cls is DeviceBatch else mstar.KVPoolFp8(gk.t, gv.t, d.k_scale, d.v_scale)
    return d, gk, gv


def ragged_decode_batch(seed=1, D=128, p=16, Hq=14, Hkv=2):
    lens = [1, 0, 17, 63, 64, 65, 300, 1000, p - 1, p + 1]
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(np.random.default_rng(seed), "g", lens, [min(1, l) for l in lens], Hq, Hkv, D, p,
                        2 * pages + 3)


def ragged_prefill_batch(seed=2, p=16, Hq=14, Hkv=2):
    lens, q_lens = [200 + 40, 64, 33 + 300, 1, 0, 129 + 16], [200, 64, 33, 1, 0, 129]
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(np.random.default_rng(seed), "gp", lens, q_lens, Hq, Hkv, 128, p, 2 * pages + 3)


@pytest.mark.parametrize("D,p", [(128, 16), (64, 32)])
@pytest.mark.parametrize("parts", [0, 1, 3])
def test_append_and_decode_write_inside_their_buffers(D, p, parts):
    b = ragged_decode_batch(D=D, p=p)
    d, gk, gv = guarded_batch(b)
    d.append()
    S, Hq = b.num_seqs, b.num_q_heads
    out, lse = Guarded((S, Hq, D), torch.bfloat16), Guarded((S, Hq), torch.float32)
    np_ = parts if parts > 0 else mstar.decode_auto_partitions(S, b.num_kv_heads, b.max_seq_len)
    ws = Guarded((mstar.decode_workspace_bytes(S, Hq, D, np_),), torch.uint8)
    mstar.paged_attn_decode(out.t, d.q_decode, d.pool, d.block_table, d.seq_lens, b.max_seq_len, float(b.scale),
                            num_partitions=parts, workspace=ws.t, lse_out=lse.t)
    torch.cuda.synchronize()
    for g, n in ((gk, "k_pool"), (gv, "v_pool"), (out, "out"), (lse, "lse"), (ws, "workspace")):
        g.check("decode D=%d p=%d parts=%d %s" % (D, p, parts, n))


def test_cascade_decode_writes_inside_its_buffers():
    from tests.test_gpu_cascade import cfg_batch
    shared_r = [0, 16, 640, 64]
    b = cfg_batch(4, shared_r, [[1, 70, 200], [16, 17, 1], [5, 300, 64], [63, 65, 2]], 3, 14, 2, 128, 16)
    d, gk, gv = guarded_batch(b)
    d.append()
    S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
    out, lse = Guarded((S, Hq, D), torch.bfloat16), Guarded((S, Hq), torch.float32)
    ws = Guarded((mstar.decode_cascade_workspace_bytes(S, Hq, b.num_kv_heads, D, b.max_seq_len),), torch.uint8)
    sh = torch.tensor(shared_r, dtype=torch.int32, device="cuda")
    mstar.paged_attn_decode_cascade(out.t, d.q_decode, d.pool, d.block_table, d.seq_lens, sh, 3, b.max_seq_len,
                                    float(b.scale), workspace=ws.t, lse_out=lse.t)
    torch.cuda.synchronize()
    for g, n in ((gk, "k_pool"), (gv, "v_pool"), (out, "out"), (lse, "lse"), (ws, "workspace")):
        g.check("cascade " + n)


@pytest.mark.parametrize("mma_sync", [False, True])
@pytest.mark.parametrize("causal", [True, False])
def test_prefill_writes_inside_its_buffers(mma_sync, causal):
    b = ragged_prefill_batch()
    d, gk, gv = guarded_batch(b)
    d.append()
    T, Hq, D = b.total_q, b.num_q_heads, b.head_dim
    out, lse = Guarded((T, Hq, D), torch.bfloat16), Guarded((T, Hq), torch.float32)
    ws = Guarded((mstar.prefill_workspace_bytes(b.num_seqs, T, Hq, D),), torch.uint8)
    mstar.paged_attn_prefill(out.t, d.q, d.cu_seqlens_q, d.pool, d.block_table, d.seq_lens, b.max_q_len,
                             b.max_seq_len, float(b.scale), causal=causal, workspace=ws.t, lse_out=lse.t,
                             mma_sync=mma_sync)
    torch.cuda.synchronize()
    for g, n in ((gk, "k_pool"), (gv, "v_pool"), (out, "out"), (lse, "lse"), (ws, "workspace")):
        g.check("prefill mma_sync=%d causal=%d %s" % (mma_sync, causal, n))


def test_fp8_append_decode_prefill_write_inside_their_buffers():
    b = ragged_decode_batch(seed=5, Hq=14, Hkv=2)
    ks, vs = W.fp8_page_scales(1, b.num_pages, b.num_kv_heads)
    d, gk, gv = guarded_batch(b, cls=DeviceBatchFp8, k_scale=ks, v_scale=vs)
    d.quantise_store()
    d.append()
    S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
    out, lse = Guarded((S, Hq, D), torch.bfloat16), Guarded((S, Hq), torch.float32)
    ws = Guarded((mstar.decode_workspace_bytes(S, Hq, D, mstar.decode_auto_partitions(S, b.num_kv_heads,
                                                                                      b.max_seq_len)),), torch.uint8)
    mstar.paged_attn_decode_fp8(out.t, d.q_decode, d.pool, d.block_table, d.seq_lens, b.max_seq_len, float(b.scale),
                                num_partitions=0, workspace=ws.t, lse_out=lse.t)
    torch.cuda.synchronize()
    for g, n in ((gk, "k_pool8"), (gv, "v_pool8"), (out, "out"), (lse, "lse"), (ws, "workspace")):
        g.check("fp8 decode " + n)
    bp = ragged_prefill_batch(seed=6)
    ks, vs = W.fp8_page_scales(2, bp.num_pages, bp.num_kv_heads)
    dp, gk, gv = guarded_batch(bp, cls=DeviceBatchFp8, k_scale=ks, v_scale=vs)
    dp.quantise_store()
    dp.append()
    T, Hq = bp.total_q, bp.num_q_heads
    out, lse = Guarded((T, Hq, 128), torch.bfloat16), Guarded((T, Hq), torch.float32)
    ws = Guarded((mstar.prefill_fp8_workspace_bytes(bp.num_seqs, T, Hq, bp.num_kv_heads, bp.page_size,
                                                    bp.max_seq_len),), torch.uint8)
    mstar.paged_attn_prefill_fp8(out.t, bf16_tensor(bp.q), torch.from_numpy(bp.cu_seqlens_q).cuda(), dp.pool,
                                 dp.block_table, dp.seq_lens, bp.max_q_len, bp.max_seq_len, float(bp.scale),
                                 workspace=ws.t, lse_out=lse.t)
    torch.cuda.synchronize()
    for g, n in ((gk, "k_pool8"), (gv, "v_pool8"), (out, "out"), (lse, "lse"), (ws, "workspace")):
        g.check("fp8 prefill " + n)


def test_page_moves_slot_mapping_and_merge_write_inside_their_buffers():
    b = ragged_decode_batch(seed=9)
    d, gk, gv = guarded_batch(b)
    d.append()
    # gather to contiguous rows
    cu = np.zeros(b.num_seqs + 1, dtype=np.int32)
    cu[1:] = np.cumsum(b.seq_lens)
    kg = Guarded((int(cu[-1]), b.num_kv_heads, b.head_dim), torch.bfloat16)
    vg = Guarded((int(cu[-1]), b.num_kv_heads, b.head_dim), torch.bfloat16)
    mstar.kv_gather(kg.t, vg.t, d.pool, d.block_table, d.seq_lens, torch.from_numpy(cu).cuda())
    # copy the used pages onto free pages of the same pool (incl. a skipped pair)
    used = np.zeros(b.num_pages, dtype=bool)
    used[b.used_pages] = True
    free = np.flatnonzero(~used)
    n = min(len(free), len(b.used_pages))
    src = b.used_pages[:n].astype(np.int64).copy()
    dst = free[:n].astype(np.int64).copy()
    src[0] = -1
    mstar.kv_copy_pages(d.pool, d.pool, torch.from_numpy(dst).cuda(), torch.from_numpy(src).cuda())
    # slot mapping
    sm = Guarded((b.total_q,), torch.int64)
    mstar.build_slot_mapping(d.block_table, d.cu_seqlens_q, d.seq_lens, b.total_q, b.page_size, sm.t)
    # merge of two states
    N, D = 37, 128
    o, l = Guarded((N, D), torch.bfloat16), Guarded((N,), torch.float32)
    r = lambda *s: torch.randn(*s, device="cuda")
    mstar.merge_attn_states(o.t, r(N, D), r(N), r(N, D), r(N), lse_out=l.t)
    torch.cuda.synchronize()
    for g, nme in ((gk, "k_pool"), (gv, "v_pool"), (kg, "k_out"), (vg, "v_out"), (sm, "slot_mapping"), (o, "merge out"),
                   (l, "merge lse")):
        g.check("moves " + nme)
