"""Device plumbing shared by the GPU tests, ``bench.py`` and ``smoke()``: upload a seeded batch
(any object with the fields of ``workloads.PagedBatch``) and call the C-ABI binding on it.

PyTorch is used for device memory only; every step of the path runs in ``libmstar_attn.so``.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as mstar


def bf16_tensor(bits: np.ndarray, device="cuda") -> torch.Tensor:
    """uint16 bit patterns -> bf16 tensor on the device (no value conversion)."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16))
    return t.to(device).view(torch.bfloat16)


def bits_of(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 bit patterns on the host."""
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def f64_of(t: torch.Tensor) -> np.ndarray:
    return t.detach().to(torch.float64).cpu().numpy()


class DeviceBatch:
    """Device-resident copy of a PagedBatch: pool (NaN poison + store rows), tables, Q, new K/V rows."""

    def __init__(self, b, device="cuda", layout="HND"):
        self.b = b
        shape = (b.num_pages, b.num_kv_heads, b.page_size, b.head_dim)
        if layout == "HND":
            self.k_pool = torch.full(shape, float("nan"), dtype=torch.bfloat16, device=device)
            self.v_pool = torch.full(shape, float("nan"), dtype=torch.bfloat16, device=device)
        else:  # token-major storage viewed as [pages, Hkv, p, D]: exercises the stride arguments
            nhd = (b.num_pages, b.page_size, b.num_kv_heads, b.head_dim)
            self.k_pool = torch.full(nhd, float("nan"), dtype=torch.bfloat16, device=device).permute(0, 2, 1, 3)
            self.v_pool = torch.full(nhd, float("nan"), dtype=torch.bfloat16, device=device).permute(0, 2, 1, 3)
        idx = torch.from_numpy(b.used_pages).to(device)
        step = 2048
        for a in range(0, len(b.used_pages), step):
            self.k_pool[idx[a:a + step]] = bf16_tensor(b.k_store[a:a + step], device)
            self.v_pool[idx[a:a + step]] = bf16_tensor(b.v_store[a:a + step], device)
        self.pool = mstar.KVPool(self.k_pool, self.v_pool)
        self.block_table = torch.from_numpy(b.block_table).to(device)
        self.seq_lens = torch.from_numpy(b.seq_lens).to(device)
        self.cu_seqlens_q = torch.from_numpy(b.cu_seqlens_q).to(device)
        self.q = bf16_tensor(b.q, device)
        if int(b.q_lens.max(initial=0)) <= 1:   # decode: one query row per sequence (zeros where L = 0)
            qd = np.zeros((b.num_seqs, b.num_q_heads, b.head_dim), dtype=np.uint16)
            has = b.q_lens > 0
            qd[has] = b.q[b.cu_seqlens_q[:-1][has]]
            self.q_decode = bf16_tensor(qd, device)
        self.k_new = bf16_tensor(b.k_new, device)
        self.v_new = bf16_tensor(b.v_new, device)
        self.slot_mapping = torch.from_numpy(b.slot_mapping).to(device)

    def append(self):
        mstar.kv_append(self.pool, self.k_new, self.v_new, self.slot_mapping)

    def decode(self, num_partitions=0, out_dtype=torch.bfloat16, want_lse=True):
        b = self.b
        S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
        dev = self.q_decode.device
        out = torch.full((S, Hq, D), float("nan"), dtype=out_dtype, device=dev)
        lse = torch.full((S, Hq), float("nan"), dtype=torch.float32, device=dev) if want_lse else None
        msl = b.max_seq_len
        parts = num_partitions if num_partitions > 0 else mstar.decode_auto_partitions(S, b.num_kv_heads, msl)
        ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, D, parts), dtype=torch.uint8, device=dev)
        ws.fill_(0xFF)  # NaN-pattern garbage: the workspace needs no initialisation
        mstar.paged_attn_decode(out, self.q_decode, self.pool, self.block_table, self.seq_lens, msl, float(b.scale),
                                num_partitions=num_partitions, workspace=ws, lse_out=lse)
        return out, lse

    def decode_cascade(self, n_branches, shared_lens, out_dtype=torch.bfloat16, want_lse=True):
        """mstar_paged_attn_decode_cascade on the batch (request-major branches, shared_lens int32 per request)."""
        b = self.b
        S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
        dev = self.q_decode.device
        out = torch.full((S, Hq, D), float("nan"), dtype=out_dtype, device=dev)
        lse = torch.full((S, Hq), float("nan"), dtype=torch.float32, device=dev) if want_lse else None
        ws = torch.empty(mstar.decode_cascade_workspace_bytes(S, Hq, b.num_kv_heads, D, b.max_seq_len),
                         dtype=torch.uint8, device=dev)
        ws.fill_(0xFF)
        sh = torch.from_numpy(np.ascontiguousarray(shared_lens, dtype=np.int32)).to(dev)
        mstar.paged_attn_decode_cascade(out, self.q_decode, self.pool, self.block_table, self.seq_lens, sh,
                                        n_branches, b.max_seq_len, float(b.scale), workspace=ws, lse_out=lse)
        return out, lse

    def prefill(self, causal=True, out_dtype=torch.bfloat16, want_lse=True, mma_sync=False):
        b = self.b
        T, Hq, D = b.total_q, b.num_q_heads, b.head_dim
        out = torch.full((T, Hq, D), float("nan"), dtype=out_dtype, device=self.q.device)
        lse = torch.full((T, Hq), float("nan"), dtype=torch.float32, device=self.q.device) if want_lse else None
        ws = torch.empty(mstar.prefill_workspace_bytes(b.num_seqs, T, Hq, D), dtype=torch.uint8,
                         device=self.q.device)
        mstar.paged_attn_prefill(out, self.q, self.cu_seqlens_q, self.pool, self.block_table, self.seq_lens,
                                 b.max_q_len, b.max_seq_len, float(b.scale), causal=causal, workspace=ws,
                                 lse_out=lse, mma_sync=mma_sync)
        return out, lse

    def store_rows_bits(self):
        """Pool rows of the used pages as uint16 bits [U, Hkv, p, D] (for whole-store comparisons)."""
        idx = torch.from_numpy(self.b.used_pages).to(self.k_pool.device)
        return bits_of(self.k_pool[idx]), bits_of(self.v_pool[idx])


class DeviceBatchFp8:
    """Device-resident quantised copy of a PagedBatch (head_dim 128): uint8 pools of E4M3 codes (0x7F poison), fp32
    scales [num_pages, Hkv], and the batch's bf16 store rows kept as rows to quantise: ``quantise_store()`` writes
    them with ``mstar_kv_append_fp8`` (so the pool content is produced by the product's own kernel), ``append()``
    adds the step's new rows, ``decode()`` runs ``mstar_paged_attn_decode_fp8``."""

    def __init__(self, b, k_scale: np.ndarray, v_scale: np.ndarray, device="cuda", layout="HND"):
        self.b = b
        shape = (b.num_pages, b.num_kv_heads, b.page_size, b.head_dim)
        if layout == "HND":
            self.k_pool = torch.full(shape, 0x7F, dtype=torch.uint8, device=device)
            self.v_pool = torch.full(shape, 0x7F, dtype=torch.uint8, device=device)
        else:
            nhd = (b.num_pages, b.page_size, b.num_kv_heads, b.head_dim)
            self.k_pool = torch.full(nhd, 0x7F, dtype=torch.uint8, device=device).permute(0, 2, 1, 3)
            self.v_pool = torch.full(nhd, 0x7F, dtype=torch.uint8, device=device).permute(0, 2, 1, 3)
        self.k_scale = torch.from_numpy(np.ascontiguousarray(k_scale, dtype=np.float32)).to(device)
        self.v_scale = torch.from_numpy(np.ascontiguousarray(v_scale, dtype=np.float32)).to(device)
        self.pool = mstar.KVPoolFp8(self.k_pool, self.v_pool, self.k_scale, self.v_scale)
        self.block_table = torch.from_numpy(b.block_table).to(device)
        self.seq_lens = torch.from_numpy(b.seq_lens).to(device)
        qd = np.zeros((b.num_seqs, b.num_q_heads, b.head_dim), dtype=np.uint16)
        has = b.q_lens > 0
        qd[has] = b.q[b.cu_seqlens_q[:-1][has]]
        self.q_decode = bf16_tensor(qd, device)
        self.k_new = bf16_tensor(b.k_new, device)
        self.v_new = bf16_tensor(b.v_new, device)
        self.slot_mapping = torch.from_numpy(b.slot_mapping).to(device)
        self.device = device

    def quantise_store(self, chunk_pages: int = 4096):
        """The batch's store rows (state before the step) -> codes, through mstar_kv_append_fp8."""
        b = self.b
        p = b.page_size
        U = len(b.used_pages)
        for a in range(0, U, chunk_pages):
            e = min(U, a + chunk_pages)
            # [u, Hkv, p, D] -> token-major rows [u * p, Hkv, D]
            rows_k = np.ascontiguousarray(b.k_store[a:e].transpose(0, 2, 1, 3)).reshape(-1, b.num_kv_heads, b.head_dim)
            rows_v = np.ascontiguousarray(b.v_store[a:e].transpose(0, 2, 1, 3)).reshape(-1, b.num_kv_heads, b.head_dim)
            slots = (b.used_pages[a:e].astype(np.int64)[:, None] * p + np.arange(p, dtype=np.int64)[None, :]).reshape(-1)
            mstar.kv_append_fp8(self.pool, bf16_tensor(rows_k, self.device), bf16_tensor(rows_v, self.device),
                                torch.from_numpy(slots).to(self.device))

    def append(self):
        mstar.kv_append_fp8(self.pool, self.k_new, self.v_new, self.slot_mapping)

    def decode(self, num_partitions=0, out_dtype=torch.bfloat16, want_lse=True):
        b = self.b
        S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
        dev = self.q_decode.device
        out = torch.full((S, Hq, D), float("nan"), dtype=out_dtype, device=dev)
        lse = torch.full((S, Hq), float("nan"), dtype=torch.float32, device=dev) if want_lse else None
        msl = b.max_seq_len
        parts = num_partitions if num_partitions > 0 else mstar.decode_auto_partitions(S, b.num_kv_heads, msl)
        ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, D, parts), dtype=torch.uint8, device=dev)
        ws.fill_(0xFF)
        mstar.paged_attn_decode_fp8(out, self.q_decode, self.pool, self.block_table, self.seq_lens, msl,
                                    float(b.scale), num_partitions=num_partitions, workspace=ws, lse_out=lse)
        return out, lse

    def prefill(self, causal=True, out_dtype=torch.bfloat16, want_lse=True):
        b = self.b
        T, Hq, D = b.total_q, b.num_q_heads, b.head_dim
        q = bf16_tensor(b.q, self.device)
        cu = torch.from_numpy(b.cu_seqlens_q).to(self.device)
        out = torch.full((T, Hq, D), float("nan"), dtype=out_dtype, device=self.device)
        lse = torch.full((T, Hq), float("nan"), dtype=torch.float32, device=self.device) if want_lse else None
        ws = torch.empty(mstar.prefill_fp8_workspace_bytes(b.num_seqs, T, Hq, b.num_kv_heads, b.page_size,
                                                           b.max_seq_len), dtype=torch.uint8, device=self.device)
        ws.fill_(0xFF)
        mstar.paged_attn_prefill_fp8(out, q, cu, self.pool, self.block_table, self.seq_lens, b.max_q_len,
                                     b.max_seq_len, float(b.scale), workspace=ws, causal=causal, lse_out=lse)
        return out, lse

    def store_codes(self):
        """Pool codes of the used pages [U, Hkv, p, D] uint8 on the host."""
        idx = torch.from_numpy(self.b.used_pages).to(self.k_pool.device)
        return self.k_pool[idx].cpu().numpy(), self.v_pool[idx].cpu().numpy()
