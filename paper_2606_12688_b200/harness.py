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
