"""Thin ctypes binding of ``include/mstar_attn.h``: argument marshalling only.

Every step of the path runs in the CUDA kernels of ``libmstar_attn.so``; there is no CPU or PyTorch
fallback -- if the library is missing or a call fails this module raises.  PyTorch provides device
memory and streams only: tensors cross the boundary as raw device pointers, the stream as
``torch.cuda.current_stream().cuda_stream``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

_PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG_DIR, "libmstar_attn.so")

MSTAR_OK = 0
MSTAR_ERR_WORKSPACE_TOO_SMALL = -3
MSTAR_FLAG_OUT_F32 = 1
MSTAR_FLAG_PREFILL_MMA_SYNC = 2
MSTAR_FLAG_PREFILL_REUSE_PLAN = 4
MSTAR_FLAG_LOGITS_BF16 = 8
MSTAR_FLAG_SAMPLE_ADVANCE_STEP = 16
MSTAR_FLAG_SAMPLE_ONE_CTA = 32

EXPORTS = (
    "mstar_kv_append",
    "mstar_kv_append_fp8",
    "mstar_paged_attn_decode_fp8",
    "mstar_paged_attn_prefill_fp8_workspace_bytes",
    "mstar_paged_attn_prefill_fp8",
    "mstar_kv_copy_pages",
    "mstar_kv_gather",
    "mstar_merge_attn_states",
    "mstar_paged_attn_decode_workspace_bytes",
    "mstar_paged_attn_decode",
    "mstar_paged_attn_decode_auto_partitions",
    "mstar_paged_attn_decode_static",
    "mstar_paged_attn_decode_cascade_workspace_bytes",
    "mstar_paged_attn_decode_cascade",
    "mstar_paged_attn_prefill_workspace_bytes",
    "mstar_paged_attn_prefill",
    "mstar_build_slot_mapping",
    "mstar_sample_tokens",
    "mstar_last_launch_count",
    "mstar_status_string",
    "mstar_version",
)


class MstarError(RuntimeError):
    pass


class _KvPoolStruct(ctypes.Structure):
    _fields_ = [
        ("k_pool", ctypes.c_void_p),
        ("v_pool", ctypes.c_void_p),
        ("num_pages", ctypes.c_int64),
        ("page_size", ctypes.c_int32),
        ("num_kv_heads", ctypes.c_int32),
        ("head_dim", ctypes.c_int32),
        ("stride_page", ctypes.c_int64),
        ("stride_head", ctypes.c_int64),
        ("stride_token", ctypes.c_int64),
    ]


_lib = None


def load_library() -> ctypes.CDLL:
    """Load the C-ABI library (built in-tree by ``paper_2606_12688_b200.build``).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MstarError(
            "%s not found: build it with `python -m paper_2606_12688_b200.build` "
            "(there is no CPU fallback)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    c = ctypes
    lib.mstar_kv_append.restype = c.c_int
    lib.mstar_kv_append.argtypes = [c.POINTER(_KvPoolStruct), c.c_void_p, c.c_void_p, c.c_void_p, c.c_int64,
                                    c.c_void_p]
    lib.mstar_kv_append_fp8.restype = c.c_int
    lib.mstar_kv_append_fp8.argtypes = [c.POINTER(_KvPoolStruct), c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                                        c.c_void_p, c.c_int64, c.c_void_p]
    lib.mstar_paged_attn_decode_fp8.restype = c.c_int
    lib.mstar_paged_attn_decode_fp8.argtypes = [
        c.c_void_p, c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_void_p, c.c_void_p, c.c_int64,
        c.c_void_p, c.c_int32, c.c_int32, c.c_int32, c.c_float, c.c_int32, c.c_uint32, c.c_void_p, c.c_size_t,
        c.c_void_p]
    lib.mstar_paged_attn_prefill_fp8_workspace_bytes.restype = c.c_size_t
    lib.mstar_paged_attn_prefill_fp8_workspace_bytes.argtypes = [c.c_int32] * 6
    lib.mstar_paged_attn_prefill_fp8.restype = c.c_int
    lib.mstar_paged_attn_prefill_fp8.argtypes = [
        c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_void_p, c.c_void_p,
        c.c_int64, c.c_void_p, c.c_int32, c.c_int32, c.c_int32, c.c_int32, c.c_int32, c.c_float, c.c_int32,
        c.c_uint32, c.c_void_p, c.c_size_t, c.c_void_p]
    lib.mstar_sample_tokens.restype = c.c_int
    lib.mstar_sample_tokens.argtypes = [c.c_void_p, c.c_void_p, c.c_int64, c.c_int32, c.c_int32, c.c_void_p,
                                        c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_uint32, c.c_void_p]
    lib.mstar_kv_copy_pages.restype = c.c_int
    lib.mstar_kv_copy_pages.argtypes = [c.POINTER(_KvPoolStruct), c.POINTER(_KvPoolStruct), c.c_void_p, c.c_void_p,
                                        c.c_int64, c.c_void_p]
    lib.mstar_kv_gather.restype = c.c_int
    lib.mstar_kv_gather.argtypes = [c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_int64,
                                    c.c_void_p, c.c_void_p, c.c_int32, c.c_int64, c.c_void_p]
    lib.mstar_merge_attn_states.restype = c.c_int
    lib.mstar_merge_attn_states.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                                            c.c_void_p, c.c_int64, c.c_int32, c.c_uint32, c.c_void_p]
    lib.mstar_paged_attn_decode_workspace_bytes.restype = c.c_size_t
    lib.mstar_paged_attn_decode_workspace_bytes.argtypes = [c.c_int32] * 4
    lib.mstar_paged_attn_decode_auto_partitions.restype = c.c_int32
    lib.mstar_paged_attn_decode_auto_partitions.argtypes = [c.c_int32] * 3
    lib.mstar_paged_attn_decode.restype = c.c_int
    lib.mstar_paged_attn_decode.argtypes = [
        c.c_void_p, c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_int64, c.c_void_p,
        c.c_int32, c.c_int32, c.c_int32, c.c_float, c.c_int32, c.c_uint32, c.c_void_p, c.c_size_t, c.c_void_p]
    lib.mstar_paged_attn_decode_static.restype = c.c_int
    lib.mstar_paged_attn_decode_static.argtypes = [
        c.c_void_p, c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_int64, c.c_void_p,
        c.c_int32, c.c_int32, c.c_int32, c.c_float, c.c_int32, c.c_uint32, c.c_void_p]
    lib.mstar_paged_attn_decode_cascade_workspace_bytes.restype = c.c_size_t
    lib.mstar_paged_attn_decode_cascade_workspace_bytes.argtypes = [c.c_int32] * 5
    lib.mstar_paged_attn_decode_cascade.restype = c.c_int
    lib.mstar_paged_attn_decode_cascade.argtypes = [
        c.c_void_p, c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_int64, c.c_void_p, c.c_void_p,
        c.c_int32, c.c_int32, c.c_int32, c.c_int32, c.c_float, c.c_uint32, c.c_void_p, c.c_size_t, c.c_void_p]
    lib.mstar_paged_attn_prefill_workspace_bytes.restype = c.c_size_t
    lib.mstar_paged_attn_prefill_workspace_bytes.argtypes = [c.c_int32] * 4
    lib.mstar_paged_attn_prefill.restype = c.c_int
    lib.mstar_paged_attn_prefill.argtypes = [
        c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.POINTER(_KvPoolStruct), c.c_void_p, c.c_int64,
        c.c_void_p, c.c_int32, c.c_int32, c.c_int32, c.c_int32, c.c_int32, c.c_float, c.c_int32, c.c_uint32,
        c.c_void_p, c.c_size_t, c.c_void_p]
    lib.mstar_build_slot_mapping.restype = c.c_int
    lib.mstar_build_slot_mapping.argtypes = [c.c_void_p, c.c_int64, c.c_void_p, c.c_void_p, c.c_int32, c.c_int32,
                                             c.c_int32, c.c_void_p, c.c_void_p]
    lib.mstar_last_launch_count.restype = c.c_int32
    lib.mstar_last_launch_count.argtypes = []
    lib.mstar_status_string.restype = c.c_char_p
    lib.mstar_status_string.argtypes = [c.c_int]
    lib.mstar_version.restype = c.c_char_p
    lib.mstar_version.argtypes = []
    _lib = lib
    return lib


def status_string(status: int) -> str:
    return load_library().mstar_status_string(int(status)).decode()


def version() -> str:
    return load_library().mstar_version().decode()


def last_launch_count() -> int:
    return int(load_library().mstar_last_launch_count())


def _check(status: int, what: str) -> None:
    if status != MSTAR_OK:
        raise MstarError("%s failed: %s (%d)" % (what, status_string(status), status))


def _stream() -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t: Optional[torch.Tensor]) -> ctypes.c_void_p:
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _want(t: torch.Tensor, dtype, name: str) -> None:
    if not t.is_cuda:
        raise MstarError("%s must be a CUDA tensor (the C ABI takes device pointers)" % name)
    if t.dtype != dtype:
        raise MstarError("%s must be %s, got %s" % (name, dtype, t.dtype))
    if not t.is_contiguous():
        raise MstarError("%s must be contiguous" % name)


class KVPool:
    """The paged K/V pool: two bf16 tensors viewed as [num_pages, Hkv, page_size, D] (any strides whose
    innermost is 1).  Holds references to the tensors; owns nothing else."""

    def __init__(self, k_pool: torch.Tensor, v_pool: torch.Tensor):
        for t, nm in ((k_pool, "k_pool"), (v_pool, "v_pool")):
            if not t.is_cuda or t.dtype != torch.bfloat16 or t.dim() != 4 or t.stride(3) != 1:
                raise MstarError("%s must be a CUDA bf16 tensor [num_pages, Hkv, page_size, D] with unit inner stride" % nm)
        if k_pool.shape != v_pool.shape or k_pool.stride() != v_pool.stride():
            raise MstarError("k_pool and v_pool must share shape and strides")
        self.k_pool, self.v_pool = k_pool, v_pool
        self.num_pages, self.num_kv_heads, self.page_size, self.head_dim = (int(x) for x in k_pool.shape)
        self.c = _KvPoolStruct(
            k_pool.data_ptr(), v_pool.data_ptr(), self.num_pages, self.page_size, self.num_kv_heads,
            self.head_dim, int(k_pool.stride(0)), int(k_pool.stride(1)), int(k_pool.stride(2)))


class KVPoolFp8:
    """The quantised pool: two uint8 tensors of E4M3 codes viewed as [num_pages, Hkv, page_size, 128] plus fp32
    scales [num_pages, Hkv] (value = e4m3(code) * scale[page][head])."""

    def __init__(self, k_pool: torch.Tensor, v_pool: torch.Tensor, k_scale: torch.Tensor, v_scale: torch.Tensor):
        for t, nm in ((k_pool, "k_pool"), (v_pool, "v_pool")):
            if not t.is_cuda or t.dtype != torch.uint8 or t.dim() != 4 or t.stride(3) != 1:
                raise MstarError("%s must be a CUDA uint8 tensor [num_pages, Hkv, page_size, D] with unit inner stride" % nm)
        if k_pool.shape != v_pool.shape or k_pool.stride() != v_pool.stride():
            raise MstarError("k_pool and v_pool must share shape and strides")
        self.k_pool, self.v_pool = k_pool, v_pool
        self.num_pages, self.num_kv_heads, self.page_size, self.head_dim = (int(x) for x in k_pool.shape)
        for t, nm in ((k_scale, "k_scale"), (v_scale, "v_scale")):
            _want(t, torch.float32, nm)
            if tuple(t.shape) != (self.num_pages, self.num_kv_heads):
                raise MstarError("%s must be [num_pages, Hkv]" % nm)
        self.k_scale, self.v_scale = k_scale, v_scale
        self.c = _KvPoolStruct(
            k_pool.data_ptr(), v_pool.data_ptr(), self.num_pages, self.page_size, self.num_kv_heads,
            self.head_dim, int(k_pool.stride(0)), int(k_pool.stride(1)), int(k_pool.stride(2)))


    def as_bit_pool(self) -> "KVPool":
        """The same bytes described as a bf16 pool of head_dim 64 (two codes per 16-bit element): what the bit-copy
        entry points (mstar_kv_copy_pages, mstar_kv_gather) take to move pages of a quantised pool.  The scales
        [num_pages, Hkv] travel separately (they are the caller's)."""
        return KVPool(self.k_pool.view(torch.bfloat16), self.v_pool.view(torch.bfloat16))


def kv_append_fp8(pool: KVPoolFp8, k_new: torch.Tensor, v_new: torch.Tensor, slot_mapping: torch.Tensor) -> None:
    """mstar_kv_append_fp8: quantise k_new/v_new [T,Hkv,D] bf16 to E4M3 codes at slot_mapping [T] int64."""
    _want(k_new, torch.bfloat16, "k_new"); _want(v_new, torch.bfloat16, "v_new")
    _want(slot_mapping, torch.int64, "slot_mapping")
    T = int(slot_mapping.shape[0])
    if tuple(k_new.shape) != (T, pool.num_kv_heads, pool.head_dim) or k_new.shape != v_new.shape:
        raise MstarError("k_new/v_new must be [T, Hkv, D]")
    lib = load_library()
    _check(lib.mstar_kv_append_fp8(ctypes.byref(pool.c), _ptr(pool.k_scale), _ptr(pool.v_scale), _ptr(k_new),
                                   _ptr(v_new), _ptr(slot_mapping), T, _stream()), "mstar_kv_append_fp8")


def paged_attn_decode_fp8(out: torch.Tensor, q: torch.Tensor, pool: KVPoolFp8, block_table: torch.Tensor,
                          seq_lens: torch.Tensor, max_seq_len: int, scale: float, num_partitions: int = 0,
                          workspace: Optional[torch.Tensor] = None, lse_out: Optional[torch.Tensor] = None) -> None:
    """mstar_paged_attn_decode_fp8: decode over the quantised pool; arguments as paged_attn_decode."""
    _want(q, torch.bfloat16, "q"); _want(block_table, torch.int32, "block_table")
    _want(seq_lens, torch.int32, "seq_lens")
    S, Hq, D = (int(x) for x in q.shape)
    flags = 0
    if out.dtype == torch.float32:
        flags |= MSTAR_FLAG_OUT_F32
    elif out.dtype != torch.bfloat16:
        raise MstarError("out must be bf16 or fp32")
    if not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != (S, Hq, D):
        raise MstarError("out must be a contiguous CUDA tensor [S, Hq, D]")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    lib = load_library()
    _check(lib.mstar_paged_attn_decode_fp8(
        _ptr(out), _ptr(lse_out), _ptr(q), ctypes.byref(pool.c), _ptr(pool.k_scale), _ptr(pool.v_scale),
        _ptr(block_table), int(block_table.stride(0)) if block_table.dim() == 2 else 0, _ptr(seq_lens), S, Hq,
        int(max_seq_len), float(scale), int(num_partitions), flags, _ptr(workspace), ws_bytes, _stream()),
        "mstar_paged_attn_decode_fp8")


def kv_append(pool: KVPool, k_new: torch.Tensor, v_new: torch.Tensor, slot_mapping: torch.Tensor) -> None:
    """mstar_kv_append: scatter k_new/v_new [T,Hkv,D] bf16 into the pool at slot_mapping [T] int64."""
    _want(k_new, torch.bfloat16, "k_new"); _want(v_new, torch.bfloat16, "v_new")
    _want(slot_mapping, torch.int64, "slot_mapping")
    T = int(slot_mapping.shape[0])
    if tuple(k_new.shape) != (T, pool.num_kv_heads, pool.head_dim) or k_new.shape != v_new.shape:
        raise MstarError("k_new/v_new must be [T, Hkv, D]")
    lib = load_library()
    _check(lib.mstar_kv_append(ctypes.byref(pool.c), _ptr(k_new), _ptr(v_new), _ptr(slot_mapping), T, _stream()),
           "mstar_kv_append")


def kv_copy_pages(dst_pool: KVPool, src_pool: KVPool, dst_pages: torch.Tensor, src_pages: torch.Tensor) -> None:
    """mstar_kv_copy_pages: page src_pages[i] of src_pool -> page dst_pages[i] of dst_pool (int64, device)."""
    _want(dst_pages, torch.int64, "dst_pages"); _want(src_pages, torch.int64, "src_pages")
    if dst_pages.shape != src_pages.shape or dst_pages.dim() != 1:
        raise MstarError("dst_pages and src_pages must be 1-D and of equal length")
    lib = load_library()
    _check(lib.mstar_kv_copy_pages(ctypes.byref(dst_pool.c), ctypes.byref(src_pool.c), _ptr(dst_pages),
                                   _ptr(src_pages), int(dst_pages.shape[0]), _stream()), "mstar_kv_copy_pages")


def kv_gather(k_out: torch.Tensor, v_out: torch.Tensor, pool: KVPool, block_table: torch.Tensor,
              seq_lens: torch.Tensor, cu_seqlens_out: torch.Tensor) -> None:
    """mstar_kv_gather: pool -> contiguous k_out / v_out [total, Hkv, D] bf16 through the block table."""
    _want(k_out, torch.bfloat16, "k_out"); _want(v_out, torch.bfloat16, "v_out")
    _want(block_table, torch.int32, "block_table"); _want(seq_lens, torch.int32, "seq_lens")
    _want(cu_seqlens_out, torch.int32, "cu_seqlens_out")
    S = int(seq_lens.shape[0])
    if k_out.shape != v_out.shape or tuple(k_out.shape[1:]) != (pool.num_kv_heads, pool.head_dim):
        raise MstarError("k_out / v_out must be [total, Hkv, D]")
    lib = load_library()
    _check(lib.mstar_kv_gather(_ptr(k_out), _ptr(v_out), ctypes.byref(pool.c), _ptr(block_table),
                               int(block_table.stride(0)) if block_table.dim() == 2 else 0, _ptr(seq_lens),
                               _ptr(cu_seqlens_out), S, int(k_out.shape[0]), _stream()), "mstar_kv_gather")


def merge_attn_states(out: torch.Tensor, out_a: torch.Tensor, lse_a: torch.Tensor, out_b: torch.Tensor,
                      lse_b: torch.Tensor, row_map_a: Optional[torch.Tensor] = None,
                      lse_out: Optional[torch.Tensor] = None) -> None:
    """mstar_merge_attn_states: LSE merge of two fp32 attention states [.., D] into out [N, D] (bf16 or fp32)."""
    for t, nm in ((out_a, "out_a"), (lse_a, "lse_a"), (out_b, "out_b"), (lse_b, "lse_b")):
        _want(t, torch.float32, nm)
    if row_map_a is not None:
        _want(row_map_a, torch.int32, "row_map_a")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    D = int(out.shape[-1])
    N = out.numel() // D
    flags = MSTAR_FLAG_OUT_F32 if out.dtype == torch.float32 else 0
    if out.dtype not in (torch.float32, torch.bfloat16) or not out.is_contiguous():
        raise MstarError("out must be contiguous bf16 or fp32")
    if out_b.numel() != N * D or lse_b.numel() != N:
        raise MstarError("state B must have the rows of out")
    lib = load_library()
    _check(lib.mstar_merge_attn_states(_ptr(out), _ptr(lse_out), _ptr(out_a), _ptr(lse_a), _ptr(row_map_a),
                                       _ptr(out_b), _ptr(lse_b), N, D, flags, _stream()), "mstar_merge_attn_states")


def decode_auto_partitions(num_seqs: int, num_kv_heads: int, max_seq_len: int) -> int:
    return int(load_library().mstar_paged_attn_decode_auto_partitions(num_seqs, num_kv_heads, max_seq_len))


def decode_workspace_bytes(num_seqs: int, num_q_heads: int, head_dim: int, max_partitions: int) -> int:
    return int(load_library().mstar_paged_attn_decode_workspace_bytes(num_seqs, num_q_heads, head_dim,
                                                                       max_partitions))


def paged_attn_decode(out: torch.Tensor, q: torch.Tensor, pool: KVPool, block_table: torch.Tensor,
                      seq_lens: torch.Tensor, max_seq_len: int, scale: float, num_partitions: int = 0,
                      workspace: Optional[torch.Tensor] = None, lse_out: Optional[torch.Tensor] = None) -> None:
    """mstar_paged_attn_decode.  out [S,Hq,D] bf16 or fp32 (fp32 selects MSTAR_FLAG_OUT_F32)."""
    _want(q, torch.bfloat16, "q"); _want(block_table, torch.int32, "block_table")
    _want(seq_lens, torch.int32, "seq_lens")
    S, Hq, D = (int(x) for x in q.shape)
    flags = 0
    if out.dtype == torch.float32:
        flags |= MSTAR_FLAG_OUT_F32
    elif out.dtype != torch.bfloat16:
        raise MstarError("out must be bf16 or fp32")
    if not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != (S, Hq, D):
        raise MstarError("out must be a contiguous CUDA tensor [S, Hq, D]")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    lib = load_library()
    _check(lib.mstar_paged_attn_decode(
        _ptr(out), _ptr(lse_out), _ptr(q), ctypes.byref(pool.c), _ptr(block_table),
        int(block_table.stride(0)) if block_table.dim() == 2 else 0, _ptr(seq_lens), S, Hq, int(max_seq_len),
        float(scale), int(num_partitions), flags, _ptr(workspace), ws_bytes, _stream()), "mstar_paged_attn_decode")


MSTAR_DECODE_STATIC_WORKSPACE_BYTES = 48 << 20


def paged_attn_decode_static(out: torch.Tensor, q: torch.Tensor, pool: KVPool, block_table: torch.Tensor,
                             seq_lens: torch.Tensor, max_seq_len: int, scale: float, num_partitions: int = 0,
                             lse_out: Optional[torch.Tensor] = None) -> None:
    """mstar_paged_attn_decode_static: the decode call with its scratch in the library's static device array
    (MSTAR_DECODE_STATIC_WORKSPACE_BYTES; nothing is allocated).  Calls that overlap on the GPU race on that array."""
    _want(q, torch.bfloat16, "q"); _want(block_table, torch.int32, "block_table")
    _want(seq_lens, torch.int32, "seq_lens")
    S, Hq, D = (int(x) for x in q.shape)
    flags = 0
    if out.dtype == torch.float32:
        flags |= MSTAR_FLAG_OUT_F32
    elif out.dtype != torch.bfloat16:
        raise MstarError("out must be bf16 or fp32")
    if not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != (S, Hq, D):
        raise MstarError("out must be a contiguous CUDA tensor [S, Hq, D]")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    lib = load_library()
    status = lib.mstar_paged_attn_decode_static(
        _ptr(out), _ptr(lse_out), _ptr(q), ctypes.byref(pool.c), _ptr(block_table),
        int(block_table.stride(0)) if block_table.dim() == 2 else 0, _ptr(seq_lens), S, Hq, int(max_seq_len),
        float(scale), int(num_partitions), flags, _stream())
    if status == MSTAR_ERR_WORKSPACE_TOO_SMALL:
        raise MstarError("mstar_paged_attn_decode_static: this geometry needs more scratch than the static array "
                         "holds (%d bytes); use paged_attn_decode with a caller-owned workspace"
                         % MSTAR_DECODE_STATIC_WORKSPACE_BYTES)
    _check(status, "mstar_paged_attn_decode_static")


def decode_cascade_workspace_bytes(num_seqs: int, num_q_heads: int, num_kv_heads: int, head_dim: int,
                                   max_seq_len: int) -> int:
    return int(load_library().mstar_paged_attn_decode_cascade_workspace_bytes(num_seqs, num_q_heads, num_kv_heads,
                                                                               head_dim, max_seq_len))


def paged_attn_decode_cascade(out: torch.Tensor, q: torch.Tensor, pool: KVPool, block_table: torch.Tensor,
                              seq_lens: torch.Tensor, shared_lens: torch.Tensor, n_branches: int, max_seq_len: int,
                              scale: float, workspace: torch.Tensor, lse_out: Optional[torch.Tensor] = None) -> None:
    """mstar_paged_attn_decode_cascade: decode of request-major CFG branches that share prefix pages.
    shared_lens [S / n_branches] int32 on the device."""
    _want(q, torch.bfloat16, "q"); _want(block_table, torch.int32, "block_table")
    _want(seq_lens, torch.int32, "seq_lens"); _want(shared_lens, torch.int32, "shared_lens")
    S, Hq, D = (int(x) for x in q.shape)
    if n_branches < 1 or S % n_branches or int(shared_lens.shape[0]) != S // n_branches:
        raise MstarError("shared_lens must have one entry per request (num_seqs / n_branches)")
    flags = 0
    if out.dtype == torch.float32:
        flags |= MSTAR_FLAG_OUT_F32
    elif out.dtype != torch.bfloat16:
        raise MstarError("out must be bf16 or fp32")
    if not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != (S, Hq, D):
        raise MstarError("out must be a contiguous CUDA tensor [S, Hq, D]")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    lib = load_library()
    _check(lib.mstar_paged_attn_decode_cascade(
        _ptr(out), _ptr(lse_out), _ptr(q), ctypes.byref(pool.c), _ptr(block_table),
        int(block_table.stride(0)) if block_table.dim() == 2 else 0, _ptr(seq_lens), _ptr(shared_lens), S,
        int(n_branches), Hq, int(max_seq_len), float(scale), flags, _ptr(workspace), ws_bytes, _stream()),
        "mstar_paged_attn_decode_cascade")


def prefill_workspace_bytes(num_seqs: int, total_q: int, num_q_heads: int, head_dim: int) -> int:
    return int(load_library().mstar_paged_attn_prefill_workspace_bytes(num_seqs, total_q, num_q_heads, head_dim))


def paged_attn_prefill(out: torch.Tensor, q: torch.Tensor, cu_seqlens_q: torch.Tensor, pool: KVPool,
                       block_table: torch.Tensor, seq_lens: torch.Tensor, max_q_len: int, max_seq_len: int,
                       scale: float, causal: bool = True, workspace: Optional[torch.Tensor] = None,
                       lse_out: Optional[torch.Tensor] = None, mma_sync: bool = False,
                       reuse_plan: bool = False) -> None:
    """mstar_paged_attn_prefill.  q/out [T,Hq,D]; K/V of the new tokens must already be in the pool.
    ``mma_sync=True`` sets MSTAR_FLAG_PREFILL_MMA_SYNC (diagnostic: the warp-level MMA kernel);
    ``reuse_plan=True`` sets MSTAR_FLAG_PREFILL_REUSE_PLAN (``workspace`` holds the plan of a previous call on the
    same batch geometry, e.g. the previous layer)."""
    _want(q, torch.bfloat16, "q"); _want(cu_seqlens_q, torch.int32, "cu_seqlens_q")
    _want(block_table, torch.int32, "block_table"); _want(seq_lens, torch.int32, "seq_lens")
    T, Hq, D = (int(x) for x in q.shape)
    S = int(cu_seqlens_q.shape[0]) - 1
    flags = MSTAR_FLAG_PREFILL_MMA_SYNC if mma_sync else 0
    if reuse_plan:
        flags |= MSTAR_FLAG_PREFILL_REUSE_PLAN
    if out.dtype == torch.float32:
        flags |= MSTAR_FLAG_OUT_F32
    elif out.dtype != torch.bfloat16:
        raise MstarError("out must be bf16 or fp32")
    if not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != (T, Hq, D):
        raise MstarError("out must be a contiguous CUDA tensor [T, Hq, D]")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    lib = load_library()
    _check(lib.mstar_paged_attn_prefill(
        _ptr(out), _ptr(lse_out), _ptr(q), _ptr(cu_seqlens_q), ctypes.byref(pool.c), _ptr(block_table),
        int(block_table.stride(0)) if block_table.dim() == 2 else 0, _ptr(seq_lens), S, T, int(max_q_len),
        int(max_seq_len), Hq, float(scale), 1 if causal else 0, flags, _ptr(workspace), ws_bytes, _stream()),
        "mstar_paged_attn_prefill")


def prefill_fp8_workspace_bytes(num_seqs: int, total_q: int, num_q_heads: int, num_kv_heads: int, page_size: int,
                                max_seq_len: int) -> int:
    return int(load_library().mstar_paged_attn_prefill_fp8_workspace_bytes(num_seqs, total_q, num_q_heads,
                                                                            num_kv_heads, page_size, max_seq_len))


def paged_attn_prefill_fp8(out: torch.Tensor, q: torch.Tensor, cu_seqlens_q: torch.Tensor, pool: "KVPoolFp8",
                           block_table: torch.Tensor, seq_lens: torch.Tensor, max_q_len: int, max_seq_len: int,
                           scale: float, workspace: torch.Tensor, causal: bool = True,
                           lse_out: Optional[torch.Tensor] = None) -> None:
    """mstar_paged_attn_prefill_fp8.  q/out [T,Hq,D]; the new tokens' codes must already be in the pool."""
    _want(q, torch.bfloat16, "q"); _want(cu_seqlens_q, torch.int32, "cu_seqlens_q")
    _want(block_table, torch.int32, "block_table"); _want(seq_lens, torch.int32, "seq_lens")
    T, Hq, D = (int(x) for x in q.shape)
    S = int(cu_seqlens_q.shape[0]) - 1
    flags = 0
    if out.dtype == torch.float32:
        flags |= MSTAR_FLAG_OUT_F32
    elif out.dtype != torch.bfloat16:
        raise MstarError("out must be bf16 or fp32")
    if not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != (T, Hq, D):
        raise MstarError("out must be a contiguous CUDA tensor [T, Hq, D]")
    if lse_out is not None:
        _want(lse_out, torch.float32, "lse_out")
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    lib = load_library()
    _check(lib.mstar_paged_attn_prefill_fp8(
        _ptr(out), _ptr(lse_out), _ptr(q), _ptr(cu_seqlens_q), ctypes.byref(pool.c), _ptr(pool.k_scale),
        _ptr(pool.v_scale), _ptr(block_table), int(block_table.stride(0)) if block_table.dim() == 2 else 0,
        _ptr(seq_lens), S, T, int(max_q_len), int(max_seq_len), Hq, float(scale), 1 if causal else 0, flags,
        _ptr(workspace), ws_bytes, _stream()), "mstar_paged_attn_prefill_fp8")


def sample_tokens(tokens_out: torch.Tensor, logits: torch.Tensor, seeds: torch.Tensor, step: torch.Tensor,
                  temperature: Optional[torch.Tensor] = None, top_k: Optional[torch.Tensor] = None,
                  top_p: Optional[torch.Tensor] = None, advance_step: bool = False, one_cta: bool = False) -> None:
    """mstar_sample_tokens.  logits [B, V] fp32 or bf16 (unit inner stride); seeds [B] int64 bit patterns of the
    uint64 keys; step: one int64 on the device (the uint64 counter).  ``one_cta=True`` sets
    MSTAR_FLAG_SAMPLE_ONE_CTA (the single-CTA-per-row kernel; same tokens)."""
    if logits.dim() != 2 or logits.stride(1) != 1 or not logits.is_cuda:
        raise MstarError("logits must be a CUDA tensor [B, V] with unit inner stride")
    B, V = (int(x) for x in logits.shape)
    flags = 0
    if logits.dtype == torch.bfloat16:
        flags |= MSTAR_FLAG_LOGITS_BF16
    elif logits.dtype != torch.float32:
        raise MstarError("logits must be fp32 or bf16")
    _want(tokens_out, torch.int32, "tokens_out"); _want(seeds, torch.int64, "seeds"); _want(step, torch.int64, "step")
    if temperature is not None:
        _want(temperature, torch.float32, "temperature")
    if top_k is not None:
        _want(top_k, torch.int32, "top_k")
    if top_p is not None:
        _want(top_p, torch.float32, "top_p")
    if advance_step:
        flags |= MSTAR_FLAG_SAMPLE_ADVANCE_STEP
    if one_cta:
        flags |= MSTAR_FLAG_SAMPLE_ONE_CTA
    lib = load_library()
    _check(lib.mstar_sample_tokens(_ptr(tokens_out), _ptr(logits), int(logits.stride(0)), B, V, _ptr(temperature),
                                   _ptr(top_k), _ptr(top_p), _ptr(seeds), _ptr(step), flags, _stream()),
           "mstar_sample_tokens")


def build_slot_mapping(block_table: torch.Tensor, cu_seqlens_q: torch.Tensor, seq_lens: torch.Tensor,
                       total_q: int, page_size: int, slot_mapping_out: torch.Tensor) -> None:
    """mstar_build_slot_mapping: device-side slot mapping of the step's new tokens."""
    _want(block_table, torch.int32, "block_table"); _want(cu_seqlens_q, torch.int32, "cu_seqlens_q")
    _want(seq_lens, torch.int32, "seq_lens"); _want(slot_mapping_out, torch.int64, "slot_mapping_out")
    S = int(seq_lens.shape[0])
    lib = load_library()
    _check(lib.mstar_build_slot_mapping(_ptr(block_table), int(block_table.stride(0)), _ptr(cu_seqlens_q),
                                        _ptr(seq_lens), S, int(total_q), int(page_size), _ptr(slot_mapping_out),
                                        _stream()), "mstar_build_slot_mapping")
