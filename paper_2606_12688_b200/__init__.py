"""B200 (sm_100a) paged-KV attention: the hot path of the M* serving runtime (arxiv/paper_2606_12688).

The product is the C-ABI library ``libmstar_attn.so`` (``include/mstar_attn.h``); this package is its thin
Python binding.  Names mirror the C entry points:

    kv_append            <- mstar_kv_append
    kv_append_fp8        <- mstar_kv_append_fp8        (quantising append into an E4M3 pool)
    paged_attn_decode_fp8 <- mstar_paged_attn_decode_fp8 (decode over the E4M3 pool)
    paged_attn_prefill_fp8 <- mstar_paged_attn_prefill_fp8 (prefill / flow step over the E4M3 pool)
    paged_attn_decode    <- mstar_paged_attn_decode   (split-K + LSE combine)
    paged_attn_prefill   <- mstar_paged_attn_prefill  (causal over a cached prefix)
    build_slot_mapping   <- mstar_build_slot_mapping
    kv_copy_pages        <- mstar_kv_copy_pages       (page moves pool -> pool)
    kv_gather            <- mstar_kv_gather           (pool -> contiguous rows)
    merge_attn_states    <- mstar_merge_attn_states   (LSE merge of two attention states)
    sample_tokens        <- mstar_sample_tokens       (CUDA-graph-compatible temperature / top-k / top-p sampling)
    paged_attn_decode_cascade <- mstar_paged_attn_decode_cascade (CFG branches sharing prefix pages, one call)
    paged_attn_decode_static <- mstar_paged_attn_decode_static (decode with its scratch in the library's static device array)

There is no CPU fallback: without the built library every call raises ``MstarError``.
"""
from .binding import (  # noqa: F401
    EXPORTS,
    KVPool,
    KVPoolFp8,
    LIB_PATH,
    MSTAR_DECODE_STATIC_WORKSPACE_BYTES,
    MSTAR_FLAG_LOGITS_BF16,
    MSTAR_FLAG_OUT_F32,
    MSTAR_FLAG_PREFILL_MMA_SYNC,
    MSTAR_FLAG_PREFILL_REUSE_PLAN,
    MstarError,
    build_slot_mapping,
    decode_auto_partitions,
    decode_cascade_workspace_bytes,
    decode_workspace_bytes,
    kv_append,
    kv_append_fp8,
    kv_copy_pages,
    kv_gather,
    last_launch_count,
    load_library,
    merge_attn_states,
    paged_attn_decode,
    paged_attn_decode_cascade,
    paged_attn_decode_fp8,
    paged_attn_decode_static,
    paged_attn_prefill,
    paged_attn_prefill_fp8,
    prefill_fp8_workspace_bytes,
    prefill_workspace_bytes,
    sample_tokens,
    status_string,
    version,
)
