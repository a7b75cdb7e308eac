/*
 * mstar_attn.h -- C ABI of the B200 (sm_100a) paged-KV attention library.
 *
 * The one data-parallel hot path of the M* serving runtime (arxiv/paper_2606_12688): attention over
 * a paged KV cache.  PAPER.md:134 (sec. 3.3) -- "KVCacheEngine, a modality-agnostic transformer
 * engine with FlashInfer-based paged-attention KV-cache state"; PAPER.md:198 -- "three labels over a
 * single paged KV pool ... each denoise step can then apply paged attention, reading page tables in
 * place"; PAPER.md:430 (App. I) -- "paged-attention prefill and decode".  The paper gives no formula;
 * the operations are the textbook ones restated in DESIGN.md section 1 and oracle/mstar_oracle.c.
 *
 * Conventions common to every entry point
 *   - Every pointer named "device" is a CUDA device pointer; plain scalars are host values.
 *     `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - OWNERSHIP: the library allocates and frees no device memory.  All buffers, including the
 *     workspace, are the caller's.  Workspace contents need no initialisation and are clobbered.
 *   - ASYNC: a call only enqueues work on `stream` and never synchronises, so a sequence of calls
 *     is CUDA-graph capturable (PAPER.md:134, :212 rely on CUDA-graph replay).  All per-sequence
 *     metadata (block_table, seq_lens, cu_seqlens_q, slot_mapping) is read on the DEVICE; the host
 *     passes only shape bounds.
 *   - ERRORS: the return value is an mstar_status.  0 = enqueued.  A negative value means nothing
 *     was enqueued: NULL/misaligned pointers, unsupported geometry, workspace too small, or a CUDA
 *     launch error (MSTAR_ERR_CUDA; cudaGetLastError is consumed).  Device-side CONTENT (page ids
 *     out of range, seq_len beyond the block-table row, duplicate slots) is not validated:
 *     undefined behaviour.
 *   - dtype: Q, K, V, out are bf16 (bit patterns; the header has no bf16 type on purpose).
 *     Accumulation is fp32.  `scale` multiplies q.k before the softmax (natural exponent).
 *   - GQA: query head h reads KV head h / (num_q_heads / num_kv_heads).
 *   - Slots of the pool that hold no token (tails of last pages, unreferenced pages) may contain
 *     anything, including NaN/Inf; results do not depend on them.
 *   - Results are run-to-run deterministic (no floating-point atomics).
 */
#ifndef MSTAR_ATTN_H_
#define MSTAR_ATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MSTAR_OK = 0,
    MSTAR_ERR_INVALID_ARG = -1,
    MSTAR_ERR_UNSUPPORTED = -2,
    MSTAR_ERR_WORKSPACE_TOO_SMALL = -3,
    MSTAR_ERR_CUDA = -4
} mstar_status;

/* flags */
#define MSTAR_FLAG_OUT_F32 1u /* `out` is fp32 instead of bf16 (diagnostic: separates kernel error from
                                 output rounding).  Unknown bits => MSTAR_ERR_INVALID_ARG. */
#define MSTAR_FLAG_PREFILL_MMA_SYNC 2u /* prefill only, diagnostic: use the warp-level mma.sync kernel instead
                                          of the tcgen05/TMEM kernel (about a fifth of its rate at head_dim 128,
                                          0.4 at head_dim 64).  Both head dims take the tcgen05 kernel otherwise. */

#define MSTAR_FLAG_PREFILL_REUSE_PLAN 4u /* prefill only: `workspace` still holds the plan a previous call built
                                          for the SAME cu_seqlens_q, seq_lens, head geometry and causal flag (the
                                          next layer of the same forward pass): skip the plan kernel. */

#define MSTAR_FLAG_LOGITS_BF16 8u          /* mstar_sample_tokens only: `logits` is bf16 instead of fp32 */
#define MSTAR_FLAG_SAMPLE_ADVANCE_STEP 16u /* mstar_sample_tokens only: add 1 to *step behind the sampling kernel, so
                                              that every replay of a captured graph draws fresh numbers */
#define MSTAR_FLAG_SAMPLE_ONE_CTA 32u      /* mstar_sample_tokens only: one CTA per row re-reading the row from L2 (the
                                              path of vocabularies beyond the cluster kernel's capacity of 8 x 49 152
                                              tokens) instead of a cluster per row that keeps the row in shared
                                              memory; same token either way */

/*
 * The paged K/V pool ("a single paged KV pool").  Caller-owned device memory, bf16.
 * Element (page, kv_head, token_in_page, d) of K lives at
 *     k_pool + page*stride_page + kv_head*stride_head + token_in_page*stride_token + d     (elements)
 * and likewise for V.  The default "HND" layout [num_pages][Hkv][page_size][D] has
 * stride_token = D, stride_head = page_size*D, stride_page = Hkv*page_size*D; a token-major "NHD"
 * pool (stride_head = D, stride_token = Hkv*D) is equally valid.  Strides must be multiples of 8
 * elements (16 B) and the base pointers 128-B aligned (TMA requirements).
 * Supported: page_size in {16, 32}; head_dim in {64, 128}; num_pages*Hkv*page_size < 2^31 rows.
 */
typedef struct {
    void* k_pool;
    void* v_pool;
    int64_t num_pages;
    int32_t page_size;
    int32_t num_kv_heads;
    int32_t head_dim;
    int64_t stride_page;
    int64_t stride_head;
    int64_t stride_token;
} mstar_kv_pool;

/*
 * mstar_kv_append ("reshape_and_cache"; step a1 of DESIGN.md).  Writes the step's new K/V rows into
 * their pages once, instead of concatenating K/V "at every layer and for every step".
 *   k_new, v_new   device, [num_tokens][Hkv][D] bf16, contiguous, 16-B aligned
 *   slot_mapping   device, [num_tokens] int64; slot = page*page_size + token_in_page; slot < 0 = skip
 * Bit copy; other slots keep their bits.  Two tokens naming the same slot in one call: undefined.
 */
int mstar_kv_append(const mstar_kv_pool* pool, const void* k_new, const void* v_new,
                    const int64_t* slot_mapping, int64_t num_tokens, void* stream);

/*
 * mstar_kv_copy_pages / mstar_kv_gather: the page moves behind "paging, offload,
 * by-reference transfer" and prefill/decode disaggregation.  Bit copies.
 *   copy_pages: for i in 0..num_pairs-1, all heads and slots of page src_pages[i] of src_pool (K and V) are
 *               written to page dst_pages[i] of dst_pool.  The pools must agree in page_size, num_kv_heads and
 *               head_dim (strides may differ; they may be the same pool; a pool may live in pinned host memory
 *               that is mapped into the device address space).  dst_pages, src_pages: device, int64; a negative
 *               id skips the pair.  A page that is written by one pair and read or written by another pair of the
 *               same call: undefined.
 *   gather:     k_out/v_out [total_tokens][Hkv][D] bf16 contiguous, 16-B aligned; row cu_seqlens_out[s] + j gets
 *               token j of sequence s, j < seq_lens[s], read through block_table (the inverse of append).
 *               cu_seqlens_out: device, [S+1] int32, non-decreasing, cu[s+1]-cu[s] >= seq_lens[s]; rows of a
 *               sequence's range past seq_lens[s] are not written.
 */
int mstar_kv_copy_pages(const mstar_kv_pool* dst_pool, const mstar_kv_pool* src_pool, const int64_t* dst_pages,
                        const int64_t* src_pages, int64_t num_pairs, void* stream);
int mstar_kv_gather(void* k_out, void* v_out, const mstar_kv_pool* pool, const int32_t* block_table,
                    int64_t block_table_stride, const int32_t* seq_lens, const int32_t* cu_seqlens_out,
                    int32_t num_seqs, int64_t total_tokens, void* stream);

/*
 * mstar_paged_attn_decode (steps a2 + a3): one query token per sequence over block-table K/V, as a
 * split-K ("flash-decoding") pass plus a log-sum-exp combine.
 *   out            device, [S][Hq][D] bf16 (fp32 with MSTAR_FLAG_OUT_F32)
 *   lse_out        device, [S][Hq] fp32 natural-log LSE = ln sum_j exp(scale*q.k_j), or NULL
 *   q              device, [S][Hq][D] bf16 contiguous, 16-B aligned
 *   block_table    device, [S][block_table_stride] int32; row s lists the physical page of logical
 *                  page 0,1,...; only the first ceil(seq_lens[s]/page_size) entries are read
 *   seq_lens       device, [S] int32, KV length of each sequence (0 => out = 0, lse = -inf)
 *   max_seq_len    host upper bound on seq_lens (sizes the partition grid; may over-estimate)
 *   num_partitions split-K partitions per sequence.  P >= 1: partition i of a sequence covers tokens
 *                  [i*c, (i+1)*c) with c = ceil(max_seq_len/P) rounded up to a multiple of 64; partitions
 *                  past a sequence's end are empty; 1 = no combine pass.  0 = balanced: the 64-token
 *                  tiles of all (sequence, kv head) streams are laid end to end and every CTA takes an
 *                  contiguous range of equal cost (tiles + 2 per stream), so ragged batches finish together; a stream that lies inside
 *                  one range is finished by its CTA, a stream cut by range boundaries (at most one per
 *                  CTA) is merged by the combine pass (the cut points depend on seq_lens and the SM
 *                  count only, never on page ids).
 *   workspace      device, >= mstar_paged_attn_decode_workspace_bytes(...) bytes, 16-B aligned
 *   scale          must be positive and finite (MSTAR_ERR_INVALID_ARG otherwise)
 * Requires Hq % Hkv == 0.  Hq/Hkv <= 16 heads share one pass over a kv head's K/V; a larger group is processed as d
 * sub-groups of Hq/Hkv/d <= 16 heads, d the smallest such divisor (32 = 2 x 16, 24 = 2 x 12, 17 = 17 x 1), each a
 * stream of its own over the same K/V, whose repeated reads are L2 hits (cascade calls: MSTAR_ERR_UNSUPPORTED above
 * 16).  num_seqs <= 16384
 * (MSTAR_ERR_UNSUPPORTED: the per-sequence work-list prefix sums live in shared memory).
 */
size_t mstar_paged_attn_decode_workspace_bytes(int32_t num_seqs, int32_t num_q_heads, int32_t head_dim,
                                               int32_t max_partitions);
int mstar_paged_attn_decode(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool,
                            const int32_t* block_table, int64_t block_table_stride,
                            const int32_t* seq_lens, int32_t num_seqs, int32_t num_q_heads,
                            int32_t max_seq_len, float scale, int32_t num_partitions, uint32_t flags,
                            void* workspace, size_t workspace_bytes, void* stream);
/* Partial slots per (sequence, head) the choice num_partitions = 0 needs; pass it as max_partitions when sizing
 * the workspace. */
int32_t mstar_paged_attn_decode_auto_partitions(int32_t num_seqs, int32_t num_kv_heads,
                                                int32_t max_seq_len);

/*
 * Quantised pool ("fp8 K/V pages with per-page scales"; the KV-cache state of
 * PAPER.md:134 at half the bytes per token).  The pool holds one byte per element: an OCP E4M3 ("fn") code
 * (sign, 4 exponent bits of bias 7, 3 mantissa bits; 0x7F / 0xFF = NaN, no infinities, largest magnitude 448).
 * An element's value is  e4m3(code) * scale[page][kv head]  with caller-owned fp32 scales
 *   k_scale, v_scale   device, [num_pages][Hkv] fp32, positive and finite (not validated).
 * The pool is described by an mstar_kv_pool whose k_pool / v_pool point at the bytes and whose strides count
 * elements (= bytes); head_dim 128 only (a token row is one 128-byte line), page_size 16 or 32, strides
 * multiples of 16.
 *
 * mstar_kv_append_fp8: quantise and scatter the step's new rows.  For every element x (bf16) of a row that goes to
 * (page, h):  y = fp32(x) / scale[page][h]  in IEEE fp32 (round to nearest even);  code = y rounded to nearest
 * E4M3 value, ties to the even code, magnitudes above 448 (and infinities) saturate to +-448, NaN -> 0x7F.
 * Arguments as mstar_kv_append; bit-exact by definition (R24-R25).
 *
 * mstar_paged_attn_decode_fp8: mstar_paged_attn_decode on the dequantised K and V; all other arguments, the
 * partition rules and the workspace size are those of mstar_paged_attn_decode, with partition lengths rounded up to
 * the kernel's stage size (128 tokens, or 192 when Hq/Hkv <= 8 and max_seq_len > 8192) instead of 64.  Codes are converted to bf16
 * exactly in the kernel; k_scale multiplies the logits of a page, v_scale its probabilities (fp32).  Slots at or
 * past seq_len may hold any byte.  NaN codes inside a sequence give undefined output.
 *
 * Page moves of a quantised pool are the bit copies above on the same bytes described as a bf16 pool of head_dim 64
 * (two codes per element, all strides halved): mstar_kv_copy_pages / mstar_kv_gather need no fp8 variant.  The scale
 * rows of the moved pages are the caller's to copy.
 */
int mstar_kv_append_fp8(const mstar_kv_pool* pool8, const float* k_scale, const float* v_scale, const void* k_new,
                        const void* v_new, const int64_t* slot_mapping, int64_t num_tokens, void* stream);
int mstar_paged_attn_decode_fp8(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool8,
                                const float* k_scale, const float* v_scale, const int32_t* block_table,
                                int64_t block_table_stride, const int32_t* seq_lens, int32_t num_seqs,
                                int32_t num_q_heads, int32_t max_seq_len, float scale, int32_t num_partitions,
                                uint32_t flags, void* workspace, size_t workspace_bytes, void* stream);

/*
 * mstar_paged_attn_prefill_fp8: mstar_paged_attn_prefill (incl. causal = 0, the flow step) on the dequantised K and V
 * of a quantised pool (same pool8 / k_scale / v_scale as above; the new tokens' codes must already be in the pool:
 * mstar_kv_append_fp8 first).  All other arguments as mstar_paged_attn_prefill; flags: MSTAR_FLAG_OUT_F32 only.
 * Prefill is bound by the tensor pipe, not by K/V bytes, and the 16-bit MMA takes no E4M3 operand, so the call first
 * writes the referenced pages DEQUANTISED to fp16 -- e4m3(code) * scale, the product exact in fp32, rounded once to
 * nearest even (11 significant bits; magnitudes above 65504 saturate, below 2^-14 round to multiples of 2^-24) -- to a
 * compact scratch pool in the workspace (num_seqs * ceil(max_seq_len / page_size) pages: size the workspace with the
 * function below; max_seq_len must be a true upper bound here) and then runs the tcgen05 kernel of
 * mstar_paged_attn_prefill on it with fp16 operands (Q converted from bf16 in shared memory, P rounded to fp16).
 * Tolerances as the bf16 path.
 *   workspace      device, >= mstar_paged_attn_prefill_fp8_workspace_bytes(...) bytes, 256-B aligned
 */
size_t mstar_paged_attn_prefill_fp8_workspace_bytes(int32_t num_seqs, int32_t total_q, int32_t num_q_heads,
                                                    int32_t num_kv_heads, int32_t page_size, int32_t max_seq_len);
int mstar_paged_attn_prefill_fp8(void* out, float* lse_out, const void* q, const int32_t* cu_seqlens_q,
                                 const mstar_kv_pool* pool8, const float* k_scale, const float* v_scale,
                                 const int32_t* block_table, int64_t block_table_stride, const int32_t* seq_lens,
                                 int32_t num_seqs, int32_t total_q, int32_t max_q_len, int32_t max_seq_len,
                                 int32_t num_q_heads, float scale, int32_t causal, uint32_t flags, void* workspace,
                                 size_t workspace_bytes, void* stream);

/*
 * mstar_merge_attn_states: log-sum-exp merge of two normalised attention states over
 * disjoint key sets, row by row -- the last step of a shared-prefix ("cascade") decode for CFG branches whose
 * labels reference the same prefix pages:
 *     M = max(lse_a, lse_b);  out = (e^{lse_a-M} out_a + e^{lse_b-M} out_b) / (e^{lse_a-M} + e^{lse_b-M});
 *     lse = M + ln(e^{lse_a-M} + e^{lse_b-M})           (natural log; a state with lse = -inf has weight 0)
 *   out        device, [num_rows][D] bf16 (fp32 with MSTAR_FLAG_OUT_F32); lse_out [num_rows] fp32 or NULL
 *   out_a      device, [*][D] fp32, lse_a [*] fp32; row r of the result reads row row_map_a[r] of state A
 *              (row_map_a: device int32 [num_rows], or NULL for the identity)
 *   out_b      device, [num_rows][D] fp32, lse_b [num_rows] fp32
 * The two states are the fp32 outputs (MSTAR_FLAG_OUT_F32) and LSEs of two attention calls over disjoint key sets
 * (a caller that splits a context by hand; mstar_paged_attn_decode_cascade needs no such step).
 */
int mstar_merge_attn_states(void* out, float* lse_out, const float* out_a, const float* lse_a,
                            const int32_t* row_map_a, const float* out_b, const float* lse_b, int64_t num_rows,
                            int32_t head_dim, uint32_t flags, void* stream);

/*
 * mstar_paged_attn_decode_static: mstar_paged_attn_decode (sec. 4.1; SURVEY.md sec. 8(a) a2 + a3) for
 * callers that cannot allocate device memory -- code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc.  It takes no workspace: the split-K partials and cut records live in a file-scope device array
 * of MSTAR_DECODE_STATIC_WORKSPACE_BYTES inside the library (every GPU that loads the library holds it until the
 * process exits), whose device address the library resolves once per device (cudaGetSymbolAddress with that device
 * current; make the first call on a device outside stream capture).  No cudaMalloc, cudaFree or allocating library
 * routine is called.  Same kernels, launches and results (bit for bit) as mstar_paged_attn_decode; all arguments,
 * flags and errors as there, except:
 *   - a geometry whose workspace (mstar_paged_attn_decode_workspace_bytes(num_seqs, num_q_heads, head_dim, P) with
 *     P = num_partitions, or mstar_paged_attn_decode_auto_partitions(...) when num_partitions = 0) exceeds
 *     MSTAR_DECODE_STATIC_WORKSPACE_BYTES is refused with MSTAR_ERR_WORKSPACE_TOO_SMALL and nothing is launched
 *     (48 MiB holds every BASELINE decode config in balanced mode: 4.3 MB config 5 with 16 partitions, 9.6 MB
 *     talker, 29.8 MB config 2, 35.1 MB thinker);
 *   - ALL calls on a device share the array, which keeps the last call's contents (nothing in it has to start at
 *     zero: every slot that is read is written by the same call).  Calls that overlap on the GPU -- two streams, or
 *     two host threads -- race on it: serialise them, or give each stream its own workspace through
 *     mstar_paged_attn_decode.
 */
#define MSTAR_DECODE_STATIC_WORKSPACE_BYTES (48u << 20)
int mstar_paged_attn_decode_static(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool,
                                   const int32_t* block_table, int64_t block_table_stride, const int32_t* seq_lens,
                                   int32_t num_seqs, int32_t num_q_heads, int32_t max_seq_len, float scale,
                                   int32_t num_partitions, uint32_t flags, void* stream);

/*
 * mstar_paged_attn_decode_cascade: mstar_paged_attn_decode for CFG branches whose labels
 * reference the same prefix pages -- "three labels over a single paged KV pool ... reading page tables in place"
 * (the Parallel region LLM / LLM_cfg_text / LLM_cfg_img of PAPER.md:104-106).  The result is that of
 * mstar_paged_attn_decode on the same arguments (same definition, same tolerances); the shared pages of a request
 * pass through shared memory once for up to three of its branches (G = Hq / Hkv <= 8: one consumer warp group per
 * branch works on the same tile; four or more branches go in groups of three; G > 8: every branch reads the prefix
 * itself).
 *   Sequences are request-major: sequence r * n_branches + b is branch b of request r (num_seqs % n_branches == 0).
 *   shared_lens    device, [num_seqs / n_branches] int32: the first shared_lens[r] tokens of every branch of request
 *                  r are the same tokens -- the block-table rows of the branches hold the same page ids for them.
 *                  Multiples of page_size, <= the seq_len of every branch (values past a branch's seq_len:
 *                  undefined).  0 = nothing shared.
 * One call = one split-K launch over prefix streams (the kernel's Q load fetches the rows of every branch, q stays
 * in its natural [S][Hq][D] layout) and suffix streams, laid end to end in 64-token tiles and cut
 * into CTA ranges of equal cost as in the balanced mode of mstar_paged_attn_decode, plus one combine launch that merges the
 * prefix and suffix pieces of every (sequence, head) row by log-sum-exp.  Deterministic, CUDA-graph capturable.
 * bf16 pool only.  Other arguments, flags and errors as mstar_paged_attn_decode (num_partitions is always 0).
 */
size_t mstar_paged_attn_decode_cascade_workspace_bytes(int32_t num_seqs, int32_t num_q_heads, int32_t num_kv_heads,
                                                       int32_t head_dim, int32_t max_seq_len);
int mstar_paged_attn_decode_cascade(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool,
                                    const int32_t* block_table, int64_t block_table_stride,
                                    const int32_t* seq_lens, const int32_t* shared_lens, int32_t num_seqs,
                                    int32_t n_branches, int32_t num_q_heads, int32_t max_seq_len, float scale,
                                    uint32_t flags, void* workspace, size_t workspace_bytes, void* stream);

/*
 * mstar_paged_attn_prefill (step a4): many query tokens per sequence, causal over a cached prefix.
 * Query row i (0-based within sequence s, n_s = cu_seqlens_q[s+1]-cu_seqlens_q[s] rows) attends to
 * KV positions j <= (seq_lens[s] - n_s) + i when causal != 0 (bottom-right aligned mask), to all
 * seq_lens[s] positions when causal == 0.  The new tokens' K/V are read from the pool: call
 * mstar_kv_append first (same stream).
 *   out            device, [total_q][Hq][D] bf16 (fp32 with MSTAR_FLAG_OUT_F32)
 *   lse_out        device, [total_q][Hq] fp32 or NULL
 *   q              device, [total_q][Hq][D] bf16 contiguous, ragged by cu_seqlens_q
 *   cu_seqlens_q   device, [S+1] int32, cu_seqlens_q[0] = 0, cu_seqlens_q[S] = total_q
 *   seq_lens       device, [S] int32, total KV length INCLUDING the new tokens (>= n_s)
 *   max_q_len, max_seq_len   host upper bounds on n_s and seq_lens
 *   scale          must be positive and finite (MSTAR_ERR_INVALID_ARG otherwise)
 *   workspace      device, >= mstar_paged_attn_prefill_workspace_bytes(...) bytes, 16-B aligned.  Holds the
 *                  device-built attention plan (PAPER.md:136 builds its plan on the CPU): work units sorted
 *                  heaviest first plus the work counter.  Contents need no initialisation.
 */
size_t mstar_paged_attn_prefill_workspace_bytes(int32_t num_seqs, int32_t total_q, int32_t num_q_heads,
                                                int32_t head_dim);
int mstar_paged_attn_prefill(void* out, float* lse_out, const void* q, const int32_t* cu_seqlens_q,
                             const mstar_kv_pool* pool, const int32_t* block_table,
                             int64_t block_table_stride, const int32_t* seq_lens, int32_t num_seqs,
                             int32_t total_q, int32_t max_q_len, int32_t max_seq_len,
                             int32_t num_q_heads, float scale, int32_t causal, uint32_t flags,
                             void* workspace, size_t workspace_bytes, void* stream);

/*
 * mstar_sample_tokens (last clause): the "cuda-graph-compatible sampling plugin" of the
 * KVCacheEngine.  One token per row from softmax(logits / temperature) restricted by top-k and
 * top-p, drawn with one uniform number per row; all state is device memory, the call only enqueues, so it can be
 * captured and replayed.  Definition (R28, oracle/sampling.py):
 *   z = logits / T.  top-k (0 < k < vocab): keep the tokens with z >= the k-th largest z (ties kept).  top-p
 *   (0 < p < 1): of the kept tokens in descending probability, the shortest prefix of mass >= p, ties with its last
 *   token kept.  u = (x + 1/2) / 2^32 with x = word 0 of Philox4x32-10, counter (step mod 2^32, step div 2^32, row, 0),
 *   key (seed mod 2^32, seed div 2^32).  Token = the first kept index whose running sum of probabilities (index order)
 *   exceeds u times the kept mass.  T = 0: the argmax of the row (lowest index among equals).
 *   tokens_out   device, [num_rows] int32
 *   logits       device, [num_rows][row_stride] fp32 (bf16 with MSTAR_FLAG_LOGITS_BF16), vocab <= row_stride; NaN
 *                entries: undefined; -inf entries never win
 *   temperature  device, [num_rows] fp32 >= 0, or NULL (= 1)
 *   top_k        device, [num_rows] int32 (<= 0 or >= vocab: off), or NULL
 *   top_p        device, [num_rows] fp32 (<= 0 or >= 1: off), or NULL
 *   seeds        device, [num_rows] uint64;  step: device, one uint64 shared by the rows
 * Probabilities are fixed-point (floor(2^32 * exp(z - z_max)), exponential in fp32) and all sums are integers, so the
 * result is run-to-run deterministic; against the fp64 definition a token is correct when u lies within rounding
 * (1e-5) of its interval of the running sum.
 */
int mstar_sample_tokens(int32_t* tokens_out, const void* logits, int64_t row_stride, int32_t num_rows, int32_t vocab,
                        const float* temperature, const int32_t* top_k, const float* top_p, const uint64_t* seeds,
                        uint64_t* step, uint32_t flags, void* stream);

/*
 * mstar_build_slot_mapping: device-side helper so that append -> prefill stays graph-capturable.
 * slot_mapping_out[cu_seqlens_q[s] + i] = block_table[s][j / page_size]*page_size + j % page_size
 * with j = seq_lens[s] - n_s + i.   slot_mapping_out: device, [total_q] int64.
 */
int mstar_build_slot_mapping(const int32_t* block_table, int64_t block_table_stride,
                             const int32_t* cu_seqlens_q, const int32_t* seq_lens, int32_t num_seqs,
                             int32_t total_q, int32_t page_size, int64_t* slot_mapping_out, void* stream);

/* Number of kernels the last call on this thread enqueued (bench.py's gpu_launches claim). */
int32_t mstar_last_launch_count(void);

/* Human-readable name of a status code (static storage). */
const char* mstar_status_string(int status);

/* Library version, "major.minor.patch" (static storage). */
const char* mstar_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MSTAR_ATTN_H_ */
