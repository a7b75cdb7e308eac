// kv_transfer.cu -- page moves around the paged K/V pool: the data-path half of
// "paging, offload, by-reference transfer" and of prefill/decode disaggregation:
//   mstar_kv_copy_pages   whole pages pool -> pool (same or different pool, e.g. a staging pool in pinned host
//                         memory mapped into the device address space), K and V, all heads;
//   mstar_kv_gather       pool -> contiguous [tokens][Hkv][D] through the block table (the inverse of append).
// Both are HBM-bound bit copies: one thread per 16-byte chunk, LDG.128 -> STG.128, several chunks in flight per
// thread, 64-bit addressing, strides honoured (HND and NHD pools).  Algorithmic bytes: 2 * Hkv * D * 2 B per token
// (page_size tokens per page) read + the same written.
#include "host_common.h"

namespace mstar {

// Coherent streaming load (not the read-only .nc path): mstar_kv_copy_pages may read and write the same pool in one
// launch, and .nc is only defined for data no thread of the grid writes.
__device__ __forceinline__ int4 ldg_stream16(const void* p) {
    int4 r;
    asm volatile("ld.global.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

struct PoolGeom {
    uint16_t* k;
    uint16_t* v;
    int64_t stride_page, stride_head, stride_token;
};

template <int UNROLL>
__global__ void __launch_bounds__(256) kv_copy_pages_kernel(PoolGeom dst, PoolGeom src,
                                                            const int64_t* __restrict__ dst_pages,
                                                            const int64_t* __restrict__ src_pages, int64_t n_chunks,
                                                            int32_t cpr /* D/8 */, int32_t page_size, int32_t Hkv) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t chunks_per_page = (int64_t)Hkv * page_size * cpr;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < n_chunks; i0 += stride * UNROLL) {
        int4 kv[UNROLL], vv[UNROLL];
        int64_t d[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int64_t i = i0 + u * stride;
            d[u] = -1;
            if (i < n_chunks) {
                const int64_t pair = i / chunks_per_page;
                int64_t r = i - pair * chunks_per_page;
                const int32_t h = (int32_t)(r / ((int64_t)page_size * cpr));
                r -= (int64_t)h * page_size * cpr;
                const int32_t tok = (int32_t)(r / cpr);
                const int32_t c = (int32_t)(r - (int64_t)tok * cpr);
                const int64_t sp = __ldg(src_pages + pair), dp = __ldg(dst_pages + pair);
                if (sp >= 0 && dp >= 0) {
                    const int64_t so = sp * src.stride_page + h * src.stride_head + tok * src.stride_token + c * 8;
                    d[u] = dp * dst.stride_page + h * dst.stride_head + tok * dst.stride_token + c * 8;
                    kv[u] = ldg_stream16(src.k + so);
                    vv[u] = ldg_stream16(src.v + so);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            if (d[u] >= 0) {
                *reinterpret_cast<int4*>(dst.k + d[u]) = kv[u];
                *reinterpret_cast<int4*>(dst.v + d[u]) = vv[u];
            }
        }
    }
}

template <int UNROLL>
__global__ void __launch_bounds__(256) kv_gather_kernel(PoolGeom src, const int32_t* __restrict__ block_table,
                                                        int64_t bt_stride, const int32_t* __restrict__ seq_lens,
                                                        const int32_t* __restrict__ cu_out, int32_t S,
                                                        uint16_t* __restrict__ k_out, uint16_t* __restrict__ v_out,
                                                        int64_t n_chunks, int32_t cpr, int32_t page_size,
                                                        int32_t Hkv) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t chunks_per_tok = (int64_t)Hkv * cpr;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < n_chunks; i0 += stride * UNROLL) {
        int4 kv[UNROLL], vv[UNROLL];
        bool on[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int64_t i = i0 + u * stride;
            on[u] = false;
            if (i < n_chunks) {
                const int64_t t = i / chunks_per_tok;  // output token row
                const int64_t r = i - t * chunks_per_tok;
                const int32_t h = (int32_t)(r / cpr);
                const int32_t c = (int32_t)(r - (int64_t)h * cpr);
                int lo = 0, hi = S;  // cu_out[lo] <= t < cu_out[hi]
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (__ldg(cu_out + mid) <= t) lo = mid; else hi = mid;
                }
                const int32_t j = (int32_t)(t - __ldg(cu_out + lo));
                if (j < __ldg(seq_lens + lo)) {  // rows past a sequence's length (padding in cu_out) are left alone
                    const int64_t page = __ldg(block_table + (int64_t)lo * bt_stride + j / page_size);
                    const int64_t so = page * src.stride_page + h * src.stride_head +
                                       (int64_t)(j % page_size) * src.stride_token + c * 8;
                    kv[u] = ldg_stream16(src.k + so);
                    vv[u] = ldg_stream16(src.v + so);
                    on[u] = true;
                }
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            if (on[u]) {
                const int64_t i = i0 + u * stride;
                reinterpret_cast<int4*>(k_out)[i] = kv[u];
                reinterpret_cast<int4*>(v_out)[i] = vv[u];
            }
        }
    }
}

// In-flight depth (A/B on one box, thinker pool p = 16 / a 4 x 32768 batch p = 32): copy_pages with 4 loads per thread
// takes 99.3 / 172.0 us on 4 blocks per SM against 101.3 / 176.1 on 8 and 142 / 226 on 2; the gather with 1 load per
// thread on 8 blocks per SM 111.6 / 185 us against 121.8 / 183 with 4 loads (its dependent look-ups -- cu_seqlens
// search, block table -- already keep many rows in flight).
static unsigned copy_grid(int64_t n_chunks, int unroll, int blocks_per_sm) {
    int64_t blocks = (n_chunks + 256LL * unroll - 1) / (256LL * unroll);
    const int64_t max_blocks = (int64_t)device_sm_count() * blocks_per_sm;
    if (blocks > max_blocks) blocks = max_blocks;
    return (unsigned)(blocks < 1 ? 1 : blocks);
}

static PoolGeom geom_of(const mstar_kv_pool* p) {
    return PoolGeom{(uint16_t*)p->k_pool, (uint16_t*)p->v_pool, p->stride_page, p->stride_head, p->stride_token};
}

}  // namespace mstar

extern "C" int mstar_kv_copy_pages(const mstar_kv_pool* dst_pool, const mstar_kv_pool* src_pool,
                                   const int64_t* dst_pages, const int64_t* src_pages, int64_t num_pairs,
                                   void* stream) {
    using namespace mstar;
    launch_count_reset();
    int rc = check_pool(dst_pool);
    if (rc != MSTAR_OK) return rc;
    rc = check_pool(src_pool);
    if (rc != MSTAR_OK) return rc;
    if (dst_pool->page_size != src_pool->page_size || dst_pool->num_kv_heads != src_pool->num_kv_heads ||
        dst_pool->head_dim != src_pool->head_dim)
        return MSTAR_ERR_INVALID_ARG;
    if (num_pairs < 0) return MSTAR_ERR_INVALID_ARG;
    if (num_pairs == 0) return MSTAR_OK;
    if (!dst_pages || !src_pages || !aligned(dst_pages, 8) || !aligned(src_pages, 8)) return MSTAR_ERR_INVALID_ARG;
    const int32_t cpr = src_pool->head_dim / 8;
    const int64_t n_chunks = num_pairs * src_pool->num_kv_heads * src_pool->page_size * cpr;
    constexpr int UNROLL = 4;
    kv_copy_pages_kernel<UNROLL><<<copy_grid(n_chunks, UNROLL, 4), 256, 0, (cudaStream_t)stream>>>(
        geom_of(dst_pool), geom_of(src_pool), dst_pages, src_pages, n_chunks, cpr, src_pool->page_size,
        src_pool->num_kv_heads);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}

extern "C" int mstar_kv_gather(void* k_out, void* v_out, const mstar_kv_pool* pool, const int32_t* block_table,
                               int64_t block_table_stride, const int32_t* seq_lens, const int32_t* cu_seqlens_out,
                               int32_t num_seqs, int64_t total_tokens, void* stream) {
    using namespace mstar;
    launch_count_reset();
    int rc = check_pool(pool);
    if (rc != MSTAR_OK) return rc;
    if (num_seqs < 0 || total_tokens < 0) return MSTAR_ERR_INVALID_ARG;
    if (num_seqs == 0 || total_tokens == 0) return MSTAR_OK;
    if (!k_out || !v_out || !block_table || !seq_lens || !cu_seqlens_out) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(k_out, 16) || !aligned(v_out, 16)) return MSTAR_ERR_INVALID_ARG;
    const int32_t cpr = pool->head_dim / 8;
    const int64_t n_chunks = total_tokens * pool->num_kv_heads * cpr;
    constexpr int UNROLL = 1;
    kv_gather_kernel<UNROLL><<<copy_grid(n_chunks, UNROLL, 8), 256, 0, (cudaStream_t)stream>>>(
        geom_of(pool), block_table, block_table_stride, seq_lens, cu_seqlens_out, num_seqs, (uint16_t*)k_out,
        (uint16_t*)v_out, n_chunks, cpr, pool->page_size, pool->num_kv_heads);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}
