// kv_append.cu -- step a1: scatter the step's new K/V rows into their pool pages (bit copy).
//
// HBM-bound copy with no arithmetic: every thread moves 16-B vectors with LDG.128 -> STG.128;
// consecutive threads move consecutive 16-B chunks of one (token, kv head) row, so both the
// contiguous read of k_new/v_new and the scattered write (D*2-byte runs) are fully coalesced.
// Algorithmic bytes per new token: 2 * Hkv * D * 2 B read + the same written.
#include "host_common.h"

namespace mstar {

__device__ __forceinline__ int4 ldg_stream(const int4* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

template <int UNROLL>
__global__ void __launch_bounds__(256) kv_append_kernel(uint16_t* __restrict__ k_pool, uint16_t* __restrict__ v_pool,
                                                        const uint16_t* __restrict__ k_new,
                                                        const uint16_t* __restrict__ v_new,
                                                        const int64_t* __restrict__ slot_mapping, int64_t n_chunks,
                                                        int32_t chunks_per_row /* D/8 */, int32_t Hkv,
                                                        int32_t page_size, int64_t stride_page, int64_t stride_head,
                                                        int64_t stride_token) {
    // a decode launched behind this append may start its set-up now; it reads the pool only after this grid is done
    asm volatile("griddepcontrol.launch_dependents;");
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i0 < n_chunks; i0 += stride * UNROLL) {
        int4 kv[UNROLL], vv[UNROLL];
        int64_t dst[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int64_t i = i0 + u * stride;
            dst[u] = -1;
            if (i < n_chunks) {
                const int64_t row = i / chunks_per_row;  // (token, head)
                const int32_t c = (int32_t)(i - row * chunks_per_row);
                const int64_t t = row / Hkv;
                const int32_t h = (int32_t)(row - t * Hkv);
                const int64_t slot = __ldg(slot_mapping + t);
                if (slot >= 0) {
                    const int64_t page = slot / page_size;
                    const int64_t off = slot - page * page_size;
                    dst[u] = page * stride_page + h * stride_head + off * stride_token + (int64_t)c * 8;
                    kv[u] = ldg_stream(reinterpret_cast<const int4*>(k_new) + i);
                    vv[u] = ldg_stream(reinterpret_cast<const int4*>(v_new) + i);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            if (dst[u] >= 0) {
                *reinterpret_cast<int4*>(k_pool + dst[u]) = kv[u];
                *reinterpret_cast<int4*>(v_pool + dst[u]) = vv[u];
            }
        }
    }
}

__global__ void build_slot_mapping_kernel(const int32_t* __restrict__ block_table, int64_t bt_stride,
                                          const int32_t* __restrict__ cu_seqlens_q,
                                          const int32_t* __restrict__ seq_lens, int32_t num_seqs, int32_t page_size,
                                          int64_t* __restrict__ slot_out) {
    for (int s = blockIdx.y; s < num_seqs; s += gridDim.y) {
        const int r0 = cu_seqlens_q[s], n = cu_seqlens_q[s + 1] - r0;
        const int P = seq_lens[s] - n;
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
            const int j = P + i;
            const int64_t page = block_table[(int64_t)s * bt_stride + j / page_size];
            slot_out[r0 + i] = page * page_size + j % page_size;
        }
    }
}

}  // namespace mstar

extern "C" int mstar_kv_append(const mstar_kv_pool* pool, const void* k_new, const void* v_new,
                               const int64_t* slot_mapping, int64_t num_tokens, void* stream) {
    using namespace mstar;
    launch_count_reset();
    int rc = check_pool(pool);
    if (rc != MSTAR_OK) return rc;
    if (num_tokens < 0) return MSTAR_ERR_INVALID_ARG;
    if (num_tokens == 0) return MSTAR_OK;
    if (!k_new || !v_new || !slot_mapping) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(k_new, 16) || !aligned(v_new, 16) || !aligned(slot_mapping, 8)) return MSTAR_ERR_INVALID_ARG;
    const int32_t cpr = pool->head_dim / 8;
    const int64_t n_chunks = num_tokens * pool->num_kv_heads * cpr;
    constexpr int UNROLL = 4;
    const int threads = 256;
    int64_t blocks = (n_chunks + (int64_t)threads * UNROLL - 1) / ((int64_t)threads * UNROLL);
    const int64_t max_blocks = (int64_t)device_sm_count() * 8;  // 8 x 256 threads resident per SM
    if (blocks > max_blocks) blocks = max_blocks;
    kv_append_kernel<UNROLL><<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(
        (uint16_t*)pool->k_pool, (uint16_t*)pool->v_pool, (const uint16_t*)k_new, (const uint16_t*)v_new, slot_mapping,
        n_chunks, cpr, pool->num_kv_heads, pool->page_size, pool->stride_page, pool->stride_head, pool->stride_token);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}

extern "C" int mstar_build_slot_mapping(const int32_t* block_table, int64_t block_table_stride,
                                        const int32_t* cu_seqlens_q, const int32_t* seq_lens, int32_t num_seqs,
                                        int32_t total_q, int32_t page_size, int64_t* slot_mapping_out, void* stream) {
    using namespace mstar;
    launch_count_reset();
    if (num_seqs < 0 || total_q < 0 || (page_size != 16 && page_size != 32)) return MSTAR_ERR_INVALID_ARG;
    if (num_seqs == 0 || total_q == 0) return MSTAR_OK;
    if (!block_table || !cu_seqlens_q || !seq_lens || !slot_mapping_out) return MSTAR_ERR_INVALID_ARG;
    int per_seq = (total_q + num_seqs - 1) / num_seqs;
    dim3 grid((unsigned)((per_seq + 255) / 256 > 64 ? 64 : (per_seq + 255) / 256), (unsigned)(num_seqs > 4096 ? 4096 : num_seqs));
    build_slot_mapping_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(block_table, block_table_stride, cu_seqlens_q,
                                                                      seq_lens, num_seqs, page_size, slot_mapping_out);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}
