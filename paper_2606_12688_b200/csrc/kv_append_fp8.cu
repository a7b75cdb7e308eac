// kv_append_fp8.cu -- quantising K/V append: bf16 rows -> E4M3 codes in an fp8 page pool.
//
// Definition (include/mstar_attn.h, R24-R25): code = RNE_satfinite_e4m3( fp32(x) / scale[page][h] ) with
// the division in IEEE fp32.  HBM-bound like kv_append: one thread reads a 16-B chunk (8 bf16) of the K row and of
// the V row (LDG.128, streaming), divides by the page's scale (div.rn.f32), converts with
// cvt.rn.satfinite.e4m3x2.f32 and writes 8 bytes of each pool; consecutive threads cover one (token, head) row,
// so a row leaves as one 128-byte line.  Algorithmic bytes per new token: 2*Hkv*D*2 read + 2*Hkv*D written.
#include <cuda_fp8.h>

#include "host_common.h"

namespace mstar {

__device__ __forceinline__ int4 ldg_stream16(const int4* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

// two bf16 (packed in w) -> two E4M3 codes (low byte = low half of w)
__device__ __forceinline__ uint32_t quant2(uint32_t w, float scale) {
    const float x0 = __uint_as_float(w << 16), x1 = __uint_as_float(w & 0xffff0000u);
    const float2 y = make_float2(__fdiv_rn(x0, scale), __fdiv_rn(x1, scale));
    return (uint32_t)__nv_cvt_float2_to_fp8x2(y, __NV_SATFINITE, __NV_E4M3);
}
__device__ __forceinline__ uint2 quant8(const int4& v, float scale) {
    uint2 r;
    r.x = quant2((uint32_t)v.x, scale) | (quant2((uint32_t)v.y, scale) << 16);
    r.y = quant2((uint32_t)v.z, scale) | (quant2((uint32_t)v.w, scale) << 16);
    return r;
}

__global__ void __launch_bounds__(256) kv_append_fp8_kernel(uint8_t* __restrict__ k_pool, uint8_t* __restrict__ v_pool,
                                                            const float* __restrict__ k_scale,
                                                            const float* __restrict__ v_scale,
                                                            const uint16_t* __restrict__ k_new,
                                                            const uint16_t* __restrict__ v_new,
                                                            const int64_t* __restrict__ slot_mapping, int64_t n_chunks,
                                                            int32_t chunks_per_row /* D/8 */, int32_t Hkv,
                                                            int32_t page_size, int64_t stride_page, int64_t stride_head,
                                                            int64_t stride_token) {
    // a decode launched behind this append may start its set-up now; it reads the pool only after this grid is done
    asm volatile("griddepcontrol.launch_dependents;");
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_chunks; i += stride) {
        const int64_t row = i / chunks_per_row;  // (token, head)
        const int32_t c = (int32_t)(i - row * chunks_per_row);
        const int64_t t = row / Hkv;
        const int32_t h = (int32_t)(row - t * Hkv);
        const int64_t slot = __ldg(slot_mapping + t);
        if (slot < 0) continue;
        const int64_t page = slot / page_size;
        const int64_t off = slot - page * page_size;
        const int64_t dst = page * stride_page + h * stride_head + off * stride_token + (int64_t)c * 8;
        const float ks = __ldg(k_scale + page * Hkv + h), vs = __ldg(v_scale + page * Hkv + h);
        const int4 kv = ldg_stream16(reinterpret_cast<const int4*>(k_new) + i);
        const int4 vv = ldg_stream16(reinterpret_cast<const int4*>(v_new) + i);
        *reinterpret_cast<uint2*>(k_pool + dst) = quant8(kv, ks);
        *reinterpret_cast<uint2*>(v_pool + dst) = quant8(vv, vs);
    }
}

}  // namespace mstar

extern "C" int mstar_kv_append_fp8(const mstar_kv_pool* pool, const float* k_scale, const float* v_scale,
                                   const void* k_new, const void* v_new, const int64_t* slot_mapping,
                                   int64_t num_tokens, void* stream) {
    using namespace mstar;
    launch_count_reset();
    int rc = check_pool_fp8(pool);
    if (rc != MSTAR_OK) return rc;
    if (num_tokens < 0) return MSTAR_ERR_INVALID_ARG;
    if (num_tokens == 0) return MSTAR_OK;
    if (!k_new || !v_new || !slot_mapping || !k_scale || !v_scale) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(k_new, 16) || !aligned(v_new, 16) || !aligned(slot_mapping, 8) || !aligned(k_scale, 4) ||
        !aligned(v_scale, 4))
        return MSTAR_ERR_INVALID_ARG;
    const int32_t cpr = pool->head_dim / 8;
    const int64_t n_chunks = num_tokens * pool->num_kv_heads * cpr;
    const int threads = 256;
    int64_t blocks = (n_chunks + threads - 1) / threads;
    const int64_t max_blocks = (int64_t)device_sm_count() * 8;
    if (blocks > max_blocks) blocks = max_blocks;
    kv_append_fp8_kernel<<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(
        (uint8_t*)pool->k_pool, (uint8_t*)pool->v_pool, k_scale, v_scale, (const uint16_t*)k_new,
        (const uint16_t*)v_new, slot_mapping, n_chunks, cpr, pool->num_kv_heads, pool->page_size, pool->stride_page,
        pool->stride_head, pool->stride_token);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}
