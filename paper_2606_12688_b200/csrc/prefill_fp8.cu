// prefill_fp8.cu -- mstar_paged_attn_prefill_fp8: paged prefill (and the flow step, causal = 0) over the quantised
// (E4M3) K/V pool (R24-R27).
//
// Prefill is bound by the tensor pipe, not by K/V bytes (config 3 reads 28 MB of K/V for 0.14 TFLOP), and the
// tcgen05 kind::f16 MMA takes no E4M3 operand next to a bf16 one.  So the call has two steps, both kernels of this
// library:
//   1. kv_expand_fp8_kernel   gathers the pages the batch's block table references and writes them DEQUANTISED to
//                             fp16 -- e4m3(code) * scale[page][kv head], the product taken in fp32 (exact: 4 x 24
//                             significant bits), rounded once to nearest even (11 significant bits; saturating at
//                             +-65504, multiples of 2^-24 below 2^-14) -- into a compact scratch pool in the
//                             workspace (page s * maxp + i for logical page i of sequence s), together with the
//                             identity block table of that pool.  One read of the codes, one write of twice the bytes.
//   2. prefill_plan_kernel + prefill_umma_kernel<PAGE, F16 = true> over the scratch pool: the tcgen05 / TMEM kernel of
//      prefill_umma.cu with f16 x f16 MMAs: its two idle warps convert the Q tiles from bf16 to fp16 in shared memory
//      (exact for normal magnitudes), P is rounded to fp16 instead of bf16.
// Against PREFILL_FP8 (fp64 on the exact dequantised values) the roundings are fp16's 2^-12 on K, V and P where the
// bf16 path has 2^-9 on P: the gates of the bf16 path (R11) hold with more margin (R27).
// Measured and dropped: (i) codes kept exact in the scratch pool and the scales applied in fp32 inside the softmax
// warps (a page's K scale on its scores, its V scale folded into the exponent): parity green but 50 % slower than the
// bf16 kernel -- 16 more live registers on warps that already hold a 128-column row, 90 local-memory instructions per
// stage; (ii) K in fp16 with Q left in bf16: a kind::f16 MMA with operands of two formats faults; (iii) K and V both
// rounded to bf16: the stacked bf16 roundings of V, P and the output exceed the 1e-2 row gate on rows with few keys
// (1.0-1.2e-2); (iv) K to bf16, V and P to fp16: inside the gate, but the key rounding alone costs up to 8e-3.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "host_common.h"
#include "ptx.cuh"

namespace mstar {

struct ExpandParams {
    const uint8_t* k8;
    const uint8_t* v8;
    int64_t stride_page, stride_head, stride_token;  // bytes
    const float* k_scale;  // [num_pages][Hkv]
    const float* v_scale;
    const int32_t* block_table;
    int64_t bt_stride;
    const int32_t* seq_lens;
    int32_t S, Hkv, page_size;
    int32_t maxp;       // scratch pages per sequence
    uint16_t* k16;      // scratch pools [S * maxp][Hkv][page_size][128] fp16
    uint16_t* v16;
    int32_t* bt16;      // [S][maxp] identity table of the scratch pool
};

// two E4M3 codes (low 16 bits of w) times the page's scale -> two fp16: e4m3x2 -> f16x2 and f16 -> f32 are exact, the
// fp32 product of a 4-bit and a 24-bit significand is exact, one rounding to fp16 (nearest even, saturating)
__device__ __forceinline__ uint32_t e4m3x2_dequant_f16x2(uint32_t w, float scale) {
    uint32_t h2;
    asm("{\n\t.reg .b16 lo;\n\tcvt.u16.u32 lo, %1;\n\tcvt.rn.f16x2.e4m3x2 %0, lo;\n\t}" : "=r"(h2) : "r"(w));
    const __half2 h = *reinterpret_cast<const __half2*>(&h2);
    const float2 f = __half22float2(h);
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(f.y * scale), "f"(f.x * scale));
    return r;
}

// One block per (sequence, logical page slot, kv head); 128 threads; K and V.  Thread t takes 16-byte chunk t of the
// page's page_size x 128 bytes (page 32: two rounds).
__global__ void __launch_bounds__(128) kv_expand_fp8_kernel(const ExpandParams p) {
    const int i = blockIdx.x;  // logical page of the sequence, < maxp
    const int h = blockIdx.y;
    const int s = blockIdx.z;
    const int L = max(__ldg(p.seq_lens + s), 0);
    if (h == 0 && threadIdx.x == 0) p.bt16[(size_t)s * p.maxp + i] = s * p.maxp + i;
    if (i >= (L + p.page_size - 1) / p.page_size) return;
    const int32_t page = __ldg(p.block_table + (size_t)s * p.bt_stride + i);
    const float ks = __ldg(p.k_scale + (size_t)page * p.Hkv + h);
    const float vs = __ldg(p.v_scale + (size_t)page * p.Hkv + h);
    const size_t src = (size_t)page * p.stride_page + (size_t)h * p.stride_head;
    const size_t dst = (((size_t)s * p.maxp + i) * p.Hkv + h) * p.page_size * 128;
    for (int c = threadIdx.x; c < p.page_size * 8; c += 128) {
        const int tok = c >> 3, d0 = (c & 7) * 16;
        const size_t so = src + (size_t)tok * p.stride_token + d0;
        const uint4 a = *reinterpret_cast<const uint4*>(p.k8 + so);
        const uint4 b = *reinterpret_cast<const uint4*>(p.v8 + so);
        const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
        uint32_t ko[8], vo[8];
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            ko[2 * w] = e4m3x2_dequant_f16x2(aw[w] & 0xffffu, ks);
            ko[2 * w + 1] = e4m3x2_dequant_f16x2(aw[w] >> 16, ks);
            vo[2 * w] = e4m3x2_dequant_f16x2(bw[w] & 0xffffu, vs);
            vo[2 * w + 1] = e4m3x2_dequant_f16x2(bw[w] >> 16, vs);
        }
        uint4* kd = reinterpret_cast<uint4*>(p.k16 + dst + (size_t)tok * 128 + d0);
        uint4* vd = reinterpret_cast<uint4*>(p.v16 + dst + (size_t)tok * 128 + d0);
        kd[0] = make_uint4(ko[0], ko[1], ko[2], ko[3]);
        kd[1] = make_uint4(ko[4], ko[5], ko[6], ko[7]);
        vd[0] = make_uint4(vo[0], vo[1], vo[2], vo[3]);
        vd[1] = make_uint4(vo[4], vo[5], vo[6], vo[7]);
    }
}

struct Fp8PrefillLayout {
    size_t plan, k16, v16, bt16, total;
    int32_t maxp;
};

static Fp8PrefillLayout fp8_prefill_layout(int32_t S, int32_t total_q, int32_t Hq, int32_t Hkv, int32_t page_size,
                                           int32_t max_seq_len) {
    Fp8PrefillLayout l{};
    auto up = [](size_t x, size_t a) { return (x + a - 1) / a * a; };
    l.maxp = (max_seq_len + page_size - 1) / page_size;
    if (l.maxp < 1) l.maxp = 1;
    const size_t pool_bytes = (size_t)S * l.maxp * Hkv * page_size * 128 * 2;
    l.plan = 0;
    l.k16 = up(prefill_umma_workspace_bytes(S, total_q, Hq), 1024);
    l.v16 = up(l.k16 + pool_bytes, 1024);
    l.bt16 = up(l.v16 + pool_bytes, 256);
    l.total = up(l.bt16 + (size_t)S * l.maxp * 4, 256);
    return l;
}

}  // namespace mstar

extern "C" size_t mstar_paged_attn_prefill_fp8_workspace_bytes(int32_t num_seqs, int32_t total_q, int32_t num_q_heads,
                                                               int32_t num_kv_heads, int32_t page_size,
                                                               int32_t max_seq_len) {
    if (num_seqs <= 0 || total_q < 0 || num_q_heads <= 0 || num_kv_heads <= 0 || page_size <= 0 || max_seq_len < 0)
        return 0;
    return mstar::fp8_prefill_layout(num_seqs, total_q, num_q_heads, num_kv_heads, page_size, max_seq_len).total;
}

extern "C" int mstar_paged_attn_prefill_fp8(void* out, float* lse_out, const void* q, const int32_t* cu_seqlens_q,
                                            const mstar_kv_pool* pool8, const float* k_scale, const float* v_scale,
                                            const int32_t* block_table, int64_t block_table_stride,
                                            const int32_t* seq_lens, int32_t num_seqs, int32_t total_q,
                                            int32_t max_q_len, int32_t max_seq_len, int32_t num_q_heads, float scale,
                                            int32_t causal, uint32_t flags, void* workspace, size_t workspace_bytes,
                                            void* stream) {
    using namespace mstar;
    launch_count_reset();
    int rc = check_pool_fp8(pool8);
    if (rc != MSTAR_OK) return rc;
    if (!k_scale || !v_scale || !aligned(k_scale, 4) || !aligned(v_scale, 4)) return MSTAR_ERR_INVALID_ARG;
    if (flags & ~MSTAR_FLAG_OUT_F32) return MSTAR_ERR_INVALID_ARG;
    if (num_seqs < 0 || total_q < 0 || max_q_len < 0 || max_seq_len < 0 || num_q_heads <= 0)
        return MSTAR_ERR_INVALID_ARG;
    if (!(scale > 0.f) || !(scale < 3.0e38f)) return MSTAR_ERR_INVALID_ARG;
    if (num_seqs == 0 || total_q == 0 || max_q_len == 0) return MSTAR_OK;
    if (!out || !q || !cu_seqlens_q || !block_table || !seq_lens) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(out, 16) || !aligned(q, 16)) return MSTAR_ERR_INVALID_ARG;
    const int32_t Hkv = pool8->num_kv_heads, PAGE = pool8->page_size;
    if (num_q_heads % Hkv) return MSTAR_ERR_INVALID_ARG;
    if (num_q_heads / Hkv > 128) return MSTAR_ERR_UNSUPPORTED;
    const Fp8PrefillLayout l = fp8_prefill_layout(num_seqs, total_q, num_q_heads, Hkv, PAGE, max_seq_len);
    if (!workspace || !aligned(workspace, 256)) return MSTAR_ERR_INVALID_ARG;
    if (workspace_bytes < l.total) return MSTAR_ERR_WORKSPACE_TOO_SMALL;
    if ((int64_t)num_seqs * l.maxp * Hkv * PAGE >= (int64_t(1) << 31)) return MSTAR_ERR_UNSUPPORTED;
    if (num_seqs > 65535 || Hkv > 65535) return MSTAR_ERR_UNSUPPORTED;
    uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
    cudaStream_t st = (cudaStream_t)stream;

    ExpandParams e{};
    e.k8 = reinterpret_cast<const uint8_t*>(pool8->k_pool);
    e.v8 = reinterpret_cast<const uint8_t*>(pool8->v_pool);
    e.stride_page = pool8->stride_page;
    e.stride_head = pool8->stride_head;
    e.stride_token = pool8->stride_token;
    e.k_scale = k_scale;
    e.v_scale = v_scale;
    e.block_table = block_table;
    e.bt_stride = block_table_stride;
    e.seq_lens = seq_lens;
    e.S = num_seqs;
    e.Hkv = Hkv;
    e.page_size = PAGE;
    e.maxp = l.maxp;
    e.k16 = reinterpret_cast<uint16_t*>(ws + l.k16);
    e.v16 = reinterpret_cast<uint16_t*>(ws + l.v16);
    e.bt16 = reinterpret_cast<int32_t*>(ws + l.bt16);
    kv_expand_fp8_kernel<<<dim3((unsigned)l.maxp, (unsigned)Hkv, (unsigned)num_seqs), 128, 0, st>>>(e);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);

    // the scratch pool, described like a bf16 pool (16-bit elements; the tensor maps move bytes)
    mstar_kv_pool p16{};
    p16.k_pool = e.k16;
    p16.v_pool = e.v16;
    p16.num_pages = (int64_t)num_seqs * l.maxp;
    p16.page_size = PAGE;
    p16.num_kv_heads = Hkv;
    p16.head_dim = 128;
    p16.stride_token = 128;
    p16.stride_head = (int64_t)PAGE * 128;
    p16.stride_page = (int64_t)Hkv * PAGE * 128;
    PoolMaps maps;
    rc = get_pool_maps(&p16, &maps);
    if (rc != MSTAR_OK) return rc;
    rc = launch_prefill_umma(maps, q, total_q, cu_seqlens_q, e.bt16, l.maxp, seq_lens, num_seqs, num_q_heads, Hkv, PAGE,
                             max_q_len, scale, causal ? 1 : 0, out, lse_out, (flags & MSTAR_FLAG_OUT_F32) ? 1 : 0, 0,
                             ws + l.plan, l.k16, st, /*kv_f16=*/1);
    return rc;
}
