// prefill.cu -- step a4: paged prefill attention, causal over a cached prefix.
//
// v0 kernel (warp-level MMA scaffold): one CTA per (sequence, kv head, block of 16
// query tokens).  A producer warp streams the sequence's K/V pages through the same TMA / 128-B-swizzled
// shared-memory ring as the decode kernel; consumer warp w owns query head kvh*G + w for the CTA's 16
// query rows, so the G grouped heads share every K/V stage.  S = Q K^T and O += P V use
// mma.sync.m16n8k16 bf16 with fp32 accumulation, online softmax in fp32, P rounded to bf16 before PV.
// Causal mask is bottom-right aligned: local query row i sees KV positions j <= (L - n) + i.
#include <cuda_bf16.h>

#include "host_common.h"
#include "ptx.cuh"

namespace mstar {

constexpr int kPrefillTok = 64;      // KV tokens per ring stage
constexpr int kPrefillRows = 16;     // query rows per CTA
constexpr int kPrefillMaxHeads = 8;  // consumer warps (query heads) per CTA
constexpr int kPrefillMaxStages = 8;

struct PrefillParams {
    const uint16_t* q;
    const int32_t* cu_seqlens_q;
    const int32_t* block_table;
    int64_t bt_stride;
    const int32_t* seq_lens;
    int32_t S, Hq, Hkv, G;
    int32_t head_groups;  // ceil(G / 8)
    int32_t nwc;          // consumer warps per CTA = min(G, 8)
    int32_t n_qblocks;    // ceil(max_q_len / 16)
    float scale_log2;
    void* out;
    float* lse;
    int32_t out_f32;
    int32_t causal;
    int32_t nstages;
};

template <int D>
struct PrefillSmem {
    static constexpr int kStageBytes = 2 * kPrefillTok * D * 2;
    static size_t bytes(int nstages) { return 1024 + (size_t)nstages * kStageBytes + 2 * kPrefillMaxStages * 8 + 16; }
};

template <int D, int PAGE>
__global__ void __launch_bounds__(32 * (kPrefillMaxHeads + 1), 1)
prefill_mma_kernel(const __grid_constant__ CUtensorMap kmap, const __grid_constant__ CUtensorMap vmap,
                   const PrefillParams p) {
    constexpr int TOK = kPrefillTok;
    constexpr int PPS = TOK / PAGE;
    constexpr int NH = D / 64;
    constexpr int HT = TOK * 128;
    constexpr int KBYTES = NH * HT;
    using SM = PrefillSmem<D>;

    // block -> (query block, sequence, kv head, head group); heaviest (latest) query blocks first
    int b = blockIdx.x;
    const int hg = b % p.head_groups; b /= p.head_groups;
    const int kvh = b % p.Hkv; b /= p.Hkv;
    const int s = b % p.S; b /= p.S;
    const int qb = p.n_qblocks - 1 - b;
    const int r0 = p.cu_seqlens_q[s];
    const int n = p.cu_seqlens_q[s + 1] - r0;
    const int i0 = qb * kPrefillRows;
    if (i0 >= n) return;
    const int L = p.seq_lens[s];
    const int P = L - n;
    const int rows_here = min(kPrefillRows, n - i0);
    const int kv_end = p.causal ? P + i0 + rows_here : L;
    const int ntiles = (kv_end + TOK - 1) / TOK;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const int nstages = p.nstages;
    const uint32_t ring = base;
    const uint32_t bars = ring + nstages * SM::kStageBytes;
    auto full_bar = [&](int st) { return bars + 8u * st; };
    auto empty_bar = [&](int st) { return bars + 8u * (kPrefillMaxStages + st); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nwc = p.nwc;
    if (threadIdx.x == 0) {
        for (int i = 0; i < nstages; ++i) {
            mbar_init(full_bar(i), 1);
            mbar_init(empty_bar(i), nwc);
        }
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == nwc) {
        // =============================== PRODUCER ===============================
        prefetch_tensormap(&kmap);
        prefetch_tensormap(&vmap);
        const uint64_t pol = policy_evict_last();  // K/V is re-read by the other query blocks / head groups
        constexpr int OPS = PPS * 2 * NH;
        const int op_page = lane / (2 * NH);
        const int op_isv = (lane % (2 * NH)) / NH;
        const int op_half = lane % NH;
        const uint32_t op_off = op_isv * KBYTES + op_half * HT + op_page * (PAGE * 128);
        const int32_t* bt = p.block_table + (size_t)s * p.bt_stride;
        int st = 0, ph = 0;
        for (int t = 0; t < ntiles; ++t) {
            const int rem = kv_end - t * TOK;
            const int npg = min(PPS, (rem + PAGE - 1) / PAGE);
            int pg = -1;
            if (lane < OPS && op_page < npg) pg = __ldg(bt + t * PPS + op_page);
            mbar_wait(empty_bar(st), ph ^ 1);
            if (lane == 0) mbar_arrive_expect_tx(full_bar(st), (uint32_t)(npg * PAGE * D * 2 * 2));
            __syncwarp();
            if (pg >= 0)
                tma_load_4d(ring + st * SM::kStageBytes + op_off, op_isv ? &vmap : &kmap, full_bar(st), op_half * 64,
                            0, kvh, pg, pol);
            if (++st == nstages) { st = 0; ph ^= 1; }
        }
    } else if (warp < nwc) {
        // =============================== CONSUMERS ===============================
        const int g = lane >> 2, t4 = lane & 3;
        const int hl = hg * kPrefillMaxHeads + warp;  // head within the group
        const bool active = hl < p.G;
        const int h = kvh * p.G + (active ? hl : 0);
        // rows g and g+8 of the tile (clamped: rows past n repeat the last valid row and are not stored)
        const int ia = min(i0 + g, n - 1), ib = min(i0 + g + 8, n - 1);
        const int lim_a = p.causal ? P + ia : L - 1;  // last visible KV position (inclusive)
        const int lim_b = p.causal ? P + ib : L - 1;

        uint32_t qa[D / 16][4];
        {
            const uint16_t* qra = p.q + ((size_t)(r0 + ia) * p.Hq + h) * D;
            const uint16_t* qrb = p.q + ((size_t)(r0 + ib) * p.Hq + h) * D;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                qa[ks][0] = __ldg(reinterpret_cast<const uint32_t*>(qra + ks * 16 + 2 * t4));
                qa[ks][1] = __ldg(reinterpret_cast<const uint32_t*>(qrb + ks * 16 + 2 * t4));
                qa[ks][2] = __ldg(reinterpret_cast<const uint32_t*>(qra + ks * 16 + 8 + 2 * t4));
                qa[ks][3] = __ldg(reinterpret_cast<const uint32_t*>(qrb + ks * 16 + 8 + 2 * t4));
            }
        }
        const uint32_t k_rl = (lane >> 4) * 8 + (lane & 7);
        const uint32_t k_csel = (lane >> 3) & 1;
        const uint32_t v_rl = ((lane >> 3) & 1) * 8 + (lane & 7);
        const uint32_t v_csel = lane >> 4;

        float o[D / 8][4];
#pragma unroll
        for (int j = 0; j < D / 8; ++j) o[j][0] = o[j][1] = o[j][2] = o[j][3] = 0.f;
        float m_a = -INFINITY, m_b = -INFINITY, l_a = 0.f, l_b = 0.f;

        int st = 0, ph = 0;
        for (int t = 0; t < ntiles; ++t) {
            mbar_wait(full_bar(st), ph);
            if (active) {
                const uint32_t kb = ring + st * SM::kStageBytes;
                const uint32_t vb = kb + KBYTES;
                const int j0 = t * TOK;
                float sc[TOK / 8][4];
#pragma unroll
                for (int nb = 0; nb < TOK / 8; ++nb) sc[nb][0] = sc[nb][1] = sc[nb][2] = sc[nb][3] = 0.f;
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t chunk = 2 * ks + k_csel;
#pragma unroll
                    for (int np = 0; np < TOK / 16; ++np) {
                        uint32_t b0, b1, b2, b3;
                        ldsm_x4(kb + (chunk >> 3) * HT + swz128(np * 16 + k_rl, chunk & 7), b0, b1, b2, b3);
                        mma_bf16_16816(sc[2 * np], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b0, b1);
                        mma_bf16_16816(sc[2 * np + 1], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b2, b3);
                    }
                }
                if (j0 + TOK - 1 > min(lim_a, lim_b)) {  // stage crosses the causal diagonal / sequence end
#pragma unroll
                    for (int nb = 0; nb < TOK / 8; ++nb) {
                        const int j = j0 + nb * 8 + 2 * t4;
                        if (j > lim_a) sc[nb][0] = -INFINITY;
                        if (j + 1 > lim_a) sc[nb][1] = -INFINITY;
                        if (j > lim_b) sc[nb][2] = -INFINITY;
                        if (j + 1 > lim_b) sc[nb][3] = -INFINITY;
                    }
                }
                float mxa = -INFINITY, mxb = -INFINITY;
#pragma unroll
                for (int nb = 0; nb < TOK / 8; ++nb) {
                    mxa = fmaxf(mxa, fmaxf(sc[nb][0], sc[nb][1]));
                    mxb = fmaxf(mxb, fmaxf(sc[nb][2], sc[nb][3]));
                }
                mxa = fmaxf(mxa, __shfl_xor_sync(0xffffffffu, mxa, 1));
                mxa = fmaxf(mxa, __shfl_xor_sync(0xffffffffu, mxa, 2));
                mxb = fmaxf(mxb, __shfl_xor_sync(0xffffffffu, mxb, 1));
                mxb = fmaxf(mxb, __shfl_xor_sync(0xffffffffu, mxb, 2));
                const float mna = fmaxf(m_a, mxa), mnb = fmaxf(m_b, mxb);
                const float al_a = fast_exp2((m_a - mna) * p.scale_log2);
                const float al_b = fast_exp2((m_b - mnb) * p.scale_log2);
                m_a = mna;
                m_b = mnb;
                const float msa = mna * p.scale_log2, msb = mnb * p.scale_log2;
                float rs_a = 0.f, rs_b = 0.f;
#pragma unroll
                for (int nb = 0; nb < TOK / 8; ++nb) {
                    sc[nb][0] = fast_exp2(sc[nb][0] * p.scale_log2 - msa);
                    sc[nb][1] = fast_exp2(sc[nb][1] * p.scale_log2 - msa);
                    sc[nb][2] = fast_exp2(sc[nb][2] * p.scale_log2 - msb);
                    sc[nb][3] = fast_exp2(sc[nb][3] * p.scale_log2 - msb);
                    rs_a += sc[nb][0] + sc[nb][1];
                    rs_b += sc[nb][2] + sc[nb][3];
                }
                l_a = l_a * al_a + rs_a;
                l_b = l_b * al_b + rs_b;
#pragma unroll
                for (int j = 0; j < D / 8; ++j) {
                    o[j][0] *= al_a; o[j][1] *= al_a; o[j][2] *= al_b; o[j][3] *= al_b;
                }
                // V rows >= kv_end were not loaded (stale shared memory) or hold no token (may be NaN):
                // zero them, p = 0 there for every row (0 * NaN guard)
                const bool tail = j0 + TOK > kv_end;
#pragma unroll
                for (int kt = 0; kt < TOK / 16; ++kt) {
                    const uint32_t pa0 = pack_bf16x2(sc[2 * kt][0], sc[2 * kt][1]);
                    const uint32_t pa1 = pack_bf16x2(sc[2 * kt][2], sc[2 * kt][3]);
                    const uint32_t pa2 = pack_bf16x2(sc[2 * kt + 1][0], sc[2 * kt + 1][1]);
                    const uint32_t pa3 = pack_bf16x2(sc[2 * kt + 1][2], sc[2 * kt + 1][3]);
                    uint32_t vm_lo = 0xffffffffu, vm_hi = 0xffffffffu;
                    if (tail) {
                        const int jt = j0 + kt * 16 + 2 * t4;
                        vm_lo = (jt < kv_end ? 0x0000ffffu : 0u) | (jt + 1 < kv_end ? 0xffff0000u : 0u);
                        vm_hi = (jt + 8 < kv_end ? 0x0000ffffu : 0u) | (jt + 9 < kv_end ? 0xffff0000u : 0u);
                    }
#pragma unroll
                    for (int jj = 0; jj < D / 16; ++jj) {
                        const uint32_t chunk = 2 * jj + v_csel;
                        uint32_t b0, b1, b2, b3;
                        ldsm_x4_trans(vb + (chunk >> 3) * HT + swz128(kt * 16 + v_rl, chunk & 7), b0, b1, b2, b3);
                        if (tail) { b0 &= vm_lo; b1 &= vm_hi; b2 &= vm_lo; b3 &= vm_hi; }
                        mma_bf16_16816(o[2 * jj], pa0, pa1, pa2, pa3, b0, b1);
                        mma_bf16_16816(o[2 * jj + 1], pa0, pa1, pa2, pa3, b2, b3);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(st));
            if (++st == nstages) { st = 0; ph ^= 1; }
        }
        if (active) {
            l_a += __shfl_xor_sync(0xffffffffu, l_a, 1);
            l_a += __shfl_xor_sync(0xffffffffu, l_a, 2);
            l_b += __shfl_xor_sync(0xffffffffu, l_b, 1);
            l_b += __shfl_xor_sync(0xffffffffu, l_b, 2);
            const float inv_a = 1.f / l_a, inv_b = 1.f / l_b;
            const bool wa = i0 + g < n, wb = i0 + g + 8 < n;
            const size_t oa = ((size_t)(r0 + i0 + g) * p.Hq + h) * D;
            const size_t ob = ((size_t)(r0 + i0 + g + 8) * p.Hq + h) * D;
#pragma unroll
            for (int j = 0; j < D / 8; ++j) {
                const int d = j * 8 + 2 * t4;
                if (p.out_f32) {
                    float* of = reinterpret_cast<float*>(p.out);
                    if (wa) *reinterpret_cast<float2*>(of + oa + d) = make_float2(o[j][0] * inv_a, o[j][1] * inv_a);
                    if (wb) *reinterpret_cast<float2*>(of + ob + d) = make_float2(o[j][2] * inv_b, o[j][3] * inv_b);
                } else {
                    uint16_t* oh = reinterpret_cast<uint16_t*>(p.out);
                    if (wa) *reinterpret_cast<uint32_t*>(oh + oa + d) = pack_bf16x2(o[j][0] * inv_a, o[j][1] * inv_a);
                    if (wb) *reinterpret_cast<uint32_t*>(oh + ob + d) = pack_bf16x2(o[j][2] * inv_b, o[j][3] * inv_b);
                }
            }
            if (p.lse && t4 == 0) {
                if (wa) p.lse[(size_t)(r0 + i0 + g) * p.Hq + h] = (m_a * p.scale_log2 + log2f(l_a)) * 0.6931471805599453f;
                if (wb) p.lse[(size_t)(r0 + i0 + g + 8) * p.Hq + h] = (m_b * p.scale_log2 + log2f(l_b)) * 0.6931471805599453f;
            }
        }
    }
}

template <int D, int PAGE>
static int launch_prefill(const PoolMaps& maps, PrefillParams& p, cudaStream_t stream) {
    using SM = PrefillSmem<D>;
    const int max_smem = device_max_smem_optin();
    int nstages = (int)(((int64_t)max_smem - 1024 - 2 * kPrefillMaxStages * 8 - 16) / SM::kStageBytes);
    if (nstages > 4) nstages = 4;  // 4 x 64 tokens in flight per CTA is ample for an L2-resident stream
    if (nstages < 2) return MSTAR_ERR_UNSUPPORTED;
    p.nstages = nstages;
    auto kern = prefill_mma_kernel<D, PAGE>;
    static PerDeviceOnce attr_once;  // per instantiation
    MSTAR_CUDA_OK(set_max_dynamic_smem(attr_once, kern, max_smem));
    const int64_t grid = (int64_t)p.n_qblocks * p.S * p.Hkv * p.head_groups;
    if (grid > 0x7fffffffLL) return MSTAR_ERR_UNSUPPORTED;
    kern<<<(unsigned)grid, 32 * (p.nwc + 1), SM::bytes(nstages), stream>>>(maps.k, maps.v, p);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}

}  // namespace mstar

extern "C" size_t mstar_paged_attn_prefill_workspace_bytes(int32_t num_seqs, int32_t total_q, int32_t num_q_heads,
                                                           int32_t head_dim) {
    (void)head_dim;
    if (num_seqs < 0 || total_q < 0 || num_q_heads <= 0) return 0;
    return mstar::prefill_umma_workspace_bytes(num_seqs, total_q, num_q_heads);
}

extern "C" int mstar_paged_attn_prefill(void* out, float* lse_out, const void* q, const int32_t* cu_seqlens_q,
                                        const mstar_kv_pool* pool, const int32_t* block_table,
                                        int64_t block_table_stride, const int32_t* seq_lens, int32_t num_seqs,
                                        int32_t total_q, int32_t max_q_len, int32_t max_seq_len, int32_t num_q_heads,
                                        float scale, int32_t causal, uint32_t flags, void* workspace,
                                        size_t workspace_bytes, void* stream) {
    using namespace mstar;
    (void)max_seq_len;
    launch_count_reset();
    int rc = check_pool(pool);
    if (rc != MSTAR_OK) return rc;
    if (flags & ~(MSTAR_FLAG_OUT_F32 | MSTAR_FLAG_PREFILL_MMA_SYNC | MSTAR_FLAG_PREFILL_REUSE_PLAN))
        return MSTAR_ERR_INVALID_ARG;
    if (num_seqs < 0 || total_q < 0 || max_q_len < 0 || num_q_heads <= 0) return MSTAR_ERR_INVALID_ARG;
    if (!(scale > 0.f) || !(scale < 3.0e38f)) return MSTAR_ERR_INVALID_ARG;
    if (num_seqs == 0 || total_q == 0 || max_q_len == 0) return MSTAR_OK;
    if (!out || !q || !cu_seqlens_q || !block_table || !seq_lens) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(out, 16) || !aligned(q, 16)) return MSTAR_ERR_INVALID_ARG;
    if (num_q_heads % pool->num_kv_heads) return MSTAR_ERR_INVALID_ARG;

    PrefillParams p{};
    p.q = reinterpret_cast<const uint16_t*>(q);
    p.cu_seqlens_q = cu_seqlens_q;
    p.block_table = block_table;
    p.bt_stride = block_table_stride;
    p.seq_lens = seq_lens;
    p.S = num_seqs;
    p.Hq = num_q_heads;
    p.Hkv = pool->num_kv_heads;
    p.G = num_q_heads / pool->num_kv_heads;
    p.head_groups = (p.G + kPrefillMaxHeads - 1) / kPrefillMaxHeads;
    p.nwc = p.G < kPrefillMaxHeads ? p.G : kPrefillMaxHeads;
    p.n_qblocks = (max_q_len + kPrefillRows - 1) / kPrefillRows;
    p.scale_log2 = scale * 1.4426950408889634f;
    p.out = out;
    p.lse = lse_out;
    p.out_f32 = (flags & MSTAR_FLAG_OUT_F32) ? 1 : 0;
    p.causal = causal ? 1 : 0;

    PoolMaps maps;
    rc = get_pool_maps(pool, &maps);
    if (rc != MSTAR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int D = pool->head_dim, PAGE = pool->page_size;
    if ((D == 128 || D == 64) && p.G <= 128 && !(flags & MSTAR_FLAG_PREFILL_MMA_SYNC))  // tcgen05 / TMEM path
        return launch_prefill_umma(maps, q, total_q, cu_seqlens_q, block_table, block_table_stride, seq_lens, num_seqs,
                                   num_q_heads, pool->num_kv_heads, PAGE, max_q_len, scale, p.causal, out, lse_out,
                                   p.out_f32, (flags & MSTAR_FLAG_PREFILL_REUSE_PLAN) ? 1 : 0, workspace,
                                   workspace_bytes, st, /*kv_f16=*/0, D);
    if (D == 128 && PAGE == 16) return launch_prefill<128, 16>(maps, p, st);
    if (D == 128 && PAGE == 32) return launch_prefill<128, 32>(maps, p, st);
    if (D == 64 && PAGE == 16) return launch_prefill<64, 16>(maps, p, st);
    if (D == 64 && PAGE == 32) return launch_prefill<64, 32>(maps, p, st);
    return MSTAR_ERR_UNSUPPORTED;
}
