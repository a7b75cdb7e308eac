// prefill_umma.cu -- step a4 on the 5th-generation tensor cores: paged prefill attention, causal over a
// cached prefix, with tcgen05.mma, accumulators in TMEM and TMA-fed operand tiles (head_dim 128).
//
// Design.  Persistent CTAs (one per SM), 12 warps:
//   warp 0      TMA producer: Q tiles (3-D boxes over [token][head][d]) and 128-token K / V stages gathered
//               page by page through the block table (4-D boxes, 128-B swizzle), double-buffered;
//   warp 1      MMA issuer (one elected lane): S = Q K^T (operands in shared memory) and O += P V (P read from
//               TMEM, V MN-major from shared memory), M = 128, N = 128, K = 16 per instruction;
//   warps 4-7   softmax warpgroup of Q tile A, warps 8-11 of Q tile B: thread = query row = TMEM lane;
//               tcgen05.ld S, mask, max, exp2, row sum (no shuffles: a thread owns its row), P -> bf16 ->
//               tcgen05.st into the columns S occupied; lazy rescale of O in TMEM only when the running max
//               grows by more than 2^8; epilogue O / l -> bf16 -> global.
// A work unit is (sequence, kv head, block of 2*tq query tokens), tq = floor(128 / G): the G grouped query
// heads of a kv head are packed into the 128 rows of a Q tile (row = token*G + head), so one K/V stage serves
// all of them and the causal diagonal wastes at most tq columns.  The two Q tiles of a unit ping-pong: while
// one warpgroup does softmax on its S, the tensor core works on the other tile.
// TMEM (512 columns): S_A [0,128)  S_B [128,256)  O_A [256,384)  O_B [384,512); P aliases the first 64
// columns of its S.
#include <cuda_bf16.h>

#include "host_common.h"
#include "ptx.cuh"
#include "umma.cuh"

namespace mstar {

constexpr int kPuTok = 128;       // KV tokens per stage
constexpr int kPuThreads = 384;   // 12 warps
constexpr int kPuHT = 128 * 128;  // bytes of a half tile: 128 rows x 64 bf16, 128-B swizzled
constexpr float kPuTau = 8.0f;    // lazy-rescale threshold, log2 units

struct PrefillUmmaParams {
    const int32_t* cu_seqlens_q;
    const int32_t* block_table;
    int64_t bt_stride;
    const int32_t* seq_lens;
    int32_t S, Hq, Hkv, G;
    int32_t tq;       // query tokens per Q tile = floor(128 / G)
    int32_t nqb;      // query blocks (of 2*tq tokens) per sequence, from the host bound max_q_len
    float scale_log2;
    void* out;
    float* lse;
    int32_t out_f32;
    int32_t causal;
};

struct PuUnit {
    int s, kvh, t0, n, P, L, r0, kv_end, T;
    bool valid;
};

__device__ __forceinline__ PuUnit pu_unit(const PrefillUmmaParams& p, int u) {
    PuUnit x;
    const int per = p.S * p.Hkv;
    const int qb = p.nqb - 1 - u / per;  // heaviest (latest) query blocks first
    const int rem = u % per;
    x.s = rem / p.Hkv;
    x.kvh = rem % p.Hkv;
    x.r0 = __ldg(p.cu_seqlens_q + x.s);
    x.n = __ldg(p.cu_seqlens_q + x.s + 1) - x.r0;
    x.t0 = qb * 2 * p.tq;
    x.valid = x.t0 < x.n;
    x.L = __ldg(p.seq_lens + x.s);
    x.P = x.L - x.n;
    const int rows_tok = min(2 * p.tq, x.n - x.t0);
    x.kv_end = p.causal ? x.P + x.t0 + rows_tok : x.L;
    x.T = (x.kv_end + kPuTok - 1) / kPuTok;
    return x;
}

// shared memory map (offsets from the 1024-aligned base)
constexpr int kPuQ = 0;                     // 2 tiles x 2 halves
constexpr int kPuK = 4 * kPuHT;             // 2 stages x 2 halves
constexpr int kPuV = 8 * kPuHT;             // 2 stages x 2 halves
constexpr int kPuBars = 12 * kPuHT;         // barriers
constexpr int kPuSmemBytes = 12 * kPuHT + 256 + 1024;
enum { B_QFULL = 0, B_QEMPTY, B_KFULL0, B_KFULL1, B_KEMPTY0, B_KEMPTY1, B_VFULL0, B_VFULL1, B_VEMPTY0, B_VEMPTY1,
       B_SFULL0, B_SFULL1, B_PFULL0, B_PFULL1, B_OFULL0, B_OFULL1, B_OEMPTY0, B_OEMPTY1, B_COUNT };

template <int PAGE>
__global__ void __launch_bounds__(kPuThreads, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap qmap, const __grid_constant__ CUtensorMap kmap,
                    const __grid_constant__ CUtensorMap vmap, const PrefillUmmaParams p) {
    constexpr int D = 128;
    constexpr int PPS = kPuTok / PAGE;  // pages per stage
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t bars = base + kPuBars;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(gbase + kPuBars + B_COUNT * 8);
    auto bar = [&](int i) { return bars + 8u * i; };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        mbar_init(bar(B_QFULL), 1);
        mbar_init(bar(B_QEMPTY), 1);
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar(B_KFULL0 + i), 1);
            mbar_init(bar(B_KEMPTY0 + i), 1);
            mbar_init(bar(B_VFULL0 + i), 1);
            mbar_init(bar(B_VEMPTY0 + i), 1);
            mbar_init(bar(B_SFULL0 + i), 1);
            mbar_init(bar(B_PFULL0 + i), 4);
            mbar_init(bar(B_OFULL0 + i), 1);
            mbar_init(bar(B_OEMPTY0 + i), 4);
        }
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc(smem_u32(tmem_slot), 512);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int total_units = p.nqb * p.S * p.Hkv;
    const int rows_used = p.tq * p.G;  // rows of a Q tile that carry (token, head) pairs

    if (warp == 0) {
        // =============================== TMA PRODUCER ===============================
        prefetch_tensormap(&qmap);
        prefetch_tensormap(&kmap);
        prefetch_tensormap(&vmap);
        const uint64_t pol_kv = policy_evict_last();   // K/V re-read by other query blocks of the sequence
        const uint64_t pol_q = policy_evict_first();
        // lane -> (K or V, page, half): PPS*2 ops for K on the low lanes, PPS*2 for V after them
        constexpr int OPS1 = PPS * 2;
        const int op_isv = lane / OPS1;
        const int op_page = (lane % OPS1) / 2;
        const int op_half = lane & 1;
        const bool op_on = lane < 2 * OPS1;
        uint32_t qph = 0, kvph = 0;
        int slot = 0;
        for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
            const PuUnit x = pu_unit(p, u);
            if (!x.valid) continue;
            mbar_wait(bar(B_QEMPTY), qph ^ 1);
            if (lane == 0) mbar_arrive_expect_tx(bar(B_QFULL), (uint32_t)(4 * rows_used * 128));
            __syncwarp();
            if (lane < 4)  // (tile, half)
                tma_load_3d(base + kPuQ + lane * kPuHT, &qmap, bar(B_QFULL), (lane & 1) * 64, x.kvh * p.G,
                            x.r0 + x.t0 + (lane >> 1) * p.tq, pol_q);
            qph ^= 1;
            const int32_t* bt = p.block_table + (size_t)x.s * p.bt_stride;
            for (int j = 0; j < x.T; ++j) {
                const int rem = x.kv_end - j * kPuTok;
                const int npg = min(PPS, (rem + PAGE - 1) / PAGE);
                int pg = -1;
                if (op_on && op_page < npg) pg = __ldg(bt + j * PPS + op_page);
                const uint32_t bytes = (uint32_t)(npg * PAGE * D * 2);
                mbar_wait(bar(B_KEMPTY0 + slot), kvph ^ 1);
                if (lane == 0) mbar_arrive_expect_tx(bar(B_KFULL0 + slot), bytes);
                __syncwarp();
                if (pg >= 0 && !op_isv)
                    tma_load_4d(base + kPuK + (slot * 2 + op_half) * kPuHT + op_page * (PAGE * 128), &kmap,
                                bar(B_KFULL0 + slot), op_half * 64, 0, x.kvh, pg, pol_kv);
                mbar_wait(bar(B_VEMPTY0 + slot), kvph ^ 1);
                if (lane == 0) mbar_arrive_expect_tx(bar(B_VFULL0 + slot), bytes);
                __syncwarp();
                if (pg >= 0 && op_isv)
                    tma_load_4d(base + kPuV + (slot * 2 + op_half) * kPuHT + op_page * (PAGE * 128), &vmap,
                                bar(B_VFULL0 + slot), op_half * 64, 0, x.kvh, pg, pol_kv);
                slot ^= 1;
                if (slot == 0) kvph ^= 1;
            }
        }
    } else if (warp == 1) {
        // =============================== MMA ISSUER ===============================
        const uint32_t idesc_qk = umma_idesc_bf16(128, 128, 0, 0);
        const uint32_t idesc_pv = umma_idesc_bf16(128, 128, 0, 1);
        uint32_t qph = 0, kph = 0, vph = 0, pph[2] = {0, 0}, oeph = 0;
        int ks = 0, vs = 0;
        auto issue_qk = [&](int t, int kslot) {
            if (lane == 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const uint64_t a = umma_desc_kmajor_sw128(base + kPuQ + (t * 2 + (k >> 2)) * kPuHT + (k & 3) * 32);
                    const uint64_t b = umma_desc_kmajor_sw128(base + kPuK + (kslot * 2 + (k >> 2)) * kPuHT + (k & 3) * 32);
                    umma_ss(tmem + t * 128, a, b, idesc_qk, k > 0);
                }
                umma_commit(bar(B_SFULL0 + t));
            }
        };
        auto issue_pv = [&](int t, int vslot, bool acc) {
            if (lane == 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const uint64_t b = umma_desc_mnmajor_sw128(base + kPuV + vslot * 2 * kPuHT + k * 16 * 128, kPuHT);
                    umma_ts(tmem + 256 + t * 128, tmem + t * 128 + k * 8, b, idesc_pv, (acc || k > 0) ? 1u : 0u);
                }
            }
        };
        for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
            const PuUnit x = pu_unit(p, u);
            if (!x.valid) continue;
            const int T = x.T;
            mbar_wait(bar(B_QFULL), qph);
            qph ^= 1;
            mbar_wait(bar(B_KFULL0 + ks), kph);
            tc_fence_after();
            issue_qk(0, ks);
            issue_qk(1, ks);
            if (lane == 0) {
                umma_commit(bar(B_KEMPTY0 + ks));
                if (T == 1) umma_commit(bar(B_QEMPTY));
            }
            ks ^= 1;
            if (ks == 0) kph ^= 1;
            for (int j = 0; j < T; ++j) {
                mbar_wait(bar(B_VFULL0 + vs), vph);
                if (j == T - 1) {
                    // rows of the last V stage that hold no visible token (not loaded, or NaN poison) -> 0,
                    // so that p = 0 there cannot produce 0 * NaN inside the MMA
                    const int nvalid = x.kv_end - j * kPuTok;
                    if (nvalid < kPuTok) {
                        uint8_t* vg = gbase + kPuV + vs * 2 * kPuHT;
                        for (int i = nvalid * 8 + lane; i < kPuTok * 8; i += 32) {  // 16-B chunks of 128-B rows
                            *reinterpret_cast<int4*>(vg + i * 16) = make_int4(0, 0, 0, 0);
                            *reinterpret_cast<int4*>(vg + kPuHT + i * 16) = make_int4(0, 0, 0, 0);
                        }
                        fence_proxy_async_smem();
                        __syncwarp();
                    }
                }
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    if (j == 0) mbar_wait(bar(B_OEMPTY0 + t), oeph ^ 1);
                    mbar_wait(bar(B_PFULL0 + t), pph[t]);
                    pph[t] ^= 1;
                    tc_fence_after();
                    issue_pv(t, vs, j > 0);
                    if (lane == 0) {
                        if (t == 1) umma_commit(bar(B_VEMPTY0 + vs));
                        if (j == T - 1) umma_commit(bar(B_OFULL0 + t));
                    }
                    if (j + 1 < T) {
                        if (t == 0) {
                            mbar_wait(bar(B_KFULL0 + ks), kph);
                            tc_fence_after();
                        }
                        issue_qk(t, ks);
                        if (t == 1 && lane == 0) {
                            umma_commit(bar(B_KEMPTY0 + ks));
                            if (j + 1 == T - 1) umma_commit(bar(B_QEMPTY));
                        }
                    }
                }
                if (j + 1 < T) {
                    ks ^= 1;
                    if (ks == 0) kph ^= 1;
                }
                vs ^= 1;
                if (vs == 0) vph ^= 1;
            }
            oeph ^= 1;
        }
    } else if (warp >= 4) {
        // =============================== SOFTMAX / EPILOGUE WARPGROUPS ===============================
        const int t = (warp - 4) >> 2;            // Q tile of this warpgroup
        const int row = ((warp & 3) << 5) | lane;  // TMEM lane = Q tile row
        const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t s_addr = tmem + lane_addr + t * 128;
        const uint32_t o_addr = tmem + lane_addr + 256 + t * 128;
        const int tok_l = row / p.G, head_l = row - tok_l * p.G;
        const float c = p.scale_log2;
        uint32_t sph = 0, oph = 0;
        for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
            const PuUnit x = pu_unit(p, u);
            if (!x.valid) continue;
            const int tok = x.t0 + t * p.tq + tok_l;  // query token within the sequence
            const bool row_ok = row < rows_used && tok < x.n;
            // last visible KV position of this row (rows that are not stored follow the unit bound)
            const int lim = min(p.causal ? x.P + tok : x.L - 1, x.kv_end - 1);
            float m_ref = -INFINITY, l = 0.f;
            for (int j = 0; j < x.T; ++j) {
                const int j0 = j * kPuTok;
                const bool need_mask = j0 + kPuTok - 1 > lim;
                mbar_wait(bar(B_SFULL0 + t), sph);
                sph ^= 1;
                tc_fence_after();
                // ---- pass 1: row max
                float mx = -INFINITY;
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) {
                    uint32_t r[32];
                    tmem_ld_32x32b_x32(s_addr + cb * 32, r);
                    tmem_wait_ld();
                    if (need_mask) {
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (j0 + cb * 32 + i > lim) r[i] = 0xff800000u;  // -inf
                    }
#pragma unroll
                    for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(r[i]));
                }
                // ---- running max with lazy rescale of O (TMEM) and l
                if (j == 0) {
                    m_ref = mx;
                } else {
                    const float m_new = fmaxf(m_ref, mx);
                    const bool need = (m_new - m_ref) * c > kPuTau;
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = fast_exp2((m_ref - m_new) * c);
                        l *= alpha;
                        m_ref = m_new;
#pragma unroll
                        for (int cb = 0; cb < 4; ++cb) {
                            uint32_t r[32];
                            tmem_ld_32x32b_x32(o_addr + cb * 32, r);
                            tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * alpha);
                            tmem_st_32x32b_x32(o_addr + cb * 32, r);
                        }
                        tmem_wait_st();
                    }
                }
                // ---- pass 2: p = 2^(s*c - m_ref*c), row sum, P -> bf16 -> TMEM (over the columns of S)
                const float mc = m_ref * c;
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) {
                    uint32_t r[32];
                    tmem_ld_32x32b_x32(s_addr + cb * 32, r);
                    tmem_wait_ld();
                    uint32_t pk[16];
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        float p0 = fast_exp2(__uint_as_float(r[i]) * c - mc);
                        float p1 = fast_exp2(__uint_as_float(r[i + 1]) * c - mc);
                        if (need_mask) {
                            if (j0 + cb * 32 + i > lim) p0 = 0.f;
                            if (j0 + cb * 32 + i + 1 > lim) p1 = 0.f;
                        }
                        l += p0 + p1;
                        pk[i >> 1] = pack_bf16x2(p0, p1);
                    }
                    tmem_st_32x32b_x16(s_addr + cb * 16, pk);
                }
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_PFULL0 + t));
            }
            // ---- epilogue: O / l -> out
            mbar_wait(bar(B_OFULL0 + t), oph);
            oph ^= 1;
            tc_fence_after();
            const float inv = 1.f / l;
            const size_t orow = ((size_t)(x.r0 + tok) * p.Hq + (size_t)x.kvh * p.G + head_l) * D;
#pragma unroll
            for (int cb = 0; cb < 4; ++cb) {
                uint32_t r[32];
                tmem_ld_32x32b_x32(o_addr + cb * 32, r);
                tmem_wait_ld();
                if (row_ok) {
                    if (p.out_f32) {
                        float* o = reinterpret_cast<float*>(p.out) + orow + cb * 32;
#pragma unroll
                        for (int i = 0; i < 32; i += 4)
                            *reinterpret_cast<float4*>(o + i) =
                                make_float4(__uint_as_float(r[i]) * inv, __uint_as_float(r[i + 1]) * inv,
                                            __uint_as_float(r[i + 2]) * inv, __uint_as_float(r[i + 3]) * inv);
                    } else {
                        uint16_t* o = reinterpret_cast<uint16_t*>(p.out) + orow + cb * 32;
#pragma unroll
                        for (int i = 0; i < 32; i += 8) {
                            int4 v;
                            v.x = (int)pack_bf16x2(__uint_as_float(r[i]) * inv, __uint_as_float(r[i + 1]) * inv);
                            v.y = (int)pack_bf16x2(__uint_as_float(r[i + 2]) * inv, __uint_as_float(r[i + 3]) * inv);
                            v.z = (int)pack_bf16x2(__uint_as_float(r[i + 4]) * inv, __uint_as_float(r[i + 5]) * inv);
                            v.w = (int)pack_bf16x2(__uint_as_float(r[i + 6]) * inv, __uint_as_float(r[i + 7]) * inv);
                            *reinterpret_cast<int4*>(o + i) = v;
                        }
                    }
                }
            }
            if (row_ok && p.lse)
                p.lse[(size_t)(x.r0 + tok) * p.Hq + (size_t)x.kvh * p.G + head_l] =
                    (m_ref * c + log2f(l)) * 0.6931471805599453f;
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_OEMPTY0 + t));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, 512);
}

int launch_prefill_umma(const PoolMaps& maps, const void* q, int32_t total_q, const int32_t* cu_seqlens_q,
                        const int32_t* block_table, int64_t bt_stride, const int32_t* seq_lens, int32_t S,
                        int32_t Hq, int32_t Hkv, int32_t page_size, int32_t max_q_len, float scale, int32_t causal,
                        void* out, float* lse, int32_t out_f32, cudaStream_t stream) {
    PrefillUmmaParams p{};
    p.cu_seqlens_q = cu_seqlens_q;
    p.block_table = block_table;
    p.bt_stride = bt_stride;
    p.seq_lens = seq_lens;
    p.S = S;
    p.Hq = Hq;
    p.Hkv = Hkv;
    p.G = Hq / Hkv;
    p.tq = 128 / p.G;
    p.nqb = (max_q_len + 2 * p.tq - 1) / (2 * p.tq);
    p.scale_log2 = scale * 1.4426950408889634f;
    p.out = out;
    p.lse = lse;
    p.out_f32 = out_f32;
    p.causal = causal;
    // Q view: dims (D, Hq, total_q); box (64, G, tq): rows of a tile = token * G + head
    CUtensorMap qmap;
    {
        typedef CUresult (*Fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                               const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                               CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void* fp = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess) {
            (void)cudaGetLastError();
            return MSTAR_ERR_CUDA;
        }
        cuuint64_t dims[3] = {128, (cuuint64_t)Hq, (cuuint64_t)total_q};
        cuuint64_t strides[2] = {256, (cuuint64_t)Hq * 256};
        cuuint32_t box[3] = {64, (cuuint32_t)p.G, (cuuint32_t)p.tq};
        cuuint32_t es[3] = {1, 1, 1};
        if (reinterpret_cast<Fn>(fp)(&qmap, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), dims, strides,
                                     box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return MSTAR_ERR_INVALID_ARG;
    }
    const int64_t units = (int64_t)p.nqb * S * Hkv;
    if (units > 0x7fffffffLL) return MSTAR_ERR_UNSUPPORTED;
    int grid = device_sm_count();
    if (grid > units) grid = (int)units;
    auto k16 = prefill_umma_kernel<16>;
    auto k32 = prefill_umma_kernel<32>;
    static bool attr_set = false;
    if (!attr_set) {
        MSTAR_CUDA_OK(cudaFuncSetAttribute(k16, cudaFuncAttributeMaxDynamicSharedMemorySize, kPuSmemBytes));
        MSTAR_CUDA_OK(cudaFuncSetAttribute(k32, cudaFuncAttributeMaxDynamicSharedMemorySize, kPuSmemBytes));
        attr_set = true;
    }
    if (page_size == 16)
        k16<<<grid, kPuThreads, kPuSmemBytes, stream>>>(qmap, maps.k, maps.v, p);
    else
        k32<<<grid, kPuThreads, kPuSmemBytes, stream>>>(qmap, maps.k, maps.v, p);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}

}  // namespace mstar
