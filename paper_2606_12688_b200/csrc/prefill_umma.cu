// prefill_umma.cu -- step a4 on the 5th-generation tensor cores: paged prefill attention, causal over a
// cached prefix, with tcgen05.mma, accumulators in TMEM and TMA-fed operand tiles (head_dim 128).
//
// Design.  Two launches per call:
//   prefill_plan_kernel   one CTA: the device-side attention plan (where the plan is built on
//                         the CPU).  Enumerates the work units of the batch, counting-sorts them by cost
//                         (KV stages), heaviest first, writes one 32-byte descriptor per unit and zeroes the
//                         work counter.
//   prefill_umma_kernel   persistent CTAs (one per SM), 12 warps, units pulled from the plan with an atomic
//                         counter (longest-processing-time-first, so the tail is one light unit):
//     warp 8      TMA producer + scheduler: Q tiles (3-D boxes over [token][head][d]) and 128-token K / V stages
//                 gathered page by page through the block table (4-D boxes, 128-B swizzle), double-buffered;
//     warp 9      MMA issuer (one elected lane): S = Q K^T (operands in shared memory) and O += P V (P read from
//                 TMEM, V MN-major from shared memory), M = 128, N = 128, K = 16 per instruction;
//     warps 0-3   softmax warpgroup of Q tile A, warps 4-7 of Q tile B: thread = query row = TMEM lane.  The
//                 whole S row is pulled into registers once (tcgen05.ld), masked on diagonal stages only,
//                 3-input max, packed f32x2 scale/subtract, ex2, bf16 pack, tcgen05.st over the columns S
//                 occupied, handed to the MMA warp in two 64-column halves so P V starts while the second half
//                 is still in the SFU; row sums are taken after the hand-off.  O is rescaled in TMEM only when
//                 the running max grows by more than 2^8 (lazy rescale); epilogue O / l -> bf16 -> global.
//   setmaxnreg moves registers from warps 8-11 (88) to the softmax warpgroups (208).
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
constexpr int kPuThreads = 384;   // 12 warps: 0-7 softmax, 8 TMA, 9 MMA (10, 11 only hand their registers over)
// The warp scheduler of an SM sub-partition favours the highest warp id among its eligible warps (measured), so
// the two latency-critical single-lane roles sit above the issue-heavy softmax warps that share their schedulers.
constexpr int kPuTmaWarp = 8;
constexpr int kPuMmaWarp = 9;
constexpr int kPuHT = 128 * 128;  // bytes of a half tile: 128 rows x 64 bf16, 128-B swizzled
constexpr int kPuSplit = 96;      // keys of a stage in the first P hand-off (the second carries the rest)
constexpr float kPuTau = 8.0f;    // lazy-rescale threshold, log2 units
constexpr int kPlanBuckets = 1024;
constexpr int kPlanHeaderInts = 8;  // [0] work counter  [1] CTAs done  [2] number of units

// One work unit, as the plan kernel writes it and every role reads it (32 bytes).
struct PuDesc {
    int s;       // sequence
    int kvh;     // kv head
    int t0;      // first query token of the unit within the sequence
    int n;       // query tokens of the sequence
    int P;       // cached prefix of the sequence (seq_len - n)
    int r0;      // first global query row of the sequence
    int kv_end;  // KV positions [0, kv_end) are visible to at least one row of the unit
    int T;       // KV stages of 128 tokens; 0 terminates
};

struct PrefillUmmaParams {
    const int32_t* block_table;
    int64_t bt_stride;
    int32_t* plan;
    int32_t Hq, G;
    int32_t tq;  // query tokens per Q tile = floor(128 / G)
    float scale_log2;
    void* out;
    float* lse;
    int32_t out_f32;
    int32_t causal;
};


// ------------------------------------------------------------------------------------------------ plan
__global__ void __launch_bounds__(kPlanBuckets)
prefill_plan_kernel(const int32_t* __restrict__ cu_seqlens_q, const int32_t* __restrict__ seq_lens, int S, int Hkv,
                    int tq, int nqb, int causal, int32_t* __restrict__ plan) {
    __shared__ int hist[kPlanBuckets];
    __shared__ int scan[kPlanBuckets];
    const int tid = threadIdx.x;
    // let the attention grid start its prologue now; it waits (griddepcontrol.wait) for this grid to finish
    asm volatile("griddepcontrol.launch_dependents;");
    hist[tid] = 0;
    __syncthreads();
    const int64_t total = (int64_t)nqb * S;
    auto unit_of = [&](int64_t i, PuDesc& d) -> bool {
        d.s = (int)(i % S);
        const int qb = (int)(i / S);
        d.r0 = __ldg(cu_seqlens_q + d.s);
        d.n = __ldg(cu_seqlens_q + d.s + 1) - d.r0;
        d.t0 = qb * 2 * tq;
        if (d.t0 >= d.n) return false;
        const int L = __ldg(seq_lens + d.s);
        d.P = L - d.n;
        const int rows_tok = min(2 * tq, d.n - d.t0);
        d.kv_end = causal ? d.P + d.t0 + rows_tok : L;
        d.T = (d.kv_end + kPuTok - 1) / kPuTok;
        return d.T > 0;
    };
    for (int64_t i = tid; i < total; i += kPlanBuckets) {
        PuDesc d;
        if (unit_of(i, d)) atomicAdd(&hist[min(d.T, kPlanBuckets - 1)], Hkv);
    }
    __syncthreads();
    // suffix sums (heaviest bucket first in the list): thread tid owns bucket b = last - tid, so an inclusive PREFIX
    // scan over tid is the sum over the buckets >= b; warp shuffles + one pass over the 32 warp totals (the
    // log-step scan through shared memory cost 20 block barriers, a third of this kernel's time)
    const int b = kPlanBuckets - 1 - tid, lane = tid & 31, wrp = tid >> 5;
    const int mine = hist[b];
    int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) scan[wrp] = incl;
    __syncthreads();
    if (wrp == 0) {
        const int w = scan[lane];
        int wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        scan[32 + lane] = wi - w;      // exclusive offset of warp `lane`
        if (lane == 31) scan[64] = wi;  // all units
    }
    __syncthreads();
    const int num_units = scan[64];
    hist[b] = incl + scan[32 + wrp] - mine;  // cursor: first list position of bucket b
    __syncthreads();
    PuDesc* list = reinterpret_cast<PuDesc*>(plan + kPlanHeaderInts);
    for (int64_t i = tid; i < total; i += kPlanBuckets) {
        PuDesc d;
        if (unit_of(i, d)) {
            const int pos = atomicAdd(&hist[min(d.T, kPlanBuckets - 1)], Hkv);
            for (int h = 0; h < Hkv; ++h) {
                d.kvh = h;
                int4* dst = reinterpret_cast<int4*>(list + pos + h);
                dst[0] = make_int4(d.s, d.kvh, d.t0, d.n);
                dst[1] = make_int4(d.P, d.r0, d.kv_end, d.T);
            }
        }
    }
    if (tid == 0) {
        plan[0] = 0;
        plan[1] = 0;
        plan[2] = num_units;
    }
}

// shared memory map (offsets from the 1024-aligned base)
constexpr int kPuQ = 0;                     // 2 tiles x 2 halves
constexpr int kPuK = 4 * kPuHT;             // 2 stages x 2 halves
constexpr int kPuV = 8 * kPuHT;             // 2 stages x 2 halves
constexpr int kPuO = 12 * kPuHT;            // 2 tiles x one 64-column half of the bf16 output (TMA-store staging)
constexpr int kPuBars = 14 * kPuHT;         // barriers
enum { B_QFULL0 = 0, B_QFULL1, B_QEMPTY0, B_QEMPTY1, B_KFULL0, B_KFULL1, B_KEMPTY0, B_KEMPTY1, B_VFULL0, B_VFULL1,
       B_VEMPTY0, B_VEMPTY1, B_SFULL0, B_SFULL1, B_PFULL00, B_PFULL01, B_PFULL10, B_PFULL11, B_OFULL0, B_OFULL1,
       B_OEMPTY0, B_OEMPTY1, B_UFULL0, B_UFULL1, B_UEMPTY0, B_UEMPTY1, B_QCONV0, B_QCONV1, B_COUNT };
constexpr int kPuDesc = kPuBars + 256;      // 2 unit descriptors (32 B each)
constexpr int kPuTmemSlot = kPuDesc + 64;
constexpr int kPuSmemBytes = 14 * kPuHT + 512 + 1024;
static_assert(B_COUNT * 8 <= 256, "barrier area");

// packed fp32x2 helpers (FFMA2 / FADD2 on sm_100) and the 3-input max (FMNMX3)
__device__ __forceinline__ void ffma2_bcast(float& d0, float& d1, float a0, float a1, float b, float c) {
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\t"
        "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %4};\n\tmov.b64 rc, {%5, %5};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d0), "=f"(d1)
        : "f"(a0), "f"(a1), "f"(b), "f"(c));
}
__device__ __forceinline__ void fadd2(float& d0, float& d1, float a0, float a1, float b0, float b1) {
    asm("{\n\t.reg .b64 ra, rb, rd;\n\t"
        "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
        "add.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d0), "=f"(d1)
        : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

__device__ __forceinline__ PuDesc pu_read_desc(const uint8_t* gbase, int uslot) {
    const int4* src = reinterpret_cast<const int4*>(gbase + kPuDesc + uslot * 32);
    const int4 a = src[0], b = src[1];
    PuDesc d;
    d.s = a.x; d.kvh = a.y; d.t0 = a.z; d.n = a.w;
    d.P = b.x; d.r0 = b.y; d.kv_end = b.z; d.T = b.w;
    return d;
}

// F16 (mstar_paged_attn_prefill_fp8): the pool tiles hold fp16 instead of bf16 (the dequantised E4M3 scratch pool).
// Both operands of a kind::f16 MMA must have one format (a bf16 x f16 instruction raises an illegal-instruction
// fault, measured), so warps 10 and 11 -- idle in the bf16 kernel -- convert the Q tiles of every unit from bf16 to
// fp16 in shared memory as soon as they land (exact for |q| in [2^-14, 65504]) and hand them to the MMA warp, and P
// is rounded to fp16: Q K^T and P V are f16 x f16 MMAs.
// D = head_dim, 128 or 64.  head_dim 64 uses the first 64-column half of every Q / K / V tile and staging buffer and
// the first 64 TMEM columns of each O accumulator (Q K^T contracts over 4 instead of 8 k-steps, P V has N = 64); the
// shared-memory and TMEM maps stay those of head_dim 128.
template <int PAGE, bool F16, int D = 128>
__global__ void __launch_bounds__(kPuThreads, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap qmap, const __grid_constant__ CUtensorMap kmap,
                    const __grid_constant__ CUtensorMap vmap, const __grid_constant__ CUtensorMap omap,
                    const PrefillUmmaParams p) {
    static_assert(D == 128 || D == 64, "head_dim");
    constexpr int NH = D / 64;          // 64-column half tiles per row
    constexpr int PPS = kPuTok / PAGE;  // pages per stage
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t bars = base + kPuBars;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(gbase + kPuTmemSlot);
    auto bar = [&](int i) { return bars + 8u * i; };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar(B_QFULL0 + i), 1);
            mbar_init(bar(B_QEMPTY0 + i), 1);
            mbar_init(bar(B_KFULL0 + i), 1);
            mbar_init(bar(B_KEMPTY0 + i), 1);
            mbar_init(bar(B_VFULL0 + i), 1);
            mbar_init(bar(B_VEMPTY0 + i), 1);
            mbar_init(bar(B_SFULL0 + i), 1);
            mbar_init(bar(B_PFULL00 + 2 * i), 4);
            mbar_init(bar(B_PFULL00 + 2 * i + 1), 4);
            mbar_init(bar(B_OFULL0 + i), 1);
            mbar_init(bar(B_OEMPTY0 + i), 4);
            mbar_init(bar(B_UFULL0 + i), 1);
            mbar_init(bar(B_UEMPTY0 + i), F16 ? 11 : 9);  // MMA warp + 8 softmax warps (+ 2 Q converters)
            mbar_init(bar(B_QCONV0 + i), 1);
        }
        fence_mbar_init();
    }
    if (warp == kPuMmaWarp) {
        tmem_alloc(smem_u32(tmem_slot), 512);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int rows_used = p.tq * p.G;  // rows of a Q tile that carry (token, head) pairs

    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
        if (warp == kPuTmaWarp) {
            // =============================== TMA PRODUCER + SCHEDULER ===============================
            prefetch_tensormap(&qmap);
            prefetch_tensormap(&kmap);
            prefetch_tensormap(&vmap);
            // Programmatic dependent launch: everything above (barriers, TMEM, descriptor prefetch) overlapped the
            // tail of the previous grid in the stream (the plan kernel, or the K/V append); every read and write
            // of global memory in this kernel happens after this warp has seen that grid complete, because all
            // other roles only start on barriers this warp's loads complete.
            asm volatile("griddepcontrol.wait;" ::: "memory");
            const uint64_t pol_kv = policy_evict_last();   // K/V re-read by other query blocks of the sequence
            const uint64_t pol_q = policy_evict_first();
            // lane -> (K or V, page, half): PPS*2 ops for K on the low lanes, PPS*2 for V after them
            constexpr int OPS1 = PPS * NH;
            const int op_isv = lane / OPS1;
            const int op_page = (lane % OPS1) / NH;
            const int op_half = lane % NH;
            const bool op_on = lane < 2 * OPS1;
            const PuDesc* list = reinterpret_cast<const PuDesc*>(p.plan + kPlanHeaderInts);
            // Lane 0 owns the scheduler state.  Fetches are pipelined two units deep: the atomic for unit
            // u+2 and the descriptor load for unit u+1 are in flight while unit u's tiles are issued.  The first
            // two units of a CTA are fixed (list is sorted heaviest first): rank b and rank 2*grid-1-b, so the
            // CTA that got the heaviest unit of the first round gets the lightest of the second; everything
            // after comes from the shared counter.
            int num_units = 0, idx1 = 0;
            int4 da = make_int4(0, 0, 0, 0), db = make_int4(0, 0, 0, 0);
            if (lane == 0) {
                num_units = *reinterpret_cast<volatile int32_t*>(p.plan + 2);
                const int idx0 = (int)blockIdx.x;
                idx1 = 2 * (int)gridDim.x - 1 - (int)blockIdx.x;
                if (idx0 < num_units) {
                    const int4* e = reinterpret_cast<const int4*>(list + idx0);
                    da = __ldg(e);
                    db = __ldg(e + 1);
                }
            }
            uint32_t qph[2] = {0, 0}, kvph = 0, uph = 0;
            int slot = 0, uslot = 0;
            while (true) {
                mbar_wait(bar(B_UEMPTY0 + uslot), uph ^ 1);
                if (lane == 0) {
                    int4* dst = reinterpret_cast<int4*>(gbase + kPuDesc + uslot * 32);
                    dst[0] = da;
                    dst[1] = db;
                    mbar_arrive(bar(B_UFULL0 + uslot));
                }
                __syncwarp();
                const PuDesc x = pu_read_desc(gbase, uslot);
                uslot ^= 1;
                if (uslot == 0) uph ^= 1;
                if (x.T == 0) break;
                int idx2 = 0;
                int4 na = make_int4(0, 0, 0, 0), nb = make_int4(0, 0, 0, 0);
                if (lane == 0) {
                    idx2 = 2 * (int)gridDim.x + atomicAdd(p.plan, 1);
                    if (idx1 < num_units) {
                        const int4* e = reinterpret_cast<const int4*>(list + idx1);
                        na = __ldg(e);
                        nb = __ldg(e + 1);
                    }
                }
                const int32_t* bt = p.block_table + (size_t)x.s * p.bt_stride;
                int pg_next = -1;
                {
                    const int npg0 = min(PPS, (x.kv_end + PAGE - 1) / PAGE);
                    if (op_on && op_page < npg0) pg_next = __ldg(bt + op_page);
                }
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    mbar_wait(bar(B_QEMPTY0 + t), qph[t] ^ 1);
                    qph[t] ^= 1;
                    if (lane == 0) mbar_arrive_expect_tx(bar(B_QFULL0 + t), (uint32_t)(NH * rows_used * 128));
                    __syncwarp();
                    if (lane < NH)  // half
                        tma_load_3d(base + kPuQ + (t * 2 + lane) * kPuHT, &qmap, bar(B_QFULL0 + t), lane * 64,
                                    x.kvh * p.G, x.r0 + x.t0 + t * p.tq, pol_q);
                }
                for (int j = 0; j < x.T; ++j) {
                    const int rem = x.kv_end - j * kPuTok;
                    const int npg = min(PPS, (rem + PAGE - 1) / PAGE);
                    const int pg = pg_next;
                    pg_next = -1;
                    if (j + 1 < x.T) {  // block-table entries of the next stage, one stage ahead
                        const int npg1 = min(PPS, (rem - kPuTok + PAGE - 1) / PAGE);
                        if (op_on && op_page < npg1) pg_next = __ldg(bt + (j + 1) * PPS + op_page);
                    }
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
                da = na;
                db = nb;
                idx1 = idx2;
            }
            // Every fetch of this CTA has returned.  The last CTA out re-arms the plan (counter = 0), so the
            // same plan serves the next launch (MSTAR_FLAG_PREFILL_REUSE_PLAN).
            if (lane == 0) {
                asm volatile("" ::"r"(idx1));
                __threadfence();
                const int done = atomicAdd(p.plan + 1, 1);
                if (done == (int)gridDim.x - 1) {
                    p.plan[0] = 0;
                    p.plan[1] = 0;
                }
            }
        } else if (warp == kPuMmaWarp) {
            // =============================== MMA ISSUER ===============================
            const uint32_t fmt = F16 ? 0u : 1u;  // operand format of Q, K, P and V
            const uint32_t idesc_qk = umma_idesc_f16(128, 128, fmt, fmt, 0, 0);
            const uint32_t idesc_pv = umma_idesc_f16(128, D, fmt, fmt, 0, 1);
            uint32_t qph[2] = {0, 0}, kph = 0, vph = 0, pph[2] = {0, 0}, oeph = 0, uph = 0;
            int ks = 0, vs = 0, uslot = 0;
            // Descriptors differ only in the 14-bit start-address field (bytes >> 4) of their low word: the bases are
            // built once, the per-instruction offsets are compile-time constants.
            const uint64_t dq = umma_desc_kmajor_sw128(base + kPuQ);
            const uint64_t dk = umma_desc_kmajor_sw128(base + kPuK);
            const uint64_t dv = umma_desc_mnmajor_sw128(base + kPuV, kPuHT);
            auto issue_qk = [&](int t, int kslot) {
                if (elect_one()) {
                    const uint64_t a0 = dq + (uint64_t)(t * 2 * (kPuHT >> 4));
                    const uint64_t b0 = dk + (uint64_t)(kslot * 2 * (kPuHT >> 4));
#pragma unroll
                    for (int k = 0; k < D / 16; ++k) {
                        const uint32_t off = (uint32_t)((k >> 2) * (kPuHT >> 4) + (k & 3) * 2);
                        umma_ss(tmem + t * 128, a0 + off, b0 + off, idesc_qk, k > 0);
                    }
                    umma_commit(bar(B_SFULL0 + t));
                }
                __syncwarp();
            };
            auto issue_pv = [&](int t, int vslot, bool acc, bool second) {
                if (elect_one()) {
                    const uint64_t b0 = dv + (uint64_t)(vslot * 2 * (kPuHT >> 4));
                    const int kbeg = second ? kPuSplit / 16 : 0, kend = second ? 8 : kPuSplit / 16;
#pragma unroll
                    for (int k = kbeg; k < kend; ++k)
                        umma_ts(tmem + 256 + t * 128, tmem + t * 128 + k * 8, b0 + (uint64_t)(k * 16 * 128 >> 4), idesc_pv,
                                (acc || k > 0) ? 1u : 0u);
                }
                __syncwarp();
            };
            auto commit_if = [&](bool cond, int b) {
                if (cond && elect_one()) umma_commit(bar(b));
                __syncwarp();
            };
            while (true) {
                mbar_wait(bar(B_UFULL0 + uslot), uph);
                const PuDesc x = pu_read_desc(gbase, uslot);
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_UEMPTY0 + uslot));
                uslot ^= 1;
                if (uslot == 0) uph ^= 1;
                if (x.T == 0) break;
                const int T = x.T;
                mbar_wait(bar(B_KFULL0 + ks), kph);
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    mbar_wait(bar((F16 ? B_QCONV0 : B_QFULL0) + t), qph[t]);
                    qph[t] ^= 1;
                    tc_fence_after();
                    issue_qk(t, ks);
                    commit_if(T == 1, B_QEMPTY0 + t);
                }
                commit_if(true, B_KEMPTY0 + ks);
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
                                if (NH == 2) *reinterpret_cast<int4*>(vg + kPuHT + i * 16) = make_int4(0, 0, 0, 0);
                            }
                            fence_proxy_async_smem();
                            __syncwarp();
                        }
                    }
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        if (j == 0) mbar_wait(bar(B_OEMPTY0 + t), oeph ^ 1);
                        mbar_wait(bar(B_PFULL00 + 2 * t), pph[t]);
                        tc_fence_after();
                        issue_pv(t, vs, j > 0, false);
                        // the next K stage landed long ago: checked here, off the chain that follows the last hand-off
                        if (t == 0 && j + 1 < T) mbar_wait(bar(B_KFULL0 + ks), kph);
                        mbar_wait(bar(B_PFULL00 + 2 * t + 1), pph[t]);
                        pph[t] ^= 1;
                        tc_fence_after();
                        // one elected region for everything behind the last hand-off: the rest of P V, its commits,
                        // the next Q K^T and its commits (each elect / __syncwarp pair sits on the per-tile chain)
                        if (elect_one()) {
                            const uint64_t bv = dv + (uint64_t)(vs * 2 * (kPuHT >> 4));
#pragma unroll
                            for (int k = kPuSplit / 16; k < 8; ++k)
                                umma_ts(tmem + 256 + t * 128, tmem + t * 128 + k * 8, bv + (uint64_t)(k * 16 * 128 >> 4),
                                        idesc_pv, 1u);
                            if (t == 1) umma_commit(bar(B_VEMPTY0 + vs));
                            if (j == T - 1) umma_commit(bar(B_OFULL0 + t));
                            if (j + 1 < T) {
                                const uint64_t a0 = dq + (uint64_t)(t * 2 * (kPuHT >> 4));
                                const uint64_t b0 = dk + (uint64_t)(ks * 2 * (kPuHT >> 4));
#pragma unroll
                                for (int k = 0; k < D / 16; ++k) {
                                    const uint32_t off = (uint32_t)((k >> 2) * (kPuHT >> 4) + (k & 3) * 2);
                                    umma_ss(tmem + t * 128, a0 + off, b0 + off, idesc_qk, k > 0);
                                }
                                umma_commit(bar(B_SFULL0 + t));
                                if (j + 1 == T - 1) umma_commit(bar(B_QEMPTY0 + t));
                                if (t == 1) umma_commit(bar(B_KEMPTY0 + ks));
                            }
                        }
                        __syncwarp();
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
        } else if (F16) {
            // =============================== Q CONVERTERS (warps 10, 11; fp16 pool only) ===============================
            // warp 10 + t: Q tile t of every unit, bf16 -> fp16 in place (the conversion is elementwise, so the
            // swizzled layout does not matter), then a fence towards the tensor core's proxy and the hand-over
            const int t = warp - 10;
            uint32_t qph = 0, uph = 0;
            int uslot = 0;
            while (true) {
                mbar_wait(bar(B_UFULL0 + uslot), uph);
                const PuDesc x = pu_read_desc(gbase, uslot);
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_UEMPTY0 + uslot));
                uslot ^= 1;
                if (uslot == 0) uph ^= 1;
                if (x.T == 0) break;
                mbar_wait(bar(B_QFULL0 + t), qph);
                qph ^= 1;
                const uint32_t qt = base + kPuQ + t * 2 * kPuHT;
#pragma unroll 4
                for (int c = lane; c < NH * kPuHT / 16; c += 32) {
                    uint32_t w0, w1, w2, w3;
                    ld_shared_v4(qt + c * 16, w0, w1, w2, w3);
                    st_shared_v4(qt + c * 16, bf16x2_to_f16x2(w0), bf16x2_to_f16x2(w1), bf16x2_to_f16x2(w2),
                                 bf16x2_to_f16x2(w3));
                }
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_QCONV0 + t));
            }
        }
    } else {
        // =============================== SOFTMAX / EPILOGUE WARPGROUPS ===============================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
        const int t = warp >> 2;                   // Q tile of this warpgroup
        const int row = ((warp & 3) << 5) | lane;  // TMEM lane = Q tile row
        const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t s_addr = tmem + lane_addr + t * 128;
        const uint32_t o_addr = tmem + lane_addr + 256 + t * 128;
        const int tok_l = row / p.G, head_l = row - tok_l * p.G;
        const float c = p.scale_log2;
        uint32_t sph = 0, oph = 0, uph = 0;
        int uslot = 0;
        while (true) {
            mbar_wait(bar(B_UFULL0 + uslot), uph);
            const PuDesc x = pu_read_desc(gbase, uslot);
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_UEMPTY0 + uslot));
            uslot ^= 1;
            if (uslot == 0) uph ^= 1;
            if (x.T == 0) break;
            const int tok = x.t0 + t * p.tq + tok_l;  // query token within the sequence
            const bool row_ok = row < rows_used && tok < x.n;
            // last visible KV position of this row (rows that are not stored follow the unit bound)
            const int lim = p.causal ? min(x.P + tok, x.kv_end - 1) : x.kv_end - 1;
            float m_ref = -INFINITY, l = 0.f;
            for (int j = 0; j < x.T; ++j) {
                const int j0 = j * kPuTok;
                mbar_wait(bar(B_SFULL0 + t), sph);
                sph ^= 1;
                tc_fence_after();
                uint32_t r[128];
                if constexpr (F16) {
                    // four 32-column loads: with the converter warps resident, the two 64-column loads of the bf16
                    // instantiation measured 6.5 % slower here (152.6 -> 162.8 us on config 3, A/B on one box)
                    tmem_ld_32x32b_x32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&r[0]));
                    tmem_ld_32x32b_x32(s_addr + 32, *reinterpret_cast<uint32_t(*)[32]>(&r[32]));
                    tmem_ld_32x32b_x32(s_addr + 64, *reinterpret_cast<uint32_t(*)[32]>(&r[64]));
                    tmem_ld_32x32b_x32(s_addr + 96, *reinterpret_cast<uint32_t(*)[32]>(&r[96]));
                    tmem_wait_ld();
                } else {
                    tmem_ld_32x32b_x64(s_addr, *reinterpret_cast<uint32_t(*)[64]>(&r[0]));
                    tmem_ld_32x32b_x64(s_addr + 64, *reinterpret_cast<uint32_t(*)[64]>(&r[64]));
                    tmem_wait_ld();
                }
                // ---- mask (diagonal / last stages only; warp-uniform branch)
                if (__any_sync(0xffffffffu, j0 + kPuTok - 1 > lim)) {
                    const int rel = lim - j0;  // columns i > rel are invisible to this row
#pragma unroll
                    for (int i = 0; i < 128; ++i)
                        if (i > rel) r[i] = 0xff800000u;  // -inf
                }
                // ---- row max (3-input max, four chains)
                float mx0 = fmax3(__uint_as_float(r[0]), __uint_as_float(r[1]), __uint_as_float(r[2]));
                float mx1 = fmax3(__uint_as_float(r[3]), __uint_as_float(r[4]), __uint_as_float(r[5]));
                float mx2 = fmax3(__uint_as_float(r[6]), __uint_as_float(r[7]), __uint_as_float(r[8]));
                float mx3 = fmax3(__uint_as_float(r[9]), __uint_as_float(r[10]), __uint_as_float(r[11]));
#pragma unroll
                for (int i = 12; i < 124; i += 8) {
                    mx0 = fmax3(mx0, __uint_as_float(r[i]), __uint_as_float(r[i + 1]));
                    mx1 = fmax3(mx1, __uint_as_float(r[i + 2]), __uint_as_float(r[i + 3]));
                    mx2 = fmax3(mx2, __uint_as_float(r[i + 4]), __uint_as_float(r[i + 5]));
                    mx3 = fmax3(mx3, __uint_as_float(r[i + 6]), __uint_as_float(r[i + 7]));
                }
                mx0 = fmax3(mx0, __uint_as_float(r[124]), __uint_as_float(r[125]));
                mx1 = fmax3(mx1, __uint_as_float(r[126]), __uint_as_float(r[127]));
                const float mx = fmax3(fmaxf(mx0, mx1), mx2, mx3);
                // ---- running max with lazy rescale of O (TMEM) and l
                if (j == 0) {
                    m_ref = mx;
                } else {
                    const float m_new = fmaxf(m_ref, mx);
                    // only rows that are stored vote: tile rows past rows_used hold whatever the previous kernel
                    // left in shared memory, and a rescale they triggered would change the rounding of the whole
                    // warp from run to run (results must be bit-identical across runs, R20)
                    const bool need = row_ok && (m_new - m_ref) * c > kPuTau;
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = fast_exp2((m_ref - m_new) * c);
                        l *= alpha;
                        m_ref = m_new;
#pragma unroll
                        for (int cb = 0; cb < D / 32; ++cb) {
                            uint32_t o[32];
                            tmem_ld_32x32b_x32(o_addr + cb * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                            tmem_st_32x32b_x32(o_addr + cb * 32, o);
                        }
                        tmem_wait_st();
                    }
                }
                // ---- p = 2^(s*c - m_ref*c), P -> bf16 -> TMEM (over the columns of S), handed over in two parts:
                // the first kPuSplit keys, then the rest, so that little P V work is left after the last hand-off
                const float nmc = -m_ref * c;
                {
                    uint32_t pk[kPuSplit / 2];
#pragma unroll
                    for (int i = 0; i < kPuSplit; i += 2) {
                        float x0, x1;
                        ffma2_bcast(x0, x1, __uint_as_float(r[i]), __uint_as_float(r[i + 1]), c, nmc);
                        const float p0 = fast_exp2(x0), p1 = fast_exp2(x1);
                        r[i] = __float_as_uint(p0);
                        r[i + 1] = __float_as_uint(p1);
                        pk[i >> 1] = F16 ? pack_f16x2(p0, p1) : pack_bf16x2(p0, p1);
                    }
                    tmem_st_32x32b_x32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&pk[0]));
                    tmem_st_32x32b_x16(s_addr + 32, *reinterpret_cast<uint32_t(*)[16]>(&pk[32]));
                    tmem_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_PFULL00 + 2 * t));
                }
                {
                    uint32_t pk[(128 - kPuSplit) / 2];
#pragma unroll
                    for (int i = kPuSplit; i < 128; i += 2) {
                        float x0, x1;
                        ffma2_bcast(x0, x1, __uint_as_float(r[i]), __uint_as_float(r[i + 1]), c, nmc);
                        const float p0 = fast_exp2(x0), p1 = fast_exp2(x1);
                        r[i] = __float_as_uint(p0);
                        r[i + 1] = __float_as_uint(p1);
                        pk[(i - kPuSplit) >> 1] = F16 ? pack_f16x2(p0, p1) : pack_bf16x2(p0, p1);
                    }
                    tmem_st_32x32b_x16(s_addr + kPuSplit / 2, pk);
                    tmem_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_PFULL00 + 2 * t + 1));
                }
                // ---- row sum, after the hand-off (packed adds, four chains)
                float s0 = __uint_as_float(r[0]), s1 = __uint_as_float(r[1]);
                float s2 = __uint_as_float(r[2]), s3 = __uint_as_float(r[3]);
#pragma unroll
                for (int i = 4; i < 128; i += 4) {
                    fadd2(s0, s1, s0, s1, __uint_as_float(r[i]), __uint_as_float(r[i + 1]));
                    fadd2(s2, s3, s2, s3, __uint_as_float(r[i + 2]), __uint_as_float(r[i + 3]));
                }
                l += (s0 + s1) + (s2 + s3);
            }
            // ---- epilogue: O / l -> out
            mbar_wait(bar(B_OFULL0 + t), oph);
            oph ^= 1;
            tc_fence_after();
            const float inv = 1.f / l;
            const size_t orow = ((size_t)(x.r0 + tok) * p.Hq + (size_t)x.kvh * p.G + head_l) * D;
            uint32_t r[D];
            {
#pragma unroll
                for (int cb = 0; cb < D / 32; ++cb)
                    tmem_ld_32x32b_x32(o_addr + cb * 32, *reinterpret_cast<uint32_t(*)[32]>(&r[cb * 32]));
                tmem_wait_ld();
            }
            // O is in registers: the tensor core may start the next unit's P V on this tile
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_OEMPTY0 + t));
            // Full tiles of bf16 output leave through shared memory and one TMA store per 64-column half (the
            // box of the Q load, so rows land at (token, head)); per-thread row stores would be 32 scattered
            // 16-byte writes per instruction.  Ragged tail tiles and the fp32 diagnostic output go direct.
            const bool via_tma = !p.out_f32 && x.t0 + (t + 1) * p.tq <= x.n;
            if (via_tma) {
                const uint32_t obuf = base + kPuO + t * kPuHT;
#pragma unroll
                for (int h = 0; h < NH; ++h) {
                    // the previous store out of this buffer must have finished reading it
                    if ((warp & 3) == 0 && lane == 0) bulk_wait_group_read0();
                    named_bar_sync(1 + t, 128);
                    if (row < rows_used) {
#pragma unroll
                        for (int c8 = 0; c8 < 8; ++c8) {
                            const int i = h * 64 + c8 * 8;
                            st_shared_v4(obuf + swz128(row, c8),
                                         pack_bf16x2(__uint_as_float(r[i]) * inv, __uint_as_float(r[i + 1]) * inv),
                                         pack_bf16x2(__uint_as_float(r[i + 2]) * inv, __uint_as_float(r[i + 3]) * inv),
                                         pack_bf16x2(__uint_as_float(r[i + 4]) * inv, __uint_as_float(r[i + 5]) * inv),
                                         pack_bf16x2(__uint_as_float(r[i + 6]) * inv, __uint_as_float(r[i + 7]) * inv));
                        }
                    }
                    fence_proxy_async_smem();
                    named_bar_sync(1 + t, 128);
                    if ((warp & 3) == 0 && lane == 0) {
                        tma_store_3d(&omap, obuf, h * 64, x.kvh * p.G, x.r0 + x.t0 + t * p.tq);
                        bulk_commit_group();
                    }
                }
            }
            if (row_ok) {
                if (p.out_f32) {
                    float* o = reinterpret_cast<float*>(p.out) + orow;
#pragma unroll
                    for (int i = 0; i < D; i += 4)
                        *reinterpret_cast<float4*>(o + i) =
                            make_float4(__uint_as_float(r[i]) * inv, __uint_as_float(r[i + 1]) * inv,
                                        __uint_as_float(r[i + 2]) * inv, __uint_as_float(r[i + 3]) * inv);
                } else if (!via_tma) {
                    uint16_t* o = reinterpret_cast<uint16_t*>(p.out) + orow;
#pragma unroll
                    for (int i = 0; i < D; i += 8) {
                        int4 v;
                        v.x = (int)pack_bf16x2(__uint_as_float(r[i]) * inv, __uint_as_float(r[i + 1]) * inv);
                        v.y = (int)pack_bf16x2(__uint_as_float(r[i + 2]) * inv, __uint_as_float(r[i + 3]) * inv);
                        v.z = (int)pack_bf16x2(__uint_as_float(r[i + 4]) * inv, __uint_as_float(r[i + 5]) * inv);
                        v.w = (int)pack_bf16x2(__uint_as_float(r[i + 6]) * inv, __uint_as_float(r[i + 7]) * inv);
                        *reinterpret_cast<int4*>(o + i) = v;
                    }
                }
                if (p.lse)
                    p.lse[(size_t)(x.r0 + tok) * p.Hq + (size_t)x.kvh * p.G + head_l] =
                        (m_ref * c + log2f(l)) * 0.6931471805599453f;
            }
        }
    }
    if (warp < 8 && (warp & 3) == 0 && lane == 0) bulk_wait_group0();  // output stores issued by this thread
    tc_fence_before();
    __syncthreads();
    if (warp == kPuMmaWarp) tmem_dealloc(tmem, 512);
}

// 3-D view (D, Hq, total_q) of a [total_q][Hq][128] bf16 tensor with box (64, G, tq) and 128-byte swizzle
static int make_q_view_map(const void* ptr, int32_t total_q, int32_t Hq, int32_t G, int32_t tq, int32_t D,
                           CUtensorMap* out) {
    typedef CUresult (*Fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                           const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                           CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static Fn encode = nullptr;
    if (!encode) {
        void* fp = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess) {
            (void)cudaGetLastError();
            return MSTAR_ERR_CUDA;
        }
        encode = reinterpret_cast<Fn>(fp);
    }
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)total_q};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)Hq * D * 2};
    cuuint32_t box[3] = {64, (cuuint32_t)G, (cuuint32_t)tq};
    cuuint32_t es[3] = {1, 1, 1};
    if (encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return MSTAR_ERR_INVALID_ARG;
    return MSTAR_OK;
}

size_t prefill_umma_workspace_bytes(int32_t num_seqs, int32_t total_q, int32_t num_q_heads) {
    // header + one 32-byte descriptor per unit; units <= (total_q / (2 tq) + S) * Hkv <= total_q*Hq/128 + S*Hq
    const int64_t units = ((int64_t)total_q * num_q_heads + 127) / 128 + (int64_t)num_seqs * num_q_heads + 1;
    return (size_t)(kPlanHeaderInts * 4 + 32 * units);
}

int launch_prefill_umma(const PoolMaps& maps, const void* q, int32_t total_q, const int32_t* cu_seqlens_q,
                        const int32_t* block_table, int64_t bt_stride, const int32_t* seq_lens, int32_t S,
                        int32_t Hq, int32_t Hkv, int32_t page_size, int32_t max_q_len, float scale, int32_t causal,
                        void* out, float* lse, int32_t out_f32, int32_t reuse_plan, void* workspace,
                        size_t workspace_bytes, cudaStream_t stream, int32_t kv_f16, int32_t head_dim) {
    if (head_dim != 128 && !(head_dim == 64 && !kv_f16)) return MSTAR_ERR_UNSUPPORTED;
    PrefillUmmaParams p{};
    p.block_table = block_table;
    p.bt_stride = bt_stride;
    p.plan = reinterpret_cast<int32_t*>(workspace);
    p.Hq = Hq;
    p.G = Hq / Hkv;
    p.tq = 128 / p.G;
    p.scale_log2 = scale * 1.4426950408889634f;
    p.out = out;
    p.lse = lse;
    p.out_f32 = out_f32;
    p.causal = causal;
    const int nqb = (max_q_len + 2 * p.tq - 1) / (2 * p.tq);
    const int64_t max_units = ((int64_t)total_q / (2 * p.tq) + S) * Hkv;
    if (!workspace || !aligned(workspace, 16)) return MSTAR_ERR_INVALID_ARG;
    if (workspace_bytes < (size_t)(kPlanHeaderInts * 4 + 32 * max_units)) return MSTAR_ERR_WORKSPACE_TOO_SMALL;
    if (max_units > 0x7fffffffLL || (int64_t)nqb * S > 0x7fffffffLL) return MSTAR_ERR_UNSUPPORTED;
    // Q view: dims (D, Hq, total_q); box (64, G, tq): rows of a tile = token * G + head
    CUtensorMap qmap;
    {
        const int st = make_q_view_map(q, total_q, Hq, p.G, p.tq, head_dim, &qmap);
        if (st != MSTAR_OK) return st;
    }
    // output view for the TMA-store epilogue: same geometry as the Q view (bf16 output only)
    CUtensorMap omap = qmap;
    if (!out_f32) {
        const int st = make_q_view_map(out, total_q, Hq, p.G, p.tq, head_dim, &omap);
        if (st != MSTAR_OK) return st;
    }
    if (!reuse_plan) {
        prefill_plan_kernel<<<1, kPlanBuckets, 0, stream>>>(cu_seqlens_q, seq_lens, S, Hkv, p.tq, nqb, causal, p.plan);
        MSTAR_CUDA_OK(cudaGetLastError());
        launch_count_add(1);
    }
    int grid = device_sm_count();
    if (grid > max_units) grid = (int)max_units;
    if (grid < 1) grid = 1;
    const bool d64 = head_dim == 64;
    auto k16 = kv_f16 ? prefill_umma_kernel<16, true, 128>
                      : (d64 ? prefill_umma_kernel<16, false, 64> : prefill_umma_kernel<16, false, 128>);
    auto k32 = kv_f16 ? prefill_umma_kernel<32, true, 128>
                      : (d64 ? prefill_umma_kernel<32, false, 64> : prefill_umma_kernel<32, false, 128>);
    static PerDeviceOnce once16, once32, once16h, once32h, once16s, once32s;
    MSTAR_CUDA_OK(set_max_dynamic_smem(kv_f16 ? once16h : (d64 ? once16s : once16), k16, kPuSmemBytes));
    MSTAR_CUDA_OK(set_max_dynamic_smem(kv_f16 ? once32h : (d64 ? once32s : once32), k32, kPuSmemBytes));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kPuThreads);
    cfg.dynamicSmemBytes = kPuSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, page_size == 16 ? k16 : k32, qmap, maps.k, maps.v, omap, p));
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}

}  // namespace mstar

