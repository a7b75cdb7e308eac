// decode.cu -- steps a2 + a3: split-K ("flash-decoding") paged decode attention and its LSE combine.
//
// Design.  The path is an HBM stream: every K/V byte of every sequence is read
// exactly once, 4*G*D flops per 2*D*2 bytes.  One persistent CTA per SM; work items are
// (sequence, split-K partition, kv head).  Inside a CTA
//   * two PRODUCER warps (K half / V half of every stage) walk the block table and issues TMA tensor copies (cp.async.bulk.tensor,
//     128-B swizzle) of whole (page, kv head) slabs into a deep shared-memory ring of 64-token stages,
//     running ahead across work items so the stream never drains between items;
//   * four CONSUMER warps each own 16 tokens of every stage: S = Q K^T with warp-level bf16 MMA
//     (the G grouped query heads padded into the 16 MMA rows; the tensor pipe is otherwise idle),
//     online softmax in fp32 with warp-shuffle max / sum reductions, O += P V with MMA;
//   * at the end of an item the four warps merge their (m, l, O) through shared memory and write one
//     fp32 partial; the combine kernel merges partitions by log-sum-exp and rounds to bf16 once.
// Full/empty mbarriers per stage are the only synchronisation in the steady state.
#include <cuda_bf16.h>

#include <mutex>
#include <type_traits>

#include "host_common.h"
#include "ptx.cuh"

namespace mstar {

// Consumer warps (16 tokens of every ring stage each): 4 for a bf16 pool; 8 for an fp8 pool, where the byte -> bf16
// conversion is ALU work that two warps per scheduler overlap and a 128-token stage has the bytes of a bf16 one.
// With G <= 8 the fp8 consumer (swapped operands, 111 registers) can run 12 warps, three per scheduler: the host
// picks them for long sequences (192-token stages cost short, ragged streams more in tail tiles than they gain).
constexpr int decode_tok(int nw) { return 16 * nw; }            // tokens per ring stage
constexpr int decode_threads(int nw, int nb = 1) { return 32 * (nw * nb + 2); }  // + K and V producer warps
static int decode_pick_warps(bool fp8, int G, int max_seq_len) {
    return fp8 ? ((G <= 8 && max_seq_len > 8192) ? 12 : 8) : 4;
}
constexpr int kMaxStages = 16;
constexpr int kItemCostBf16 = 2, kItemCostFp8 = 2;  // start-up of a stream in tiles (balanced mode; measured)
constexpr int kBf16Stages = 4;  // ring depth of the bf16 kernels (launch_decode)
constexpr int kMaxDecodeGrid = 1024;  // split-K CTAs (one per SM); sizes the cut-record area of the workspace

struct DecodeParams {
    const uint16_t* q;
    const int32_t* block_table;
    int64_t bt_stride;
    const int32_t* seq_lens;
    int32_t S, Hq, Hkv, G;  // Hkv, G: VIRTUAL kv heads and heads per virtual kv head (kv_div below)
    int32_t kv_div;          // Hq/Hkv > 16: a kv head's group is split into kv_div sub-groups of G <= 16 heads, each
                             // its own stream over the same K/V (virtual kv head v reads real kv head v / kv_div)
    int32_t chunk;   // tokens per partition, multiple of the stage size (decode_tok)
    int32_t nparts;  // partition slots per (sequence, head) in the workspace (per set: a cascade row has two sets)
    int32_t slots;   // partial slots of a row = its stride in part_O / part_m / part_l (nparts; cascade 2 nparts)
    float scale_log2;
    float* part_O;  // [S*Hq][nparts][D]
    float* part_m;  // [S*Hq][nparts]   (log2 domain: max of scale*log2e*q.k)
    float* part_l;  // [S*Hq][nparts]
    void* out;
    float* lse;
    int32_t out_f32;
    int32_t direct;  // nparts == 1: write the final output, no combine pass
    int32_t nstages;
    // balanced mode (num_partitions = 0): the (sequence, kv head) streams are laid end to end in 64-token tiles and
    // every CTA takes a contiguous range of them, equal in cost (item_cost below).  A stream that lies inside one range is finished by its CTA
    // (final output, no partial); a stream cut by range boundaries yields one partial per piece, and the CTA that
    // holds its first piece records it in cut[] for the combine pass -- at most one record per CTA, since only the
    // last stream of a range can continue into the next.  chunk == decode_tok then; per_min bounds the pieces of
    // one stream by nparts.
    int32_t balanced;
    int32_t per_min;
    int32_t item_cost;  // balanced mode: the start-up of a stream (Q load, first page ids, merge, partial write) counted
                        // in tiles when the CTA ranges are cut: a stream of nt tiles costs nt + item_cost
    int4* cut;  // [gridDim.x] per CTA: {s, kvh, pieces, 0} of the cut stream that BEGINS in its range, s = -1 if none
    // quantised pool (FP8 instantiations): value = e4m3(code) * scale[page][kv head]
    const float* k_scale;
    const float* v_scale;
    // Shared-prefix cascade (mstar_paged_attn_decode_cascade; casc_B = 0 otherwise).  The work list runs over V
    // VIRTUAL sequences instead of the S real ones: first casc_R * casc_ng prefix streams -- request r, branch group
    // bg: tokens [0, shared_lens[r]) read once for the casc_bpg branches of the group, one consumer warp group per
    // branch -- then the S suffix streams, tokens [shared_lens[s / B], seq_len) of
    // sequence s.  Every stream leaves partials only (prefix pieces in slots [0, nparts), suffix pieces in
    // [nparts, 2 nparts) of a row); the cascade combine merges the two sets of every (sequence, head) row.
    int32_t V;
    int32_t casc_B, casc_bpg, casc_ng, casc_R;
    const int32_t* shared_lens;  // [casc_R]
    int32_t* vpieces;            // [V][Hkv]: pieces of a stream, written by the CTA that holds its first tile (balanced)
};

struct ItemInfo {
    int32_t s, kvh, part, tok0, ntok;
    int32_t whole;  // the item is the sequence's whole stream: the consumers write the final output
    int32_t nb;     // sequences s .. s + nb - 1 share the item's K/V, one consumer warp group each (cascade prefix
                    // streams; 1 otherwise)
};

// (x0 - bf16(x0), x1 - bf16(x1)) as bf16x2, pk = pack_bf16x2(x0, x1): the part of x a bf16 operand drops.  The
// quantised-pool kernels fold the page's V scale into P before the rounding to bf16, so in a row of a few tokens
// (L = 1: p = 1) the 2^-8 relative rounding of p * v_scale reaches the output whole, on top of the output's own
// rounding -- 2.03e-2 against the 2e-2 gate on |v| = 3.4, found by the property tests at 20 x their examples.  Items
// of a single stage (RESID) therefore feed this residual through a second P V MMA; longer items, where the
// roundings of many terms average, run the unchanged loop.
__device__ __forceinline__ uint32_t bf16x2_residual(float x0, float x1, uint32_t pk) {
    return pack_bf16x2(x0 - __uint_as_float(pk << 16), x1 - __uint_as_float(pk & 0xffff0000u));
}

// EB = bytes per pool element (2 = bf16, 1 = e4m3); NB = consumer warp groups (cascade: one per stacked branch)
template <int D, int GH, int EB, int NWARPS, int NB = 1>
struct DecodeSmem {
    static constexpr int kWarps = NWARPS;
    static constexpr int kStageBytes = 2 * 16 * kWarps * D * EB;
    static constexpr int kScaleBytes = EB == 1 ? kMaxStages * 2 * 16 * 4 : 0;  // [stage][K|V][page of the stage] fp32
    static constexpr int kQBytes = NB * GH * D * 2;
    static constexpr int kMergeBytes = NB * kWarps * GH * (D + 2) * 4;
    // fixed part after the ring: Q slots, merge buffer, barriers, item info
    static constexpr int kFixed = 2 * kQBytes + kMergeBytes + (2 * kMaxStages + 4) * 8 + 2 * 32 + kScaleBytes;
    static size_t bytes(int nstages, int S) {
        return 1024 + (size_t)nstages * kStageBytes + kFixed + (size_t)(2 * S + 1) * 4 + 16;
    }
};

__device__ __forceinline__ void store_out_vec(void* out, int out_f32, size_t idx, const float* v, int n) {
    if (out_f32) {
        float* o = reinterpret_cast<float*>(out) + idx;
        for (int i = 0; i < n; ++i) o[i] = v[i];
    } else {
        __nv_bfloat16* o = reinterpret_cast<__nv_bfloat16*>(out) + idx;
        for (int i = 0; i < n; i += 2) {
            *reinterpret_cast<uint32_t*>(o + i) = pack_bf16x2(v[i], v[i + 1]);
        }
    }
}

// MSTAR_FP8_BIAS_IN_SCALES = 1: the packed multiply is dropped; the MMAs run on code values times 2^-120 (subnormal
// codes are bf16 subnormals, which the tensor core takes exactly) and the factor is returned in two halves that keep
// every accumulator in the normal fp32 range: Q and P carry 2^60, the logits and O get the other 2^60 in fp32.
#ifndef MSTAR_FP8_BIAS_IN_SCALES
#define MSTAR_FP8_BIAS_IN_SCALES 1
#endif
constexpr float kTwo60 = 1152921504606846976.f;  // 2^60
// Two E4M3 codes -> two bf16, exactly.  PRMT picks the two bytes of w into the low byte of each 16-bit lane and
// replicates their sign bit over the high byte (selector nibbles 8..11); times 16 moves the 7 exponent / mantissa
// bits to bits [10:4]; the mask keeps them and one copy of the sign (bit 15).  That is the bf16 of the code's value
// with exponent bias 127 instead of 7 (subnormal codes land on bf16 subnormals); one packed multiply by 2^120 fixes
// the bias.  Two ALU-pipe and two FMA-pipe instructions per pair.
template <uint32_t SEL>
__device__ __forceinline__ uint32_t e4m3x2_to_bf16x2(uint32_t w) {
    uint32_t y;  // prmt in its default mode: selector nibbles 8..15 replicate the sign of byte (nibble & 7)
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(y) : "r"(w), "r"(0u), "n"(SEL));
    uint32_t x = (y * 16u) & 0x87f087f0u;
#if !MSTAR_FP8_BIAS_IN_SCALES
    asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(x) : "r"(x), "r"(0x7B807B80u));
#endif
    return x;
}
constexpr uint32_t kSelK01 = 0x9180, kSelK23 = 0xB3A2;  // bytes (0, 1) | (2, 3) of a word: 4 consecutive d of a token
constexpr uint32_t kSelV02 = 0xA280, kSelV13 = 0xB391;  // bytes (0, 2) | (1, 3): one d of two consecutive tokens

// transpose of an 8x8 b16 matrix held one row per lane group (lane (g, t4): row g, columns 2t4, 2t4+1)
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
    uint32_t d;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
    return d;
}

// NB > 1 (cascade calls): NB groups of NWARPS consumer warps work on the same ring stage, group b with the query
// rows of branch b of the item (sequence it.s + b), so the K/V of a shared prefix pass through shared memory once for
// NB branches at the per-warp cost of a single one; groups b >= it.nb only hand the stage back.
template <int D, int PAGE, int GH, bool FP8, int NWARPS, int NB = 1>
__global__ void __launch_bounds__(decode_threads(NWARPS, NB), 1)
decode_splitk_kernel(const __grid_constant__ CUtensorMap kmap, const __grid_constant__ CUtensorMap vmap,
                     const DecodeParams p) {
    constexpr int NW = NWARPS;       // consumer warps of a group (16 tokens of a stage each)
    constexpr int NC = NWARPS * NB;  // consumer warps
    constexpr int TOK = decode_tok(NWARPS);
    constexpr int PPS = TOK / PAGE;  // pages per stage
    constexpr int EB = FP8 ? 1 : 2;    // bytes per pool element
    constexpr int NH = D * EB / 128;   // 128-byte column slices per row (bf16: 64-column halves)
    constexpr int HT = TOK * 128;      // bytes of one slice tile (TOK rows x 128 B)
    constexpr int KBYTES = NH * HT;    // K part of a stage
    using SM = DecodeSmem<D, GH, EB, NWARPS, NB>;
    static_assert(!FP8 || D == 128, "fp8 pool: one 128-byte line per token row");
    constexpr int VEC = D / 32;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - smem_u32(smem_raw));
    const int nstages = p.nstages;
    const uint32_t ring = base;
    const uint32_t qbuf = ring + nstages * SM::kStageBytes;
    uint8_t* g_after = gbase + (size_t)nstages * SM::kStageBytes;
    uint16_t* qbuf_g = reinterpret_cast<uint16_t*>(g_after);
    float* merge_O = reinterpret_cast<float*>(g_after + 2 * SM::kQBytes);        // [NC][GH][D]
    float* merge_m = merge_O + NC * GH * D;                                      // [NC][GH]
    float* merge_l = merge_m + NC * GH;                                          // [NC][GH]
    uint64_t* bars_g = reinterpret_cast<uint64_t*>(g_after + 2 * SM::kQBytes + SM::kMergeBytes);
    const uint32_t bars = smem_u32(bars_g);
    ItemInfo* info = reinterpret_cast<ItemInfo*>(bars_g + 2 * kMaxStages + 4);
    float* sc_ring = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(info) + 2 * 32);  // FP8 only
    int32_t* cum = reinterpret_cast<int32_t*>(reinterpret_cast<uint8_t*>(info) + 2 * 32 + SM::kScaleBytes);  // [V + 1]
    int32_t* lens = cum + p.V + 1;                                                                              // [V]
    auto full_bar = [&](int st) { return bars + 8u * st; };
    auto empty_bar = [&](int st) { return bars + 8u * (kMaxStages + st); };
    auto qfull_bar = [&](int qs) { return bars + 8u * (2 * kMaxStages + qs); };
    auto qempty_bar = [&](int qs) { return bars + 8u * (2 * kMaxStages + 2 + qs); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < nstages; ++i) {
            mbar_init(full_bar(i), 2);  // K producer + V producer (each with its own transaction bytes)
            mbar_init(empty_bar(i), NC);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(qfull_bar(i), 1);
            mbar_init(qempty_bar(i), NC);
        }
        fence_mbar_init();
    }
    // zero the Q slots once: rows >= G are MMA padding and must stay 0 (bulk copies only write rows < G)
    for (int i = threadIdx.x; i < 2 * SM::kQBytes / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(qbuf_g)[i] = 0u;
    fence_proxy_async_smem();
    __syncthreads();
    // let the combine grid (launched with programmatic stream serialization) become resident now; it blocks in
    // griddepcontrol.wait until this grid has completed
    asm volatile("griddepcontrol.launch_dependents;");
    // This grid is itself launched with programmatic stream serialization: everything above (barrier init, Q-slot
    // zeroing) may overlap the tail of the previous kernel in the stream.  Every global read or write below -- seq_lens
    // and the block table may have been written by that kernel (a device-side step advance in a captured decode
    // loop), `out` may still be read by it -- happens after it has completed and its writes are visible.
    asm volatile("griddepcontrol.wait;" ::: "memory");

    if (warp >= NC) {
        // Two producer warps walk the same item list: warp NW loads the K half of every stage (and Q and the item
        // record), warp NW + 1 the V half.  Each TMA issue with per-lane coordinates is serialised by the hardware
        // interface, so two warps halve the issue time per stage (16 operations per stage at page size 16).
        const int op_isv = warp - NC;
        // =============================== PRODUCER ===============================
        prefetch_tensormap(&kmap);
        prefetch_tensormap(&vmap);
        // exclusive prefix sum of per-sequence partition counts -> compact work list (over the virtual sequences
        // of a cascade call: prefix streams, then suffix streams)
        const int n_prefix = p.casc_B ? p.casc_R * p.casc_ng : 0;
        auto vlen = [&](int v) -> int {
            if (!p.casc_B) return max(__ldg(p.seq_lens + v), 0);
            if (v < n_prefix) return max(__ldg(p.shared_lens + v / p.casc_ng), 0);
            const int sq = v - n_prefix;
            return max(__ldg(p.seq_lens + sq) - max(__ldg(p.shared_lens + sq / p.casc_B), 0), 0);
        };
        int carry = 0;
        auto scan_round = [&](int s0, int len) {
            const int s = s0 + lane;
            if (s < p.V) lens[s] = len;
            // fixed partitions: partitions of the sequence; balanced: its cost per kv head, tiles + start-up
            const int n = (len + p.chunk - 1) / p.chunk + ((p.balanced && len > 0) ? p.item_cost : 0);
            int incl = n;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            if (s < p.V) cum[s] = carry + incl - n;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        };
        // the lengths of the first 256 sequences are requested together (one round trip to memory instead of one
        // per 32 sequences: the serving batches are a few hundred sequences and this is the start of every CTA)
        constexpr int PRE = 8;
        int pre[PRE];
#pragma unroll
        for (int k = 0; k < PRE; ++k) pre[k] = (k * 32 + lane < p.V) ? vlen(k * 32 + lane) : 0;
#pragma unroll
        for (int k = 0; k < PRE; ++k)
            if (k * 32 < p.V) scan_round(k * 32, pre[k]);
        for (int s0 = PRE * 32; s0 < p.V; s0 += 32) scan_round(s0, (s0 + lane < p.V) ? vlen(s0 + lane) : 0);
        if (lane == 0) cum[p.V] = carry;
        __syncwarp();
        const int n_items = carry * p.Hkv;
        const uint64_t pol = policy_evict_first();
        // this lane's TMA op within a stage: (page i, K or V, 64-column half)
        constexpr int OPS = PPS * NH;
        const int op_page = lane / NH;
        const int op_half = lane % NH;
        const uint32_t op_off = op_isv * KBYTES + op_half * HT + op_page * (PAGE * 128);

        int st = 0, ph = 0, qs = 0, qph = 0;
        // hand one work item to the consumers and stream its K/V tiles into the ring
        auto emit_item = [&](int s, int kvh, int part, int tok0, int ntok, int whole) {
            const int ntiles = (ntok + TOK - 1) / TOK;
            const int kvh_r = kvh / p.kv_div;  // the pool's kv head
            int nb = 1;
            if (p.casc_B) {  // s is a virtual sequence: translate to (first real sequence, branches, token offset)
                whole = 0;
                if (s < n_prefix) {
                    const int r = s / p.casc_ng, bg = s - r * p.casc_ng;
                    nb = min(p.casc_bpg, p.casc_B - bg * p.casc_bpg);
                    s = r * p.casc_B + bg * p.casc_bpg;
                } else {
                    s -= n_prefix;
                    tok0 += max(__ldg(p.shared_lens + s / p.casc_B), 0);
                    part += p.nparts;
                }
            }
            if (!op_isv) mbar_wait(qempty_bar(qs), qph ^ 1);
            if (lane == 0 && !op_isv) {
                info[qs] = ItemInfo{s, kvh, part, tok0, ntok, whole, nb};
                mbar_arrive_expect_tx(qfull_bar(qs), (uint32_t)(nb * p.G * D * 2));
                for (int b = 0; b < nb; ++b)
                    bulk_load_1d(qbuf + qs * SM::kQBytes + b * GH * D * 2,
                                 p.q + ((size_t)(s + b) * p.Hq + (size_t)kvh * p.G) * D, (uint32_t)(p.G * D * 2),
                                 qfull_bar(qs));
            }
            qs ^= 1;
            if (qs == 0) qph ^= 1;

            const int32_t* bt = p.block_table + (size_t)s * p.bt_stride + tok0 / PAGE;
            int pg_next = -1;
            {
                const int npg0 = min(PPS, (ntok + PAGE - 1) / PAGE);
                if (lane < OPS && op_page < npg0) pg_next = __ldg(bt + op_page);
            }
            for (int t = 0; t < ntiles; ++t) {
                const int rem = ntok - t * TOK;
                const int npg = min(PPS, (rem + PAGE - 1) / PAGE);
                const int pg = pg_next;
                pg_next = -1;
                if (t + 1 < ntiles) {  // prefetch the next stage's page ids ahead of the ring wait
                    const int npg1 = min(PPS, (rem - TOK + PAGE - 1) / PAGE);
                    if (lane < OPS && op_page < npg1) pg_next = __ldg(bt + (t + 1) * PPS + op_page);
                }
                float pg_scale = 0.f;  // FP8: requested before the ring wait, which hides its latency
                if (FP8 && pg >= 0)
                    pg_scale = __ldg((op_isv ? p.v_scale : p.k_scale) + (size_t)pg * (p.Hkv / p.kv_div) + kvh_r);
                mbar_wait(empty_bar(st), ph ^ 1);
                if (FP8) {
                    if (pg >= 0) sc_ring[(st * 2 + op_isv) * 16 + op_page] = pg_scale;
                    __syncwarp();  // the scales are ordered before lane 0's (releasing) arrive
                }
                if (lane == 0) mbar_arrive_expect_tx(full_bar(st), (uint32_t)(npg * PAGE * D * EB));
                __syncwarp();
                if (pg >= 0)
                    tma_load_4d(ring + st * SM::kStageBytes + op_off, op_isv ? &vmap : &kmap, full_bar(st),
                                op_half * 64, 0, kvh_r, pg, pol);
                if (++st == nstages) { st = 0; ph ^= 1; }
            }
        };
        if (p.balanced) {
            // cum[] holds the COST of a sequence per kv head: nc = tiles + item_cost (chunk == TOK).  The streams
            // (sequence, kv head) lie end to end on the cost axis, a stream at [cum[s]*Hkv + kvh*nc, + nc): first its
            // start-up slot of item_cost units, then one unit per tile.  CTA b owns the tiles whose cost position lies
            // in [b*per, (b+1)*per): equal cost, not equal tile counts -- a CTA whose range holds many short streams
            // gets fewer tiles.
            const int K = p.item_cost;
            const int64_t N = (int64_t)carry * p.Hkv;
            int64_t per = (N + gridDim.x - 1) / gridDim.x;
            if (per < p.per_min) per = p.per_min;
            const int64_t ca = (int64_t)blockIdx.x * per;
            const int64_t cb = (ca + per < N) ? ca + per : N;
            bool cut_here = false;  // a stream begins in this range and continues past its end
            if (ca < N) {
                int lo = 0, hi = p.V;  // cum[lo]*Hkv <= ca < cum[hi]*Hkv
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if ((int64_t)cum[mid] * p.Hkv <= ca) lo = mid; else hi = mid;
                }
                int s = lo;
                int64_t c = ca;
                while (c < cb) {
                    const int nc = cum[s + 1] - cum[s], nt = nc - K;
                    const int64_t F0 = (int64_t)cum[s] * p.Hkv;
                    const int kvh = (int)((c - F0) / nc);
                    const int r = (int)((c - F0) - (int64_t)kvh * nc);
                    const int64_t cs = F0 + (int64_t)kvh * nc + K;  // cost position of the stream's first tile
                    const int tile = r > K ? r - K : 0;
                    const int64_t ct = cs + tile;                   // cost position of this tile (>= c)
                    if (ct >= cb) break;  // the range ends inside the start-up slot: the tiles belong to the next CTA
                    const int ntl = (int)(((int64_t)(nt - tile) < cb - ct) ? (nt - tile) : (cb - ct));
                    const int piece = (int)((int64_t)blockIdx.x - cs / per);
                    const int pieces = (int)((cs + nt - 1) / per - cs / per) + 1;
                    const int whole = (tile == 0 && ntl == nt) ? 1 : 0;
                    if (p.casc_B) {  // every stream leaves partials: the CTA with its first tile records the count
                        if (tile == 0 && lane == 0 && !op_isv) p.vpieces[(size_t)s * p.Hkv + kvh] = pieces;
                    } else if (tile == 0 && !whole) {
                        cut_here = true;
                        if (lane == 0 && !op_isv) p.cut[blockIdx.x] = make_int4(s, kvh, pieces, 0);
                    }
                    const int L = lens[s];
                    const int tok0 = tile * TOK;
                    emit_item(s, kvh, piece, tok0, min(L - tok0, ntl * TOK), whole);
                    c = ct + ntl;
                    if (tile + ntl == nt && kvh == p.Hkv - 1) {
                        ++s;
                        while (s < p.V && cum[s + 1] == cum[s]) ++s;  // sequences without tokens
                    }
                }
            }
            if (!p.casc_B && !cut_here && lane == 0 && !op_isv) p.cut[blockIdx.x] = make_int4(-1, 0, 0, 0);
        } else {
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                const int pi = item / p.Hkv, kvh = item - pi * p.Hkv;
                int lo = 0, hi = p.V;  // cum[lo] <= pi < cum[hi]
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (cum[mid] <= pi) lo = mid; else hi = mid;
                }
                const int s = lo, part = pi - cum[lo];
                const int L = lens[s];
                const int tok0 = part * p.chunk;
                emit_item(s, kvh, part, tok0, min(L - tok0, p.chunk), (p.direct || L <= p.chunk) ? 1 : 0);
            }
        }
        // sentinel: tell the consumers to stop
        if (!op_isv) mbar_wait(qempty_bar(qs), qph ^ 1);
        if (lane == 0 && !op_isv) {
            info[qs].ntok = -1;
            mbar_arrive(qfull_bar(qs));
        }
    } else {
        // =============================== CONSUMERS ===============================
        const int grp = warp / NW, w = warp % NW;  // warp group (branch of a stacked item), token slice of a stage
        const int g = lane >> 2, t4 = lane & 3;
        {  // empty sequences get out = 0, lse = -inf (no work item ever touches them, nor does the combine pass)
            for (int s = blockIdx.x * NC + warp; s < p.S; s += gridDim.x * NC) {
                if (__ldg(p.seq_lens + s) > 0) continue;
                for (int i = lane; i < p.Hq * D; i += 32) {
                    const size_t idx = (size_t)s * p.Hq * D + i;
                    if (p.out_f32) reinterpret_cast<float*>(p.out)[idx] = 0.f;
                    else reinterpret_cast<uint16_t*>(p.out)[idx] = 0;
                }
                if (p.lse) for (int h = lane; h < p.Hq; h += 32) p.lse[(size_t)s * p.Hq + h] = -INFINITY;
            }
        }
        // ldmatrix source rows / chunk selectors of this lane (see DESIGN.md 4.2 for the fragment maps)
        const uint32_t k_row = w * 16 + (lane >> 4) * 8 + (lane & 7);
        const uint32_t k_csel = (lane >> 3) & 1;
        const uint32_t v_row = w * 16 + ((lane >> 3) & 1) * 8 + (lane & 7);
        const uint32_t v_csel = lane >> 4;
        // FP8: one 16-byte chunk = 16 d values of a token; ldmatrix.x4 = (tokens 0-7 | 8-15) x (chunk c | c + 1)
        const uint32_t f_row = w * 16 + ((lane >> 3) & 1) * 8 + (lane & 7);
        const uint32_t f_csel = lane >> 4;

        int st = 0, ph = 0, qs = 0, qph = 0;
        while (true) {
            mbar_wait(qfull_bar(qs), qph);
            const ItemInfo it = info[qs];
            if (it.ntok < 0) break;
            const bool active = NB == 1 || grp < it.nb;  // a group without a branch in this item only frees the stages
            if constexpr (FP8 && GH == 8) {
                // ---- fp8 pool, G <= 8: operands swapped, S^T = K Q^T and O^T = V^T P^T, so the 16 MMA rows are tokens
                // (or d) and the 8 columns are the grouped heads: half the MMAs and accumulator registers of the
                // heads-as-rows form, no zero padding of the A operand.  Lane (g, t4): S^T rows = tokens g, g+8,
                // columns = heads 2t4, 2t4+1.
                uint32_t qb2[D / 16][2];  // B operand: Q^T[k slots of the 16-wide d block ks][head g]
                {
                    const uint16_t* qb = qbuf_g + qs * (SM::kQBytes / 2) + grp * GH * D;
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        qb2[ks][0] = *reinterpret_cast<const uint32_t*>(qb + g * D + ks * 16 + 4 * t4);
                        qb2[ks][1] = *reinterpret_cast<const uint32_t*>(qb + g * D + ks * 16 + 4 * t4 + 2);
                        if (MSTAR_FP8_BIAS_IN_SCALES) {  // Q * 2^60 (exact; |q| < 2^67)
                            asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(qb2[ks][0]) : "r"(qb2[ks][0]), "r"(0x5D805D80u));
                            asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(qb2[ks][1]) : "r"(qb2[ks][1]), "r"(0x5D805D80u));
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(qempty_bar(qs));
                qs ^= 1;
                if (qs == 0) qph ^= 1;

                float ot[D / 16][4];  // O^T: rows d = 16c + 2g (regs 0, 1) and 16c + 2g + 1 (regs 2, 3), columns = heads
#pragma unroll
                for (int c = 0; c < D / 16; ++c) ot[c][0] = ot[c][1] = ot[c][2] = ot[c][3] = 0.f;
                float mh0 = -INFINITY, mh1 = -INFINITY, lh0 = 0.f, lh1 = 0.f;  // heads 2t4, 2t4+1
                const int ntiles = (it.ntok + TOK - 1) / TOK;
                auto run_tiles = [&](auto resid_tag) {
                constexpr bool RESID = decltype(resid_tag)::value;  // single-stage item of a quantised pool
                for (int t = 0; t < ntiles; ++t) {
                    mbar_wait(full_bar(st), ph);
                    const int nv = min(16, it.ntok - t * TOK - w * 16);  // valid tokens in this warp's slice
                    if (active && nv > 0) {
                        const uint32_t kb = ring + st * SM::kStageBytes;
                        const uint32_t vb = kb + KBYTES;
                        float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};  // two MMA chains
#pragma unroll
                        for (int c2 = 0; c2 < D / 32; ++c2) {
                            uint32_t r0, r1, r2, r3;  // (tokens 0-7 | 8-15) x (chunk 2c2 | 2c2+1)
                            ldsm_x4(kb + swz128(f_row, 2 * c2 + f_csel), r0, r1, r2, r3);
                            mma_bf16_16816(sa, e4m3x2_to_bf16x2<kSelK01>(r0), e4m3x2_to_bf16x2<kSelK01>(r1),
                                           e4m3x2_to_bf16x2<kSelK23>(r0), e4m3x2_to_bf16x2<kSelK23>(r1),
                                           qb2[2 * c2][0], qb2[2 * c2][1]);
                            mma_bf16_16816(sb, e4m3x2_to_bf16x2<kSelK01>(r2), e4m3x2_to_bf16x2<kSelK01>(r3),
                                           e4m3x2_to_bf16x2<kSelK23>(r2), e4m3x2_to_bf16x2<kSelK23>(r3),
                                           qb2[2 * c2 + 1][0], qb2[2 * c2 + 1][1]);
                        }
                        float ksc = sc_ring[(st * 2 + 0) * 16 + (w * 16) / PAGE];  // this warp's page
                        if (MSTAR_FP8_BIAS_IN_SCALES) ksc *= kTwo60;
                        float s00 = (sa[0] + sb[0]) * ksc, s01 = (sa[1] + sb[1]) * ksc;  // token g,   heads 2t4, 2t4+1
                        float s10 = (sa[2] + sb[2]) * ksc, s11 = (sa[3] + sb[3]) * ksc;  // token g+8
                        if (g >= nv) s00 = s01 = -INFINITY;  // ragged tail: slots >= seq_len may hold any byte
                        if (g + 8 >= nv) s10 = s11 = -INFINITY;
                        // ---- online softmax per head: max over the 16 tokens = over the lanes of equal t4
                        float mx0 = fmaxf(s00, s10), mx1 = fmaxf(s01, s11);
#pragma unroll
                        for (int o2 = 4; o2 < 32; o2 <<= 1) {
                            mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, o2));
                            mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, o2));
                        }
                        const float mn0 = fmaxf(mh0, mx0), mn1 = fmaxf(mh1, mx1);
                        const float a0 = fast_exp2((mh0 - mn0) * p.scale_log2);
                        const float a1 = fast_exp2((mh1 - mn1) * p.scale_log2);
                        const float ms0 = mn0 * p.scale_log2, ms1 = mn1 * p.scale_log2;
                        mh0 = mn0;
                        mh1 = mn1;
                        const float p00 = fast_exp2(s00 * p.scale_log2 - ms0), p01 = fast_exp2(s01 * p.scale_log2 - ms1);
                        const float p10 = fast_exp2(s10 * p.scale_log2 - ms0), p11 = fast_exp2(s11 * p.scale_log2 - ms1);
                        lh0 = lh0 * a0 + (p00 + p10);
                        lh1 = lh1 * a1 + (p01 + p11);
                        // the page's V scale goes into P (the row sums keep the unscaled probabilities); P^T as the
                        // B operand = the 8x8 transposes of the two token halves
                        const float vsc = sc_ring[(st * 2 + 1) * 16 + (w * 16) / PAGE] *
                                          (MSTAR_FP8_BIAS_IN_SCALES ? kTwo60 : 1.f);
                        const uint32_t pk0 = pack_bf16x2(p00 * vsc, p01 * vsc), pk1 = pack_bf16x2(p10 * vsc, p11 * vsc);
                        const uint32_t pb0 = movmatrix_trans(pk0);
                        const uint32_t pb1 = movmatrix_trans(pk1);
                        uint32_t pl0 = 0u, pl1 = 0u;
                        if constexpr (RESID) {
                            pl0 = movmatrix_trans(bf16x2_residual(p00 * vsc, p01 * vsc, pk0));
                            pl1 = movmatrix_trans(bf16x2_residual(p10 * vsc, p11 * vsc, pk1));
                        }
                        const bool rescale = __any_sync(0xffffffffu, a0 != 1.f || a1 != 1.f);
                        uint32_t fr[4] = {0u, 0u, 0u, 0u};
#pragma unroll
                        for (int c = 0; c < D / 16; ++c) {
                            // transposed 8x8 b16 matrices = byte pairs: this lane gets V[2t4 | 2t4+1][2g | 2g+1] of the
                            // 16-wide d block c; MMA row g takes the even d, row g+8 the odd d
                            if ((c & 1) == 0) ldsm_x4_trans(vb + swz128(f_row, c + f_csel), fr[0], fr[1], fr[2], fr[3]);
                            const uint32_t lo = fr[(c & 1) * 2], hi = fr[(c & 1) * 2 + 1];
                            if (rescale) {
                                ot[c][0] *= a0; ot[c][1] *= a1; ot[c][2] *= a0; ot[c][3] *= a1;
                            }
                            mma_bf16_16816(ot[c], e4m3x2_to_bf16x2<kSelV02>(lo), e4m3x2_to_bf16x2<kSelV13>(lo),
                                           e4m3x2_to_bf16x2<kSelV02>(hi), e4m3x2_to_bf16x2<kSelV13>(hi), pb0, pb1);
                            if constexpr (RESID)
                                mma_bf16_16816(ot[c], e4m3x2_to_bf16x2<kSelV02>(lo), e4m3x2_to_bf16x2<kSelV13>(lo),
                                               e4m3x2_to_bf16x2<kSelV02>(hi), e4m3x2_to_bf16x2<kSelV13>(hi), pl0, pl1);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty_bar(st));
                    if (++st == nstages) { st = 0; ph ^= 1; }
                }
                };
                if (FP8 && ntiles == 1) run_tiles(std::true_type{}); else run_tiles(std::false_type{});
                // ---- hand (m, l, O) of this warp to the merge: row sums over the lanes of equal t4
#pragma unroll
                for (int o2 = 4; o2 < 32; o2 <<= 1) {
                    lh0 += __shfl_xor_sync(0xffffffffu, lh0, o2);
                    lh1 += __shfl_xor_sync(0xffffffffu, lh1, o2);
                }
                float* mo = merge_O + (size_t)(grp * NW + w) * GH * D;
                const float f = MSTAR_FP8_BIAS_IN_SCALES ? kTwo60 : 1.f;
#pragma unroll
                for (int c = 0; c < D / 16; ++c) {
                    *reinterpret_cast<float2*>(mo + (2 * t4) * D + c * 16 + 2 * g) = make_float2(ot[c][0] * f, ot[c][2] * f);
                    *reinterpret_cast<float2*>(mo + (2 * t4 + 1) * D + c * 16 + 2 * g) =
                        make_float2(ot[c][1] * f, ot[c][3] * f);
                }
                if (g == 0) {
                    merge_m[(grp * NW + w) * GH + 2 * t4] = mh0 * p.scale_log2;
                    merge_m[(grp * NW + w) * GH + 2 * t4 + 1] = mh1 * p.scale_log2;
                    merge_l[(grp * NW + w) * GH + 2 * t4] = lh0;
                    merge_l[(grp * NW + w) * GH + 2 * t4 + 1] = lh1;
                }
            } else {
                // Q fragments (A operand), rows = grouped query heads
                uint32_t qa[D / 16][4];
                {
                    const uint16_t* qb = qbuf_g + qs * (SM::kQBytes / 2) + grp * GH * D;
    #pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        // FP8: this lane's K bytes of a 16-wide d block are d = 4*t4 .. 4*t4+3 (one ldmatrix word), so
                        // the contraction index is permuted: MMA k-slots (2t4, 2t4+1 | 2t4+8, 2t4+9) <-> d (4t4, 4t4+1 |
                        // 4t4+2, 4t4+3); Q takes the same permutation
                        const int c0 = FP8 ? 4 * t4 : 2 * t4, c1 = FP8 ? 4 * t4 + 2 : 8 + 2 * t4;
                        qa[ks][0] = *reinterpret_cast<const uint32_t*>(qb + g * D + ks * 16 + c0);
                        qa[ks][2] = *reinterpret_cast<const uint32_t*>(qb + g * D + ks * 16 + c1);
                        if (GH == 16) {
                            qa[ks][1] = *reinterpret_cast<const uint32_t*>(qb + (g + 8) * D + ks * 16 + c0);
                            qa[ks][3] = *reinterpret_cast<const uint32_t*>(qb + (g + 8) * D + ks * 16 + c1);
                        } else {
                            qa[ks][1] = 0u;
                            qa[ks][3] = 0u;
                        }
                    }
                }
                if (FP8 && MSTAR_FP8_BIAS_IN_SCALES) {  // Q * 2^60 (exact; |q| < 2^67)
    #pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks)
    #pragma unroll
                        for (int i = 0; i < 4; ++i)
                            asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(qa[ks][i]) : "r"(qa[ks][i]), "r"(0x5D805D80u));
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(qempty_bar(qs));
                qs ^= 1;
                if (qs == 0) qph ^= 1;

                float o[D / 8][4];
    #pragma unroll
                for (int j = 0; j < D / 8; ++j) o[j][0] = o[j][1] = o[j][2] = o[j][3] = 0.f;
                float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // rows g and g+8 (raw q.k units)

                const int ntiles = (it.ntok + TOK - 1) / TOK;
                auto run_tiles = [&](auto resid_tag) {
                constexpr bool RESID = decltype(resid_tag)::value;  // single-stage item of a quantised pool
                for (int t = 0; t < ntiles; ++t) {
                    mbar_wait(full_bar(st), ph);
                    const int nv = min(16, it.ntok - t * TOK - w * 16);  // valid tokens in this warp's slice
                    if (active && nv > 0) {
                        const uint32_t kb = ring + st * SM::kStageBytes;
                        const uint32_t vb = kb + KBYTES;
                        // ---- S = Q K^T for 16 tokens (two n-blocks of 8)
                        float sc[2][4];
    #pragma unroll
                        for (int b = 0; b < 2; ++b) sc[b][0] = sc[b][1] = sc[b][2] = sc[b][3] = 0.f;
                        if constexpr (FP8) {
    #pragma unroll
                            for (int c2 = 0; c2 < D / 32; ++c2) {
                                uint32_t r0, r1, r2, r3;
                                ldsm_x4(kb + swz128(f_row, 2 * c2 + f_csel), r0, r1, r2, r3);
                                const int ka = 2 * c2, kc = 2 * c2 + 1;
                                mma_bf16_16816(sc[0], qa[ka][0], qa[ka][1], qa[ka][2], qa[ka][3],
                                               e4m3x2_to_bf16x2<kSelK01>(r0), e4m3x2_to_bf16x2<kSelK23>(r0));
                                mma_bf16_16816(sc[1], qa[ka][0], qa[ka][1], qa[ka][2], qa[ka][3],
                                               e4m3x2_to_bf16x2<kSelK01>(r1), e4m3x2_to_bf16x2<kSelK23>(r1));
                                mma_bf16_16816(sc[0], qa[kc][0], qa[kc][1], qa[kc][2], qa[kc][3],
                                               e4m3x2_to_bf16x2<kSelK01>(r2), e4m3x2_to_bf16x2<kSelK23>(r2));
                                mma_bf16_16816(sc[1], qa[kc][0], qa[kc][1], qa[kc][2], qa[kc][3],
                                               e4m3x2_to_bf16x2<kSelK01>(r3), e4m3x2_to_bf16x2<kSelK23>(r3));
                            }
                            float ksc = sc_ring[(st * 2 + 0) * 16 + (w * 16) / PAGE];  // this warp's page
                            if (MSTAR_FP8_BIAS_IN_SCALES) ksc *= kTwo60;
    #pragma unroll
                            for (int b = 0; b < 2; ++b) {
                                sc[b][0] *= ksc; sc[b][1] *= ksc; sc[b][2] *= ksc; sc[b][3] *= ksc;
                            }
                        } else {
    #pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks) {
                                const uint32_t chunk = 2 * ks + k_csel;
                                uint32_t b0, b1, b2, b3;
                                ldsm_x4(kb + (chunk >> 3) * HT + swz128(k_row, chunk & 7), b0, b1, b2, b3);
                                mma_bf16_16816(sc[0], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b0, b1);
                                mma_bf16_16816(sc[1], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b2, b3);
                            }
                        }
                        // ---- mask the ragged tail (slots >= seq_len may hold anything, incl. NaN)
                        uint32_t vmask_lo = 0xffffffffu, vmask_hi = 0xffffffffu;
                        if (nv < 16) {
    #pragma unroll
                            for (int b = 0; b < 2; ++b) {
                                const int c = b * 8 + 2 * t4;
                                if (c >= nv) sc[b][0] = sc[b][2] = -INFINITY;
                                if (c + 1 >= nv) sc[b][1] = sc[b][3] = -INFINITY;
                            }
                            vmask_lo = (2 * t4 < nv ? 0x0000ffffu : 0u) | (2 * t4 + 1 < nv ? 0xffff0000u : 0u);
                            vmask_hi = (8 + 2 * t4 < nv ? 0x0000ffffu : 0u) | (8 + 2 * t4 + 1 < nv ? 0xffff0000u : 0u);
                        }
                        // ---- online softmax (fp32), row max over the quad by shuffles
                        float mx0 = fmaxf(fmaxf(sc[0][0], sc[0][1]), fmaxf(sc[1][0], sc[1][1]));
                        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
                        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
                        const float mn0 = fmaxf(m0, mx0);
                        const float a0 = fast_exp2((m0 - mn0) * p.scale_log2);
                        const float ms0 = mn0 * p.scale_log2;
                        m0 = mn0;
                        const float p00 = fast_exp2(sc[0][0] * p.scale_log2 - ms0);
                        const float p01 = fast_exp2(sc[0][1] * p.scale_log2 - ms0);
                        const float p10 = fast_exp2(sc[1][0] * p.scale_log2 - ms0);
                        const float p11 = fast_exp2(sc[1][1] * p.scale_log2 - ms0);
                        l0 = l0 * a0 + (p00 + p01) + (p10 + p11);
                        // FP8: the page's V scale goes into P (the row sum l keeps the unscaled probabilities)
                        const float vsc = FP8 ? sc_ring[(st * 2 + 1) * 16 + (w * 16) / PAGE] *
                                                    (MSTAR_FP8_BIAS_IN_SCALES ? kTwo60 : 1.f) : 1.f;
                        uint32_t pa[4], pl[4] = {0u, 0u, 0u, 0u};
                        pa[0] = pack_bf16x2(p00 * vsc, p01 * vsc);
                        pa[2] = pack_bf16x2(p10 * vsc, p11 * vsc);
                        pa[1] = 0u;
                        pa[3] = 0u;
                        if constexpr (RESID) {
                            pl[0] = bf16x2_residual(p00 * vsc, p01 * vsc, pa[0]);
                            pl[2] = bf16x2_residual(p10 * vsc, p11 * vsc, pa[2]);
                        }
                        float a1 = 1.f;
                        if (GH == 16) {
                            float mx1 = fmaxf(fmaxf(sc[0][2], sc[0][3]), fmaxf(sc[1][2], sc[1][3]));
                            mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
                            mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
                            const float mn1 = fmaxf(m1, mx1);
                            a1 = fast_exp2((m1 - mn1) * p.scale_log2);
                            const float ms1 = mn1 * p.scale_log2;
                            m1 = mn1;
                            const float q00 = fast_exp2(sc[0][2] * p.scale_log2 - ms1);
                            const float q01 = fast_exp2(sc[0][3] * p.scale_log2 - ms1);
                            const float q10 = fast_exp2(sc[1][2] * p.scale_log2 - ms1);
                            const float q11 = fast_exp2(sc[1][3] * p.scale_log2 - ms1);
                            l1 = l1 * a1 + (q00 + q01) + (q10 + q11);
                            pa[1] = pack_bf16x2(q00 * vsc, q01 * vsc);
                            pa[3] = pack_bf16x2(q10 * vsc, q11 * vsc);
                            if constexpr (RESID) {
                                pl[1] = bf16x2_residual(q00 * vsc, q01 * vsc, pa[1]);
                                pl[3] = bf16x2_residual(q10 * vsc, q11 * vsc, pa[3]);
                            }
                        }
                        // ---- O = O * alpha + P V
                        // FP8 (issue-bound): skip the multiplies of a stage in which no row's running max moved
                        const bool rescale = !FP8 || __any_sync(0xffffffffu, a0 != 1.f || a1 != 1.f);
                        uint32_t fr[4] = {0u, 0u, 0u, 0u};
    #pragma unroll
                        for (int jj = 0; jj < D / 16; ++jj) {
                            uint32_t b0, b1, b2, b3;
                            if constexpr (FP8) {
                                // transposed 8x8 b16 matrices = byte pairs: this lane gets V[2t4 | 2t4+1][2g | 2g+1] of
                                // a 16-wide d block; n-block 2jj takes the even d (n = g <-> d = 2g), 2jj+1 the odd d
                                if ((jj & 1) == 0) ldsm_x4_trans(vb + swz128(f_row, jj + f_csel), fr[0], fr[1], fr[2], fr[3]);
                                const uint32_t lo = fr[(jj & 1) * 2], hi = fr[(jj & 1) * 2 + 1];
                                b0 = e4m3x2_to_bf16x2<kSelV02>(lo);
                                b1 = e4m3x2_to_bf16x2<kSelV02>(hi);
                                b2 = e4m3x2_to_bf16x2<kSelV13>(lo);
                                b3 = e4m3x2_to_bf16x2<kSelV13>(hi);
                            } else {
                                const uint32_t chunk = 2 * jj + v_csel;
                                ldsm_x4_trans(vb + (chunk >> 3) * HT + swz128(v_row, chunk & 7), b0, b1, b2, b3);
                            }
                            if (nv < 16) {  // 0 * NaN guard: zero V rows that hold no token
                                b0 &= vmask_lo; b1 &= vmask_hi; b2 &= vmask_lo; b3 &= vmask_hi;
                            }
                            if (rescale) {
                                o[2 * jj][0] *= a0; o[2 * jj][1] *= a0; o[2 * jj + 1][0] *= a0; o[2 * jj + 1][1] *= a0;
                                if (GH == 16) {
                                    o[2 * jj][2] *= a1; o[2 * jj][3] *= a1; o[2 * jj + 1][2] *= a1; o[2 * jj + 1][3] *= a1;
                                }
                            }
                            mma_bf16_16816(o[2 * jj], pa[0], pa[1], pa[2], pa[3], b0, b1);
                            mma_bf16_16816(o[2 * jj + 1], pa[0], pa[1], pa[2], pa[3], b2, b3);
                            if constexpr (RESID) {
                                mma_bf16_16816(o[2 * jj], pl[0], pl[1], pl[2], pl[3], b0, b1);
                                mma_bf16_16816(o[2 * jj + 1], pl[0], pl[1], pl[2], pl[3], b2, b3);
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty_bar(st));
                    if (++st == nstages) { st = 0; ph ^= 1; }
                }
                };
                if (FP8 && ntiles == 1) run_tiles(std::true_type{}); else run_tiles(std::false_type{});

                // ---- merge the four warps' (m, l, O) through shared memory
                l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
                l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
                if (GH == 16) {
                    l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
                    l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
                }
                {
                    float* mo = merge_O + (size_t)(grp * NW + w) * GH * D;
    #pragma unroll
                    for (int j = 0; j < D / 8; ++j) {
                        if constexpr (FP8) {  // n-blocks 2c | 2c+1 hold the even | odd d of block c: d = 16c + 4t4 + 0..3
                            if (j & 1) continue;
                            const float f = MSTAR_FP8_BIAS_IN_SCALES ? kTwo60 : 1.f;
                            *reinterpret_cast<float4*>(mo + g * D + j * 8 + 4 * t4) =
                                make_float4(o[j][0] * f, o[j + 1][0] * f, o[j][1] * f, o[j + 1][1] * f);
                            if (GH == 16)
                                *reinterpret_cast<float4*>(mo + (g + 8) * D + j * 8 + 4 * t4) =
                                    make_float4(o[j][2] * f, o[j + 1][2] * f, o[j][3] * f, o[j + 1][3] * f);
                        } else {
                            *reinterpret_cast<float2*>(mo + g * D + j * 8 + 2 * t4) = make_float2(o[j][0], o[j][1]);
                            if (GH == 16)
                                *reinterpret_cast<float2*>(mo + (g + 8) * D + j * 8 + 2 * t4) =
                                    make_float2(o[j][2], o[j][3]);
                        }
                    }
                    if (t4 == 0) {
                        merge_m[(grp * NW + w) * GH + g] = m0 * p.scale_log2;
                        merge_l[(grp * NW + w) * GH + g] = l0;
                        if (GH == 16) {
                            merge_m[(grp * NW + w) * GH + g + 8] = m1 * p.scale_log2;
                            merge_l[(grp * NW + w) * GH + g + 8] = l1;
                        }
                    }
                }
            }
            named_bar_sync(1 + grp, NW * 32);
            for (int r = w; r < (active ? p.G : 0); r += NW) {
                float M = -INFINITY;
#pragma unroll
                for (int x = 0; x < NW; ++x) M = fmaxf(M, merge_m[(grp * NW + x) * GH + r]);
                float acc[VEC];
#pragma unroll
                for (int i = 0; i < VEC; ++i) acc[i] = 0.f;
                float lsum = 0.f;
#pragma unroll
                for (int x = 0; x < NW; ++x) {
                    const float mx = merge_m[(grp * NW + x) * GH + r];
                    const float a = (mx == -INFINITY) ? 0.f : fast_exp2(mx - M);
                    lsum += a * merge_l[(grp * NW + x) * GH + r];
                    const float* src = merge_O + ((size_t)(grp * NW + x) * GH + r) * D + lane * VEC;
#pragma unroll
                    for (int i = 0; i < VEC; ++i) acc[i] += a * src[i];
                }
                const size_t row = (size_t)(it.s + grp) * p.Hq + (size_t)it.kvh * p.G + r;  // group = branch
                if (it.whole) {
                    const float inv = 1.f / lsum;
#pragma unroll
                    for (int i = 0; i < VEC; ++i) acc[i] *= inv;
                    store_out_vec(p.out, p.out_f32, row * D + lane * VEC, acc, VEC);
                    if (p.lse && lane == 0) p.lse[row] = (M + log2f(lsum)) * 0.6931471805599453f;
                } else {
                    float* dst = p.part_O + (row * p.slots + it.part) * D + lane * VEC;
#pragma unroll
                    for (int i = 0; i < VEC; ++i) dst[i] = acc[i];
                    if (lane == 0) {
                        p.part_m[row * p.slots + it.part] = M;
                        p.part_l[row * p.slots + it.part] = lsum;
                    }
                }
            }
            named_bar_sync(1 + grp, NW * 32);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// step a3: merge the partials of every (sequence, head) row that has more than one by log-sum-exp, normalise, round
// once.  One CTA of four warps per row; warp w takes pieces w, w + 4, ... with all of its loads in flight at once
// (a single round trip to memory for up to 16 pieces), the four warps meet in shared memory.  Rows:
//   fixed partitions  block = row; pieces = ceil(seq_len / chunk), the arithmetic the split-K kernel used; rows with
//                     one piece (or none) were finished by the split-K kernel.
//   balanced          block = (split-K CTA c, head r of the group): the cut record of c names the stream that begins
//                     in c's range and continues in the next ones, and its piece count; no record, nothing to do.
// The merge order is the piece order: deterministic.
template <int D>
__global__ void __launch_bounds__(128) decode_combine_kernel(const float* __restrict__ part_O,
                                                             const float* __restrict__ part_m,
                                                             const float* __restrict__ part_l,
                                                             const int32_t* __restrict__ seq_lens, int32_t chunk,
                                                             const int4* __restrict__ cut, int32_t G,
                                                             int32_t nparts, int32_t Hq, void* __restrict__ out,
                                                             float* __restrict__ lse, int32_t out_f32) {
    constexpr int VEC = D / 32;
    constexpr int PB = 4;  // pieces per warp per batch
    __shared__ float s_acc[4][D];
    __shared__ float s_l[4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // programmatic dependent launch: this grid may be resident before the split-K grid has finished; nothing it
    // reads (partials, cut records) is valid before this returns
    asm volatile("griddepcontrol.wait;" ::: "memory");
    int64_t row;
    int np;
    if (cut) {
        const int4 rec = cut[blockIdx.x / G];
        if (rec.x < 0) return;
        row = (int64_t)rec.x * Hq + (int64_t)rec.y * G + (blockIdx.x % G);
        np = rec.z;
    } else {
        row = blockIdx.x;
        const int L = seq_lens[row / Hq];
        np = (L + chunk - 1) / chunk;
        if (np <= 1) return;
    }
    const float* pm = part_m + row * nparts;
    const float* pl = part_l + row * nparts;
    const float* po = part_O + row * nparts * D + lane * VEC;
    float M = -INFINITY;
    for (int i = lane; i < np; i += 32) M = fmaxf(M, pm[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    float acc[VEC];
#pragma unroll
    for (int i = 0; i < VEC; ++i) acc[i] = 0.f;
    float lsum = 0.f;
    for (int i0 = warp; i0 < np; i0 += 4 * PB) {
        float v[PB][VEC], mi[PB], li[PB];
#pragma unroll
        for (int u = 0; u < PB; ++u) {
            const int i = i0 + 4 * u;
            mi[u] = -INFINITY;
            li[u] = 0.f;
#pragma unroll
            for (int e = 0; e < VEC; ++e) v[u][e] = 0.f;
            if (i < np) {
                mi[u] = pm[i];
                li[u] = pl[i];
                if constexpr (VEC == 4) {
                    const float4 t = *reinterpret_cast<const float4*>(po + (size_t)i * D);
                    v[u][0] = t.x; v[u][1] = t.y; v[u][2] = t.z; v[u][3] = t.w;
                } else {
                    const float2 t = *reinterpret_cast<const float2*>(po + (size_t)i * D);
                    v[u][0] = t.x; v[u][1] = t.y;
                }
            }
        }
#pragma unroll
        for (int u = 0; u < PB; ++u) {
            const float a = (mi[u] == -INFINITY) ? 0.f : fast_exp2(mi[u] - M);
            lsum += a * li[u];
#pragma unroll
            for (int e = 0; e < VEC; ++e) acc[e] += a * v[u][e];
        }
    }
#pragma unroll
    for (int e = 0; e < VEC; ++e) s_acc[warp][lane * VEC + e] = acc[e];
    if (lane == 0) s_l[warp] = lsum;
    __syncthreads();
    if (warp != 0) return;
    lsum = (s_l[0] + s_l[1]) + (s_l[2] + s_l[3]);
#pragma unroll
    for (int e = 0; e < VEC; ++e)
        acc[e] = (s_acc[0][lane * VEC + e] + s_acc[1][lane * VEC + e]) +
                 (s_acc[2][lane * VEC + e] + s_acc[3][lane * VEC + e]);
    const float inv = 1.f / lsum;
#pragma unroll
    for (int e = 0; e < VEC; ++e) acc[e] *= inv;
    store_out_vec(out, out_f32, (size_t)row * D + lane * VEC, acc, VEC);
    if (lse && lane == 0) lse[row] = (M + log2f(lsum)) * 0.6931471805599453f;
}

// ---------------------------------------------------------------------------------------------
// step a3 of a cascade call: one warp per (sequence, head) row merges the prefix pieces of the row's request / branch
// group (slots [0, np_p)) with the suffix pieces of its own sequence (slots [nparts, nparts + np_s)) by log-sum-exp
// in slot order (deterministic), normalises and rounds once.  Piece counts: fixed partitions -> from the lengths, the
// arithmetic the split-K kernel used; balanced -> the counts it recorded per stream.
template <int D>
__global__ void __launch_bounds__(128) decode_combine_cascade_kernel(
    const float* __restrict__ part_O, const float* __restrict__ part_m, const float* __restrict__ part_l,
    const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ shared_lens, const int32_t* __restrict__ vpieces,
    int32_t chunk, int32_t balanced, int32_t S, int32_t Hq, int32_t Hkv, int32_t G, int32_t B, int32_t bpg,
    int32_t ng, int32_t nparts, void* __restrict__ out, float* __restrict__ lse, int32_t out_f32) {
    constexpr int VEC = D / 32;
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (row >= (int64_t)S * Hq) return;
    const int s = (int)(row / Hq), h = (int)(row - (int64_t)s * Hq);
    const int L = seq_lens[s];
    if (L <= 0) return;  // zero-filled by the split-K kernel
    const int r = s / B, kvh = h / G;
    const int sh = min(max(shared_lens[r], 0), L);
    const int vp = r * ng + (s - r * B) / bpg, vs = (S / B) * ng + s;
    int np_p = 0, np_s = 0;
    if (sh > 0) np_p = balanced ? vpieces[(size_t)vp * Hkv + kvh] : (sh + chunk - 1) / chunk;
    if (L - sh > 0) np_s = balanced ? vpieces[(size_t)vs * Hkv + kvh] : (L - sh + chunk - 1) / chunk;
    const int slots = 2 * nparts;
    const float* pm = part_m + row * slots;
    const float* pl = part_l + row * slots;
    const float* po = part_O + row * slots * D + lane * VEC;
    // row maximum: lane i takes slot i of each set (at most 33 slots per set: one more round for lane 0)
    float M = -INFINITY;
    for (int i = lane; i < np_p; i += 32) M = fmaxf(M, pm[i]);
    for (int i = lane; i < np_s; i += 32) M = fmaxf(M, pm[nparts + i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    const float Mrow = M;
    float acc[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) acc[e] = 0.f;
    float lsum = 0.f;
    constexpr int PB = 4;  // pieces per batch: all loads of a batch are in flight before the first use
    for (int i0 = 0; i0 < np_p + np_s; i0 += PB) {
        float v[PB][VEC], mi[PB], li[PB];
#pragma unroll
        for (int u = 0; u < PB; ++u) {
            const int i = i0 + u;
            mi[u] = -INFINITY;
            li[u] = 0.f;
#pragma unroll
            for (int e = 0; e < VEC; ++e) v[u][e] = 0.f;
            if (i < np_p + np_s) {
                const int slot = i < np_p ? i : nparts + (i - np_p);
                mi[u] = pm[slot];
                li[u] = pl[slot];
                if constexpr (VEC == 4) {
                    const float4 t = *reinterpret_cast<const float4*>(po + (size_t)slot * D);
                    v[u][0] = t.x; v[u][1] = t.y; v[u][2] = t.z; v[u][3] = t.w;
                } else {
                    const float2 t = *reinterpret_cast<const float2*>(po + (size_t)slot * D);
                    v[u][0] = t.x; v[u][1] = t.y;
                }
            }
        }
#pragma unroll
        for (int u = 0; u < PB; ++u) {
            const float a = (mi[u] == -INFINITY) ? 0.f : fast_exp2(mi[u] - Mrow);
            lsum += a * li[u];
#pragma unroll
            for (int e = 0; e < VEC; ++e) acc[e] += a * v[u][e];
        }
    }
    const float inv = 1.f / lsum;
#pragma unroll
    for (int e = 0; e < VEC; ++e) acc[e] *= inv;
    store_out_vec(out, out_f32, (size_t)row * D + lane * VEC, acc, VEC);
    if (lse && lane == 0) lse[row] = (M + log2f(lsum)) * 0.6931471805599453f;
}

// ---------------------------------------------------------------------------------------------
static int32_t round_up(int32_t x, int32_t m) { return (x + m - 1) / m * m; }

static int32_t auto_chunk(int32_t S, int32_t Hkv, int32_t max_seq_len, int32_t tok) {
    // ~8 work items per SM at the length upper bound, 128..512-token partitions, at most 128 partitions
    const int64_t upper = (int64_t)S * Hkv * (max_seq_len > 0 ? max_seq_len : 1);
    int64_t c = upper / ((int64_t)device_sm_count() * 8);
    if (c < 128) c = 128;
    if (c > 512) c = 512;
    int32_t chunk = round_up((int32_t)c, tok);
    if ((max_seq_len + chunk - 1) / chunk > 128) chunk = round_up((max_seq_len + 127) / 128, tok);
    return chunk;
}

// num_partitions = 0: balanced mode when a sequence can span at least two tiles.  Slots per row = pieces a stream
// can be cut into: a CTA range is at least per_min = ceil(max_tiles / (slots - 1)) tiles long, so a stream of
// max_tiles tiles meets at most slots CTA ranges.
static bool balanced_plan(int32_t max_seq_len, int32_t tok, int32_t* nparts, int32_t* per_min) {
    const int32_t max_tiles = (max_seq_len + tok - 1) / tok;
    if (max_tiles < 2) return false;
    int32_t slots = (max_tiles + 1) / 2 + 1;
    if (slots > 33) slots = 33;
    *nparts = slots;
    *per_min = (max_tiles + slots - 2) / (slots - 1);
    return true;
}

static void partition_plan(int32_t S, int32_t Hkv, int32_t max_seq_len, int32_t num_partitions, int32_t tok,
                           int32_t* chunk, int32_t* nparts) {
    const int32_t msl = max_seq_len > 0 ? max_seq_len : 1;
    if (num_partitions <= 0) {
        int32_t per_min;
        if (balanced_plan(msl, tok, nparts, &per_min)) {
            *chunk = tok;
            return;
        }
        *chunk = auto_chunk(S, Hkv, msl, tok);
    } else {
        *chunk = round_up((msl + num_partitions - 1) / num_partitions, tok);
    }
    *nparts = (msl + *chunk - 1) / *chunk;
    if (num_partitions > 0 && *nparts > num_partitions) *nparts = num_partitions;
}

template <int D, int PAGE, int GH, bool FP8, int NWARPS, int NB = 1>
static int launch_decode(const PoolMaps& maps, DecodeParams& p, int max_items, cudaStream_t stream, int* grid_out) {
    using SM = DecodeSmem<D, GH, FP8 ? 1 : 2, NWARPS, NB>;
    const int max_smem = device_max_smem_optin();
    int nstages = (int)(((int64_t)max_smem - 1024 - SM::kFixed - (int64_t)(2 * p.V + 1) * 4 - 16) / SM::kStageBytes);
    if (nstages > kMaxStages) nstages = kMaxStages;
    // bf16 pool: four 32 KB stages in flight per SM (19 MB over the chip), not the six that fit -- measured on one box,
    // 60 GiB scattered pool: config 5 326.7 us with 6, 314.4 with 5, 312.3 with 4, 320.5 with 3; thinker / config 2
    // 66.5 -> 62.5 us.  The fp8 kernels (ALU-bound) measure the same from 3 stages up and keep what fits.
    if (!FP8 && nstages > kBf16Stages) nstages = kBf16Stages;
    if (nstages < 2) return MSTAR_ERR_UNSUPPORTED;
    p.nstages = nstages;
    const size_t smem = SM::bytes(nstages, p.V);
    auto kern = decode_splitk_kernel<D, PAGE, GH, FP8, NWARPS, NB>;
    static PerDeviceOnce attr_once;  // per instantiation
    MSTAR_CUDA_OK(set_max_dynamic_smem(attr_once, kern, max_smem));
    int grid = device_sm_count();
    if (grid > kMaxDecodeGrid) grid = kMaxDecodeGrid;
    if (grid > max_items) grid = max_items;
    if (grid < 1) grid = 1;
    *grid_out = grid;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(decode_threads(NWARPS, NB));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, kern, maps.k, maps.v, p));
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}

}  // namespace mstar

extern "C" int32_t mstar_paged_attn_decode_auto_partitions(int32_t num_seqs, int32_t num_kv_heads,
                                                           int32_t max_seq_len) {
    int32_t chunk, nparts;
    mstar::partition_plan(num_seqs, num_kv_heads, max_seq_len, 0, mstar::decode_tok(4), &chunk, &nparts);
    return nparts;
}

extern "C" size_t mstar_paged_attn_decode_workspace_bytes(int32_t num_seqs, int32_t num_q_heads, int32_t head_dim,
                                                          int32_t max_partitions) {
    if (num_seqs <= 0 || num_q_heads <= 0 || head_dim <= 0 || max_partitions <= 1) return 256;
    const size_t rows = (size_t)num_seqs * num_q_heads * max_partitions;
    // partials (O, m, l) + one 16-byte cut record per split-K CTA (balanced mode)
    return 256 + rows * head_dim * 4 + 2 * rows * 4 + 256 + 16 + (size_t)mstar::kMaxDecodeGrid * 16;
}

// Workspace of a cascade call: two sets of partial slots per row + one piece count per (virtual sequence, kv head).
static size_t cascade_workspace_bytes(int32_t num_seqs, int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                                      int32_t nparts) {
    const size_t rows = (size_t)num_seqs * num_q_heads * 2 * (size_t)nparts;
    return 256 + rows * head_dim * 4 + 2 * rows * 4 + 256 + 16 + (size_t)2 * num_seqs * num_kv_heads * 4 + 64;
}

// bf16 pool (k_scale == v_scale == NULL, fp8 false) or quantised pool; n_branches > 0: shared-prefix cascade
static int decode_entry(bool fp8, const float* k_scale, const float* v_scale, int32_t n_branches,
                        const int32_t* shared_lens, void* out, float* lse_out,
                        const void* q, const mstar_kv_pool* pool, const int32_t* block_table,
                        int64_t block_table_stride, const int32_t* seq_lens, int32_t num_seqs, int32_t num_q_heads,
                        int32_t max_seq_len, float scale, int32_t num_partitions, uint32_t flags, void* workspace,
                        size_t workspace_bytes, void* stream) {
    using namespace mstar;
    launch_count_reset();
    int rc = fp8 ? check_pool_fp8(pool) : check_pool(pool);
    if (rc != MSTAR_OK) return rc;
    if (fp8 && (!k_scale || !v_scale || !aligned(k_scale, 4) || !aligned(v_scale, 4))) return MSTAR_ERR_INVALID_ARG;
    if (flags & ~MSTAR_FLAG_OUT_F32) return MSTAR_ERR_INVALID_ARG;
    if (num_seqs < 0 || num_q_heads <= 0 || max_seq_len < 0 || num_partitions < 0) return MSTAR_ERR_INVALID_ARG;
    if (!(scale > 0.f) || !(scale < 3.0e38f)) return MSTAR_ERR_INVALID_ARG;  // positive and finite
    if (num_seqs == 0) return MSTAR_OK;
    if (!out || !q || !block_table || !seq_lens) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(out, 16) || !aligned(q, 16) || !aligned(block_table, 4) || !aligned(seq_lens, 4))
        return MSTAR_ERR_INVALID_ARG;
    if (num_q_heads % pool->num_kv_heads) return MSTAR_ERR_INVALID_ARG;
    // more than 16 heads per kv head: kv_div sub-groups of G <= 16 heads, each a stream of its own over the same K/V
    // (the repeats are L2 hits: the sub-groups' streams are neighbours in the work list)
    const int Greal = num_q_heads / pool->num_kv_heads;
    int kv_div = 1;
    if (Greal > 16) {
        for (int d = 2; d <= Greal; ++d)
            if (Greal % d == 0 && Greal / d <= 16) {
                kv_div = d;
                break;
            }
        if (kv_div == 1 || n_branches > 0) return MSTAR_ERR_UNSUPPORTED;  // a prime group size; cascade calls
    }
    const int G = Greal / kv_div;
    const int Hkv_v = pool->num_kv_heads * kv_div;
    if (num_seqs > 16384) return MSTAR_ERR_UNSUPPORTED;
    const bool casc = n_branches > 0;
    if (casc && (!shared_lens || !aligned(shared_lens, 4) || num_seqs % n_branches)) return MSTAR_ERR_INVALID_ARG;
    const int D = pool->head_dim, PAGE = pool->page_size;

    DecodeParams p{};
    const int nw = decode_pick_warps(fp8, G, max_seq_len);
    const int32_t tok = decode_tok(nw);
    partition_plan(num_seqs, pool->num_kv_heads, max_seq_len, num_partitions, tok, &p.chunk, &p.nparts);  // as the
    // workspace query does (mstar_paged_attn_decode_auto_partitions takes the pool's kv heads)
    if (num_partitions == 0)
        p.balanced = balanced_plan(max_seq_len > 0 ? max_seq_len : 1, tok, &p.nparts, &p.per_min) ? 1 : 0;
    p.item_cost = p.balanced ? (fp8 ? kItemCostFp8 : kItemCostBf16) : 0;
    p.direct = (p.nparts == 1) && !casc;
    p.slots = p.nparts;
    p.V = num_seqs;
    if (casc) {
        // up to three branches share one pass over the prefix, one consumer warp group each (G <= 8; above that
        // every branch reads the prefix itself)
        p.casc_B = n_branches;
        p.casc_bpg = G > 8 ? 1 : (n_branches < 3 ? n_branches : 3);
        p.casc_ng = (n_branches + p.casc_bpg - 1) / p.casc_bpg;
        p.casc_R = num_seqs / n_branches;
        p.shared_lens = shared_lens;
        p.V = p.casc_R * p.casc_ng + num_seqs;
        p.slots = 2 * p.nparts;
        const size_t need = cascade_workspace_bytes(num_seqs, num_q_heads, pool->num_kv_heads, D, p.nparts);
        if (!workspace || !aligned(workspace, 16)) return MSTAR_ERR_INVALID_ARG;
        if (workspace_bytes < need) return MSTAR_ERR_WORKSPACE_TOO_SMALL;
        const size_t rows = (size_t)num_seqs * num_q_heads * p.slots;
        p.part_O = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + 256);
        p.part_m = p.part_O + rows * D;
        p.part_l = p.part_m + rows;
        p.vpieces = reinterpret_cast<int32_t*>((reinterpret_cast<uintptr_t>(p.part_l + rows + 64) + 15) & ~uintptr_t(15));
    } else if (!p.direct) {
        const size_t need = mstar_paged_attn_decode_workspace_bytes(num_seqs, num_q_heads, D, p.nparts);
        if (!workspace || !aligned(workspace, 16)) return MSTAR_ERR_INVALID_ARG;
        if (workspace_bytes < need) return MSTAR_ERR_WORKSPACE_TOO_SMALL;
        const size_t rows = (size_t)num_seqs * num_q_heads * p.nparts;
        p.part_O = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + 256);
        p.part_m = p.part_O + rows * D;
        p.part_l = p.part_m + rows;
        p.cut = p.balanced ? reinterpret_cast<int4*>((reinterpret_cast<uintptr_t>(p.part_l + rows + 64) + 15) &
                                                     ~uintptr_t(15))
                           : nullptr;
    }
    p.q = reinterpret_cast<const uint16_t*>(q);
    p.block_table = block_table;
    p.bt_stride = block_table_stride;
    p.seq_lens = seq_lens;
    p.S = num_seqs;
    p.Hq = num_q_heads;
    p.Hkv = Hkv_v;
    p.kv_div = kv_div;
    p.G = G;
    p.scale_log2 = scale * 1.4426950408889634f;
    p.out = out;
    p.lse = lse_out;
    p.out_f32 = (flags & MSTAR_FLAG_OUT_F32) ? 1 : 0;
    p.k_scale = k_scale;
    p.v_scale = v_scale;

    PoolMaps maps;
    rc = fp8 ? get_pool_maps_fp8(pool, &maps) : get_pool_maps(pool, &maps);
    if (rc != MSTAR_OK) return rc;

    const int64_t max_items64 = (int64_t)p.V * p.nparts * Hkv_v;
    const int max_items = max_items64 > (1 << 30) ? (1 << 30) : (int)max_items64;
    cudaStream_t st = (cudaStream_t)stream;
    const bool g16 = G > 8;
    int grid = 0;
#define MSTAR_DECODE_CASE(DD, PP, F8, NWW)                                               \
    if (D == DD && PAGE == PP && fp8 == F8 && nw == NWW)                                 \
        rc = g16 ? launch_decode<DD, PP, 16, F8, NWW>(maps, p, max_items, st, &grid)     \
                 : launch_decode<DD, PP, 8, F8, NWW>(maps, p, max_items, st, &grid);
    rc = MSTAR_ERR_UNSUPPORTED;
    const bool grouped = casc && p.casc_bpg > 1;  // cascade with several consumer warp groups: launched below
    if (!grouped) {
        MSTAR_DECODE_CASE(128, 16, false, 4)
        MSTAR_DECODE_CASE(128, 32, false, 4)
        MSTAR_DECODE_CASE(64, 16, false, 4)
        MSTAR_DECODE_CASE(64, 32, false, 4)
        MSTAR_DECODE_CASE(128, 16, true, 8)
        MSTAR_DECODE_CASE(128, 32, true, 8)
        if (!g16) {  // 12 warps need the 111-register consumer of the G <= 8 form
            if (D == 128 && PAGE == 16 && fp8 && nw == 12)
                rc = launch_decode<128, 16, 8, true, 12>(maps, p, max_items, st, &grid);
            if (D == 128 && PAGE == 32 && fp8 && nw == 12)
                rc = launch_decode<128, 32, 8, true, 12>(maps, p, max_items, st, &grid);
        }
    }
#undef MSTAR_DECODE_CASE
    if (grouped) {  // bf16 pool, G <= 8: two or three consumer warp groups
#define MSTAR_CASCADE_CASE(DD, PP)                                                                  \
    if (D == DD && PAGE == PP)                                                                      \
        rc = p.casc_bpg == 2 ? launch_decode<DD, PP, 8, false, 4, 2>(maps, p, max_items, st, &grid) \
                             : launch_decode<DD, PP, 8, false, 4, 3>(maps, p, max_items, st, &grid);
        rc = MSTAR_ERR_UNSUPPORTED;
        MSTAR_CASCADE_CASE(128, 16)
        MSTAR_CASCADE_CASE(128, 32)
        MSTAR_CASCADE_CASE(64, 16)
        MSTAR_CASCADE_CASE(64, 32)
#undef MSTAR_CASCADE_CASE
    }
    if (rc != MSTAR_OK) return rc;

    if (casc) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)(((int64_t)num_seqs * num_q_heads + 3) / 4));
        cfg.blockDim = dim3(128);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        const float* cO = p.part_O;
        const float* cm = p.part_m;
        const float* cl = p.part_l;
        const int32_t* vp = p.vpieces;
        if (D == 128)
            MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, decode_combine_cascade_kernel<128>, cO, cm, cl, seq_lens, shared_lens,
                                             vp, p.chunk, p.balanced, num_seqs, num_q_heads, p.Hkv, (int32_t)G,
                                             p.casc_B, p.casc_bpg, p.casc_ng, p.nparts, out, lse_out, p.out_f32));
        else
            MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, decode_combine_cascade_kernel<64>, cO, cm, cl, seq_lens, shared_lens,
                                             vp, p.chunk, p.balanced, num_seqs, num_q_heads, p.Hkv, (int32_t)G,
                                             p.casc_B, p.casc_bpg, p.casc_ng, p.nparts, out, lse_out, p.out_f32));
        MSTAR_CUDA_OK(cudaGetLastError());
        launch_count_add(1);
    } else if (!p.direct) {
        // fixed partitions: one block per (sequence, head) row; balanced: one per (split-K CTA, head of the group)
        const int64_t blocks = p.balanced ? (int64_t)grid * G : (int64_t)num_seqs * num_q_heads;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)blocks);
        cfg.blockDim = dim3(128);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        const float* cO = p.part_O;
        const float* cm = p.part_m;
        const float* cl = p.part_l;
        const int4* ccut = p.cut;
        if (D == 128)
            MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, decode_combine_kernel<128>, cO, cm, cl, seq_lens, p.chunk, ccut,
                                             (int32_t)G, p.nparts, num_q_heads, out, lse_out, p.out_f32));
        else
            MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, decode_combine_kernel<64>, cO, cm, cl, seq_lens, p.chunk, ccut,
                                             (int32_t)G, p.nparts, num_q_heads, out, lse_out, p.out_f32));
        MSTAR_CUDA_OK(cudaGetLastError());
        launch_count_add(1);
    }
    return MSTAR_OK;
}

extern "C" int mstar_paged_attn_decode(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool,
                                       const int32_t* block_table, int64_t block_table_stride,
                                       const int32_t* seq_lens, int32_t num_seqs, int32_t num_q_heads,
                                       int32_t max_seq_len, float scale, int32_t num_partitions, uint32_t flags,
                                       void* workspace, size_t workspace_bytes, void* stream) {
    return decode_entry(false, nullptr, nullptr, 0, nullptr, out, lse_out, q, pool, block_table, block_table_stride, seq_lens,
                        num_seqs, num_q_heads, max_seq_len, scale, num_partitions, flags, workspace,
                        workspace_bytes, stream);
}

extern "C" int mstar_paged_attn_decode_fp8(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool8,
                                           const float* k_scale, const float* v_scale, const int32_t* block_table,
                                           int64_t block_table_stride, const int32_t* seq_lens, int32_t num_seqs,
                                           int32_t num_q_heads, int32_t max_seq_len, float scale,
                                           int32_t num_partitions, uint32_t flags, void* workspace,
                                           size_t workspace_bytes, void* stream) {
    return decode_entry(true, k_scale, v_scale, 0, nullptr, out, lse_out, q, pool8, block_table, block_table_stride, seq_lens,
                        num_seqs, num_q_heads, max_seq_len, scale, num_partitions, flags, workspace,
                        workspace_bytes, stream);
}

extern "C" size_t mstar_paged_attn_decode_cascade_workspace_bytes(int32_t num_seqs, int32_t num_q_heads,
                                                                  int32_t num_kv_heads, int32_t head_dim,
                                                                  int32_t max_seq_len) {
    if (num_seqs <= 0 || num_q_heads <= 0 || num_kv_heads <= 0 || head_dim <= 0) return 256;
    int32_t chunk, nparts;
    mstar::partition_plan(num_seqs, num_kv_heads, max_seq_len, 0, mstar::decode_tok(4), &chunk, &nparts);
    return cascade_workspace_bytes(num_seqs, num_q_heads, num_kv_heads, head_dim, nparts);
}

extern "C" int mstar_paged_attn_decode_cascade(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool,
                                               const int32_t* block_table, int64_t block_table_stride,
                                               const int32_t* seq_lens, const int32_t* shared_lens, int32_t num_seqs,
                                               int32_t n_branches, int32_t num_q_heads, int32_t max_seq_len,
                                               float scale, uint32_t flags, void* workspace, size_t workspace_bytes,
                                               void* stream) {
    if (n_branches < 1) return MSTAR_ERR_INVALID_ARG;
    return decode_entry(false, nullptr, nullptr, n_branches, shared_lens, out, lse_out, q, pool, block_table,
                        block_table_stride, seq_lens, num_seqs, num_q_heads, max_seq_len, scale, 0, flags, workspace,
                        workspace_bytes, stream);
}

// ------------------------------------------------------------------------------------------------------------------
// mstar_paged_attn_decode_static: the decode call for callers that cannot allocate device memory (code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The split-K partials and cut records -- the
// `workspace` of mstar_paged_attn_decode -- live in a file-scope device array of MSTAR_DECODE_STATIC_WORKSPACE_BYTES
// that every GPU which loads the library holds until the process exits.  Same kernels, same launch sequence and
// same arithmetic as mstar_paged_attn_decode; no cudaMalloc / cudaFree / allocating library routine on this path
// (nor anywhere else in the library: every other entry takes caller-owned scratch).
//
// In host code the array's NAME is a host-side stand-in, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress, resolved once per device with that device current, and cached per device ordinal.
// Contents: the array keeps whatever the last call left.  Nothing in it has to start at zero -- every partial slot
// and every cut record the combine pass reads is written by the split-K kernel of the same call (the existing path
// makes the same assumption about a caller's uninitialised workspace) -- so no clearing pass is launched.
// All calls on a device share the array: calls that overlap on the GPU (different streams, or one stream's call
// still running when another stream's starts) race on it; serialise them, or use mstar_paged_attn_decode with a
// workspace per stream.
static __device__ __align__(256) unsigned char g_decode_static_ws[MSTAR_DECODE_STATIC_WORKSPACE_BYTES];

namespace mstar {

static int decode_static_ws_address(void** out) {
    constexpr int kDevs = 64;
    static std::mutex mu;
    static void* ptrs[kDevs] = {};
    const int dev = current_device();
    std::lock_guard<std::mutex> lk(mu);
    if (dev >= 0 && dev < kDevs && ptrs[dev]) {
        *out = ptrs[dev];
        return MSTAR_OK;
    }
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_decode_static_ws);  // the CURRENT device's copy
    if (e != cudaSuccess || !ptr) {
        (void)cudaGetLastError();
        return MSTAR_ERR_CUDA;
    }
    if (dev >= 0 && dev < kDevs) ptrs[dev] = ptr;  // devices past the cache resolve the address on every call
    *out = ptr;
    return MSTAR_OK;
}

}  // namespace mstar

extern "C" int mstar_paged_attn_decode_static(void* out, float* lse_out, const void* q, const mstar_kv_pool* pool,
                                              const int32_t* block_table, int64_t block_table_stride,
                                              const int32_t* seq_lens, int32_t num_seqs, int32_t num_q_heads,
                                              int32_t max_seq_len, float scale, int32_t num_partitions,
                                              uint32_t flags, void* stream) {
    void* ws = nullptr;
    const int rc = mstar::decode_static_ws_address(&ws);
    if (rc != MSTAR_OK) return rc;
    // a geometry whose partials exceed the array comes back as MSTAR_ERR_WORKSPACE_TOO_SMALL, nothing launched
    return decode_entry(false, nullptr, nullptr, 0, nullptr, out, lse_out, q, pool, block_table, block_table_stride,
                        seq_lens, num_seqs, num_q_heads, max_seq_len, scale, num_partitions, flags, ws,
                        (size_t)MSTAR_DECODE_STATIC_WORKSPACE_BYTES, stream);
}
