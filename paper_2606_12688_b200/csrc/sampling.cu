// sampling.cu -- mstar_sample_tokens: CUDA-graph-compatible token sampling (last clause;
// PAPER.md:134 "a cuda-graph-compatible sampling plugin", :230; definition: DESIGN.md R28, oracle/sampling.py).
//
// Everything after the exponential is INTEGER arithmetic, so the result does not depend on the order in which threads
// (or CTAs) add: token weights are fixed-point, w_i = floor(2^32 * 2^((z_i - z_max) log2 e)), sums are 64-bit integers,
// the uniform number is the 64-bit fraction (x + 1/2) / 2^32 of a Philox4x32-10 word and the running sum is inverted
// in index order.  No state on the host: seeds and the step counter are device memory, so a replayed CUDA graph draws
// fresh numbers (MSTAR_FLAG_SAMPLE_ADVANCE_STEP adds 1 to the counter behind the sampling kernel).
//
// Two kernels that return the same token:
//   sample_tokens_cluster_kernel (default): a thread-block cluster per row, the row read from HBM once and kept in
//     shared memory, reductions over distributed shared memory;
//   sample_tokens_kernel (MSTAR_FLAG_SAMPLE_ONE_CTA, and vocabularies past the cluster kernel's capacity): one CTA per
//     row, the row re-read from L2 in every pass: maximum / argmax; [top-k: 8 radix-select passes on the order-
//     preserving integer image of z, 4 bits each, counting]; total weight; [top-p: 8 radix-select passes, weighing];
//     weight per warp segment; scan of the one segment that holds the target.  A radix-select pass keeps one private
//     16-bin histogram per thread in shared memory (no atomics) and reduces it afterwards.
#include <cuda_bf16.h>

#include "host_common.h"
#include "ptx.cuh"

namespace mstar {

constexpr int kSmpThreads = 1024;
constexpr int kSmpWarps = kSmpThreads / 32;

struct SampleParams {
    const void* logits;
    int64_t row_stride;  // elements
    int32_t vocab;
    int32_t bf16;
    const float* temperature;
    const int32_t* top_k;
    const float* top_p;
    const uint64_t* seeds;
    const uint64_t* step;
    int32_t* tokens;
};

__device__ __forceinline__ void philox4x32_10(uint32_t (&c)[4], uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        const uint32_t h0 = __umulhi(0xD2511F53u, c[0]), l0 = 0xD2511F53u * c[0];
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c[2]), l1 = 0xCD9E8D57u * c[2];
        const uint32_t n0 = h1 ^ c[1] ^ k0, n2 = h0 ^ c[3] ^ k1;
        c[0] = n0; c[1] = l1; c[2] = n2; c[3] = l0;
    }
}

// order-preserving map float -> uint32 (larger float, larger key; -0 and +0 share the key of +0: they are equal
// values, and the argmax takes the lowest index among equals)
__device__ __forceinline__ uint32_t order_key(float z) {
    uint32_t b = __float_as_uint(z);
    b = b == 0x80000000u ? 0u : b;
    return b ^ ((b >> 31) ? 0xffffffffu : 0x80000000u);
}

__device__ __forceinline__ uint64_t block_sum_u64(uint64_t v, uint64_t* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();  // red[] may still be read from a previous call
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    uint64_t s = 0;
#pragma unroll
    for (int w = 0; w < kSmpWarps; ++w) s += red[w];
    return s;
}

struct RowReader {
    const float* f;
    const __nv_bfloat16* h;
    float inv_t;
    int vec;  // the row starts on a 16-byte boundary: 16-byte loads
    __device__ __forceinline__ float z(int i) const {
        return (h ? __bfloat162float(h[i]) : f[i]) * inv_t;
    }
    // fn(index, z) for every index in [lo, hi) taken by thread `tid` of `nthreads`: consecutive threads take
    // consecutive 16-byte chunks, four chunks in flight per thread (lo must be a multiple of the chunk when vec is set)
    template <typename F>
    __device__ __forceinline__ void for_each(int lo, int hi, int tid, int nthreads, F fn) const {
        if (vec && f) {
            const int n4 = (hi - lo) >> 2;
            const float4* b = reinterpret_cast<const float4*>(f + lo);
            int c = tid;
            for (; c + 3 * nthreads < n4; c += 4 * nthreads) {
                float4 a[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) a[u] = __ldg(b + c + u * nthreads);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int i0 = lo + 4 * (c + u * nthreads);
                    fn(i0, a[u].x * inv_t); fn(i0 + 1, a[u].y * inv_t); fn(i0 + 2, a[u].z * inv_t);
                    fn(i0 + 3, a[u].w * inv_t);
                }
            }
            for (; c < n4; c += nthreads) {
                const float4 a0 = __ldg(b + c);
                const int i0 = lo + 4 * c;
                fn(i0, a0.x * inv_t); fn(i0 + 1, a0.y * inv_t); fn(i0 + 2, a0.z * inv_t); fn(i0 + 3, a0.w * inv_t);
            }
            for (int i = lo + 4 * n4 + tid; i < hi; i += nthreads) fn(i, f[i] * inv_t);
        } else if (vec && h) {
            const int n8 = (hi - lo) >> 3;
            const uint4* b = reinterpret_cast<const uint4*>(h + lo);
            auto chunk = [&](int i0, const uint4& a) {
                const uint32_t w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    fn(i0 + 2 * k, __uint_as_float(w[k] << 16) * inv_t);
                    fn(i0 + 2 * k + 1, __uint_as_float(w[k] & 0xffff0000u) * inv_t);
                }
            };
            int c = tid;
            for (; c + 3 * nthreads < n8; c += 4 * nthreads) {
                uint4 a[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) a[u] = __ldg(b + c + u * nthreads);
#pragma unroll
                for (int u = 0; u < 4; ++u) chunk(lo + 8 * (c + u * nthreads), a[u]);
            }
            for (; c < n8; c += nthreads) chunk(lo + 8 * c, __ldg(b + c));
            for (int i = lo + 8 * n8 + tid; i < hi; i += nthreads) fn(i, __bfloat162float(h[i]) * inv_t);
        } else {
            for (int i = lo + tid; i < hi; i += nthreads) fn(i, z(i));
        }
    }
};

// weight of a token: fixed-point 2^32 * exp(z - zmax), floor
__device__ __forceinline__ uint64_t weight_of(float z, float zmax) {
    // e in [0, 1] (ftz: no subnormals).  floor(e * 2^32) from the bits of e with shifts instead of a float -> integer
    // conversion (the conversion shares the SFU pipe with the exponential, and that pipe bounds a pass over the row)
    const uint32_t b = __float_as_uint(fast_exp2((z - zmax) * 1.4426950408889634f));
    const uint32_t m = (b & 0x007fffffu) | 0x00800000u;  // 24-bit significand, value m * 2^(exp - 150)
    const int sh = (int)(b >> 23) - 118;                 // e * 2^32 = m * 2^sh, sh <= 9
    if (b < 0x00800000u || sh < -23) return 0ull;        // e = 0 (or below 2^-32)
    return sh >= 0 ? ((uint64_t)m << sh) : (uint64_t)(m >> (-sh));
}

// Largest key theta with  sum over {i : key_i >= theta, key_i >= floor_key} of weight_i  >= target, where weight_i is 1
// (COUNT) or the token's fixed-point weight.  Returns theta; *mass_out = that sum.
template <bool COUNT>
__device__ uint32_t radix_select(const RowReader& rr, int V, float zmax, uint32_t floor_key, uint64_t target,
                                 uint64_t* hist /* [16][kSmpThreads] */, uint64_t* red, uint64_t* mass_out) {
    uint32_t theta = 0;
    uint64_t above = 0;  // weight of the tokens whose key is above every candidate of the current level
    for (int shift = 28; shift >= 0; shift -= 4) {
#pragma unroll
        for (int b = 0; b < 16; ++b) hist[b * kSmpThreads + threadIdx.x] = 0;
        const uint32_t prefix = shift == 28 ? 0u : (theta >> (shift + 4));
        rr.for_each(0, V, threadIdx.x, kSmpThreads, [&](int, float z) {
            const uint32_t key = order_key(z);
            if (key < floor_key) return;
            if (shift != 28 && (key >> (shift + 4)) != prefix) return;
            hist[((key >> shift) & 15u) * kSmpThreads + threadIdx.x] += COUNT ? 1ull : weight_of(z, zmax);
        });
        __syncthreads();
        // bin totals: warp w < 16 reduces bin w
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        if (warp < 16) {
            const int b = warp;
            uint64_t v = 0;
            for (int t = lane; t < kSmpThreads; t += 32) v += hist[b * kSmpThreads + t];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red[kSmpWarps + b] = v;
        }
        __syncthreads();
        // the largest digit d with above + sum_{b >= d} bin[b] >= target (d = 0 if none: target beyond the total)
        uint64_t cum = above;
        int d = 0;
        uint64_t above_next = above;
#pragma unroll
        for (int b = 15; b >= 0; --b) {
            const uint64_t nb = red[kSmpWarps + b];
            if (cum + nb >= target && cum < target) {
                d = b;
                above_next = cum;
            }
            cum += nb;
        }
        if (above >= target) {  // cannot happen for target <= total; keeps theta maximal otherwise
            d = 15;
            above_next = above;
        }
        theta |= (uint32_t)d << shift;
        above = above_next;
        if (shift == 0) above += red[kSmpWarps + d];  // + the tokens equal to theta: the weight of {key >= theta}
        __syncthreads();
    }
    *mass_out = above;
    return theta;
}

__global__ void __launch_bounds__(kSmpThreads) sample_tokens_kernel(const SampleParams p) {
    extern __shared__ uint64_t hist[];  // [16][kSmpThreads]
    __shared__ uint64_t red[kSmpWarps + 16];
    __shared__ uint64_t wseg[kSmpWarps];
    const int row = blockIdx.x, V = p.vocab;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float T = p.temperature ? p.temperature[row] : 1.f;
    RowReader rr;
    rr.f = p.bf16 ? nullptr : reinterpret_cast<const float*>(p.logits) + (size_t)row * p.row_stride;
    rr.h = p.bf16 ? reinterpret_cast<const __nv_bfloat16*>(p.logits) + (size_t)row * p.row_stride : nullptr;
    rr.inv_t = T > 0.f ? 1.f / T : 1.f;
    rr.vec = ((p.bf16 ? reinterpret_cast<uintptr_t>(rr.h) : reinterpret_cast<uintptr_t>(rr.f)) & 15) == 0;

    // ---- pass 1: maximum and its lowest index: max over (key << 32 | ~index)
    uint64_t best = 0;
    rr.for_each(0, V, threadIdx.x, kSmpThreads, [&](int i, float z) {
        const uint64_t c = ((uint64_t)order_key(z) << 32) | (uint32_t)(~(uint32_t)i);
        best = c > best ? c : best;
    });
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const uint64_t other = __shfl_xor_sync(0xffffffffu, best, o);
        best = other > best ? other : best;
    }
    if (lane == 0) red[warp] = best;
    __syncthreads();
    best = red[0];
#pragma unroll
    for (int w = 1; w < kSmpWarps; ++w) best = red[w] > best ? red[w] : best;
    const int argmax = (int)(~(uint32_t)best);
    if (!(T > 0.f)) {  // greedy
        if (threadIdx.x == 0) p.tokens[row] = argmax;
        return;
    }
    const float zmax = rr.z(argmax);

    // ---- top-k: the k-th largest key (ties at it are kept)
    uint32_t floor_key = 0;
    uint64_t dummy;
    const int k = p.top_k ? p.top_k[row] : 0;
    if (k > 0 && k < V) floor_key = radix_select<true>(rr, V, zmax, 0u, (uint64_t)k, hist, red, &dummy);

    // ---- total weight of the kept tokens
    auto kept_mass = [&](uint32_t fk) {
        uint64_t s = 0;
        rr.for_each(0, V, threadIdx.x, kSmpThreads, [&](int, float z) {
            if (order_key(z) >= fk) s += weight_of(z, zmax);
        });
        return block_sum_u64(s, red);
    };
    // ---- top-p: the largest key whose upper set weighs >= p * W
    const float tp = p.top_p ? p.top_p[row] : 1.f;
    uint64_t W = 0;  // without top-p the total falls out of the segment sums below
    if (tp > 0.f && tp < 1.f) {
        W = kept_mass(floor_key);
        uint64_t tgt = (uint64_t)ceil((double)tp * (double)W);
        tgt = tgt < 1 ? 1 : (tgt > W ? W : tgt);
        floor_key = radix_select<false>(rr, V, zmax, floor_key, tgt, hist, red, &W);
    }

    // ---- invert the running sum in index order: target = floor(u * W), u = (x + 1/2) / 2^32
    const uint64_t seed = p.seeds ? p.seeds[row] : 0ull, step = p.step ? *p.step : 0ull;
    uint32_t c[4] = {(uint32_t)step, (uint32_t)(step >> 32), (uint32_t)row, 0u};
    philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
    // warp w owns the contiguous segment [w * seg, (w + 1) * seg)
    const int seg = ((V + kSmpWarps - 1) / kSmpWarps + 7) & ~7;  // multiple of a 16-byte chunk of either type
    const int s0 = min(V, warp * seg), s1 = min(V, s0 + seg);
    uint64_t ws = 0;
    rr.for_each(s0, s1, lane, 32, [&](int, float z) {
        if (order_key(z) >= floor_key) ws += weight_of(z, zmax);
    });
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ws += __shfl_xor_sync(0xffffffffu, ws, o);
    __syncthreads();
    if (lane == 0) wseg[warp] = ws;
    __syncthreads();
    W = 0;
#pragma unroll
    for (int w = 0; w < kSmpWarps; ++w) W += wseg[w];
    const uint64_t target = __umul64hi(((uint64_t)c[0] << 32) | 0x80000000ull, W);
    uint64_t before = 0;
    int owner = -1;
#pragma unroll
    for (int w = 0; w < kSmpWarps; ++w) {
        if (owner < 0 && before + wseg[w] > target) owner = w;
        if (owner < 0) before += wseg[w];
    }
    if (owner < 0) {  // W == 0 cannot happen (the maximum weighs 2^32); guard
        if (threadIdx.x == 0) p.tokens[row] = argmax;
        return;
    }
    if (warp != owner) return;
    uint64_t run = before;  // weight of the kept tokens before the current round
    constexpr int RB = 8;   // rounds of 32 consecutive tokens whose loads are in flight together
    for (int base = s0; base < s1; base += 32 * RB) {
        uint64_t wv[RB];
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int i = base + 32 * r + lane;
            wv[r] = 0;
            if (i < s1) {
                const float z = rr.z(i);
                if (order_key(z) >= floor_key) wv[r] = weight_of(z, zmax);
            }
        }
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            uint64_t inc = wv[r];  // inclusive scan over the lanes
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            const unsigned hit = __ballot_sync(0xffffffffu, wv[r] > 0 && run + inc > target);
            if (hit) {
                if (lane == 0) p.tokens[row] = base + 32 * r + __ffs(hit) - 1;
                return;
            }
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Cluster kernel (the default path).  A row is split over the CTAs of a thread-block cluster (1, 2, 4 or 8 CTAs by
// vocabulary size); each CTA reads its slice from HBM exactly once and keeps it in shared memory as order-preserving
// integer keys of z, so every later pass is a pass over shared memory, and every reduction crosses the cluster through
// distributed shared memory behind one cluster barrier.  The arithmetic is the single-CTA kernel's (same keys, same
// fixed-point weights, same index-order inversion), so the two return the same token.
//   radix select: level 0 bins a token by x = z_max - z (256 bins over [0, 23); past 23 the fixed-point weight is 0),
//   which spreads the tokens that matter over the bins where the top byte of a float key would put them into two or
//   three; levels 1-4 are the four bytes of the key among the tokens of the chosen bin.  Histograms are 16-bit limbs of
//   the weights added with 32-bit shared-memory reductions (a slice has < 2^16 tokens, so a limb sum fits; sm_100 has
//   no native 64-bit shared atomic add).
constexpr int kCsThreads = 512;
constexpr int kCsWarps = kCsThreads / 32;
constexpr int kCsBins = 256;
constexpr int kCsMaxCluster = 8;
constexpr int kCsMaxSlice = 49152;          // tokens per CTA: 192 KB of keys (and < 2^16, see above)
constexpr uint32_t kKeyNegInf = 0x007fffffu;  // order_key(-inf): padding, weight 0
constexpr int kCsCand = 512;     // listed tokens per CTA
constexpr int kCsGather = 2048;  // and per cluster, for the select to finish on the gathered list
constexpr int kCsLoads = 8;                 // 16-byte loads in flight per thread in the pass over HBM

struct CsShared {
    uint32_t hist[2][3][kCsBins];  // [exchange parity][16-bit limb][digit]
    uint64_t xchg[2];              // [exchange parity]: the value this CTA publishes
    uint64_t gath[kCsMaxCluster];  // the published values of all ranks
    uint64_t wred[kCsWarps];
    uint64_t pick[3];              // crossing search: digit, weight above it, weight of it
    uint32_t ncand;                // tokens of the slice in the level-0 bin of the cut
    uint32_t cand[kCsCand];        // their keys, when they fit
    uint32_t range[2];             // the bin as a key range: first key of the bin, first key of the next bin
    uint32_t gl[kCsGather];        // the lists of all CTAs of the cluster
};

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
// all threads of all CTAs of the cluster; orders shared-memory writes before it against DSMEM reads after it
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t map_to_rank(uint32_t smem_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ uint32_t ld_cluster_u32(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ uint64_t ld_cluster_u64(uint32_t a) {
    uint64_t v;
    asm volatile("ld.shared::cluster.u64 %0, [%1];" : "=l"(v) : "r"(a) : "memory");
    return v;
}

__device__ __forceinline__ float key_to_float(uint32_t k) {
    return __uint_as_float(k ^ ((k >> 31) ? 0x80000000u : 0xffffffffu));
}

// level-0 digit: 255 - floor((zmax - z) * 255 / 23), clamped; larger z, larger (or equal) digit; digit 0 = weight 0
__device__ __forceinline__ uint32_t cs_digit0(float z, float zmax) {
    int b = __float2int_rz((zmax - z) * (255.f / 23.f));  // saturates; NaN -> 0
    b = min(max(b, 0), kCsBins - 1);
    return (uint32_t)(kCsBins - 1 - b);
}

// The fixed-point weight floor(2^32 e), e = 2^((z - zmax) log2 e) as in weight_of, as hi = floor(2^16 e) (0 .. 2^16) and
// lo = floor(2^32 e) - 2^16 hi (0 .. 2^16 - 1): two round-toward-zero additions of 2^23 leave the integer parts in the
// significand, the remainder between them is exact (it is a subset of the bits of e).  FMA-pipe instructions only; the
// one-CTA kernel gets the same integer from the bits of e with 64-bit shifts.
__device__ __forceinline__ void cs_weight(float z, float zmax, uint32_t& hi, uint32_t& lo) {
    const float e = fast_exp2((z - zmax) * 1.4426950408889634f);
    const float hf = __fadd_rz(e * 65536.f, 8388608.f);
    hi = __float_as_uint(hf) & 0x007fffffu;
    const float r = fmaf(8388608.f - hf, 65536.f, e * 4294967296.f);
    lo = __float_as_uint(__fadd_rz(r, 8388608.f)) & 0x007fffffu;
}

__device__ __forceinline__ uint64_t warp_scan_u64(uint64_t v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint64_t t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// Every CTA publishes thread 0's `mine`; afterwards sh.gath[r] holds rank r's value in every CTA.
__device__ __forceinline__ void cs_allgather(CsShared& sh, uint32_t& gen, uint64_t mine, uint32_t CS) {
    if (threadIdx.x == 0) sh.xchg[gen & 1] = mine;
    cluster_sync_all();
    if (threadIdx.x < CS) sh.gath[threadIdx.x] = ld_cluster_u64(map_to_rank(smem_u32(&sh.xchg[gen & 1]), threadIdx.x));
    __syncthreads();
    ++gen;
}

template <bool COUNT>
__device__ __forceinline__ void cs_hist_add(uint32_t* h, uint32_t d, uint32_t key, float zmax) {
    if (COUNT) {
        atomicAdd(&h[d], 1u);
    } else {
        uint32_t hi, lo;
        cs_weight(key_to_float(key), zmax, hi, lo);
        if (lo) atomicAdd(&h[d], lo);
        if (hi & 0xffffu) atomicAdd(&h[kCsBins + d], hi & 0xffffu);
        if (hi >> 16) atomicAdd(&h[2 * kCsBins + d], 1u);
    }
}

// Crossing search of one level.  tot = the level's total of digit 255 - tid in the threads tid < 256 (0 elsewhere).
// Finds the largest digit d with above + (total of the digits >= d) >= target, moves `above` to the weight above d
// and returns d.  set_target: target = ceil(tp * total of the level), clamped to [1, total], first.  Called by all
// threads; sh.pick[0] must hold ~0 (set behind a barrier that follows the previous call).
__device__ __forceinline__ uint32_t cs_cross(CsShared& sh, uint64_t tot, uint64_t& above, uint64_t& target,
                                             bool set_target, float tp) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    uint64_t incl = warp_scan_u64(tot, lane);
    if (lane == 31) sh.wred[warp] = incl;
    __syncthreads();
    uint64_t base = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kCsBins / 32; ++w) {
        const uint64_t t = sh.wred[w];
        if (w < warp) base += t;
        total += t;
    }
    if (set_target) {
        const uint64_t tgt = (uint64_t)ceil((double)tp * (double)total);
        target = tgt < 1 ? 1 : (tgt > total ? total : tgt);
    }
    incl += base;
    if (tid < kCsBins && above + incl >= target && above + (incl - tot) < target) {
        sh.pick[0] = (uint64_t)(kCsBins - 1 - tid);
        sh.pick[1] = above + (incl - tot);
    }
    __syncthreads();
    const uint64_t pd = sh.pick[0];
    if (pd == ~0ull) return 0u;  // never, for target <= total
    above = sh.pick[1];
    return (uint32_t)pd;
}

// The rest of a select behind level 0, when the tokens of bin d0 are few (the usual case): the bin is a key range
// (the level-0 digit is monotone in the key; its two ends by a 32-way search in one warp each), every CTA lists the
// keys of its slice in the range, all lists are gathered into every CTA through distributed shared memory, and the
// four key bytes are resolved on the gathered list with no further cluster traffic.  False (nothing decided) when a
// list overflows; the decision is the same in every CTA of the cluster.
template <bool COUNT>
__device__ bool cs_finish_on_list(CsShared& sh, const uint32_t* keys, int plen, float zmax, uint32_t floor_key,
                                  uint32_t d0, uint64_t above, uint64_t target, uint32_t CS, uint32_t& gen,
                                  uint32_t& theta_out) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (warp < 2) {  // warp 0: the first key of bin d0; warp 1: the first key of bin d0 + 1
        const uint32_t D = d0 + warp;
        uint32_t lo = kKeyNegInf, hi = 0xff800000u;  // the keys of -inf and +inf; digit(+inf) = 255
        if (D < (uint32_t)kCsBins) {
            while (lo < hi) {
                const uint32_t span = hi - lo, step = (span + 30u) / 31u;  // lane 31 probes hi
                const bool t = cs_digit0(key_to_float(lo + min(span, (uint32_t)lane * step)), zmax) >= D;
                const int L = __ffs(__ballot_sync(0xffffffffu, t)) - 1;
                hi = lo + min(span, (uint32_t)L * step);
                lo = L == 0 ? hi : lo + min(span, (uint32_t)(L - 1) * step) + 1u;
            }
        } else {
            lo = 0u;  // no bin above: the range is open
        }
        if (lane == 0) sh.range[warp] = lo;
    }
    if (tid == 0) sh.ncand = 0;
    __syncthreads();
    const uint32_t bin_lo = sh.range[0], khi = sh.range[1] - 1u, klo = max(bin_lo, floor_key);
    const uint4* k4 = reinterpret_cast<const uint4*>(keys);
    const int n4 = plen >> 2;
    for (int c0 = warp * 32; c0 < n4; c0 += kCsThreads) {  // the same trip count in every lane of a warp
        const bool valid = c0 + lane < n4;
        const uint4 q = valid ? k4[c0 + lane] : make_uint4(0u, 0u, 0u, 0u);
        const uint32_t kk[4] = {q.x, q.y, q.z, q.w};
        bool ps[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) ps[e] = valid && kk[e] >= klo && kk[e] <= khi;
        if (!__ballot_sync(0xffffffffu, ps[0] || ps[1] || ps[2] || ps[3])) continue;  // the usual case
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const unsigned m = __ballot_sync(0xffffffffu, ps[e]);
            if (m) {  // one atomic per warp
                uint32_t pos = 0;
                if (lane == __ffs(m) - 1) pos = atomicAdd(&sh.ncand, (uint32_t)__popc(m));
                pos = __shfl_sync(0xffffffffu, pos, __ffs(m) - 1) + __popc(m & ((1u << lane) - 1u));
                if (ps[e] && pos < (uint32_t)kCsCand) sh.cand[pos] = kk[e];
            }
        }
    }
    __syncthreads();
    cs_allgather(sh, gen, (uint64_t)sh.ncand, CS);  // its barrier also publishes cand[]
    uint32_t total = 0, offs[kCsMaxCluster];
    bool fits = true;
#pragma unroll
    for (uint32_t r = 0; r < (uint32_t)kCsMaxCluster; ++r) {
        const uint64_t cnt = r < CS ? sh.gath[r] : 0ull;
        fits = fits && cnt <= (uint64_t)kCsCand;
        offs[r] = total;
        total += (uint32_t)min(cnt, (uint64_t)kCsGather);
    }
    if (!fits || total > (uint32_t)kCsGather) return false;
    for (uint32_t g = tid; g < total; g += kCsThreads) {  // all remote loads of a thread in flight together
        uint32_t r = 0, first = 0;  // constant indices only: offs[] stays in registers
#pragma unroll
        for (uint32_t j = 1; j < (uint32_t)kCsMaxCluster; ++j)
            if (g >= offs[j]) {
                r = j;
                first = offs[j];
            }
        sh.gl[g] = ld_cluster_u32(map_to_rank(smem_u32(&sh.cand[0]), r) + 4u * (g - first));
    }
    __syncthreads();
    // One warp resolves the key bytes on the gathered list (peers read hist[] of level 0 before they arrive at the
    // barrier above, so both copies are free here).  All keys of the list lie in [bin_lo, khi]: the bytes above the
    // highest bit in which the two ends differ are common to all and are skipped.
    if (warp == 0) {
        uint32_t* h = &sh.hist[0][0][0];
        const uint32_t diff = bin_lo ^ khi;
        const int nb = diff ? 32 - __clz(diff) : 0;  // the low nb bits vary
        uint32_t theta = nb < 32 ? (bin_lo >> nb) << nb : 0u;
        for (int shift = ((nb + 7) / 8 - 1) * 8; shift >= 0; shift -= 8) {
            for (int i = lane; i < (COUNT ? 1 : 3) * kCsBins / 4; i += 32)
                reinterpret_cast<uint4*>(h)[i] = make_uint4(0u, 0u, 0u, 0u);
            __syncwarp();
            for (uint32_t i = lane; i < total; i += 32) {
                const uint32_t key = sh.gl[i];
                if (shift == 24 || (key >> (shift + 8)) == (theta >> (shift + 8)))
                    cs_hist_add<COUNT>(h, (key >> shift) & 255u, key, zmax);
            }
            __syncwarp();
            // lane l owns the digits 255 - 8 l down to 248 - 8 l
            uint64_t t[8], sum = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int d = kCsBins - 1 - 8 * lane - j;
                t[j] = (uint64_t)h[d];
                if (!COUNT) t[j] += ((uint64_t)h[kCsBins + d] << 16) + ((uint64_t)h[2 * kCsBins + d] << 32);
                sum += t[j];
            }
            const uint64_t incl = warp_scan_u64(sum, lane);
            uint64_t run = above + incl - sum;
            const unsigned hit = __ballot_sync(0xffffffffu, above + incl >= target && run < target);
            uint32_t d = 0;
            if (hit) {  // always, for target <= total
                bool found = false;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    if (!found && run + t[j] >= target) {
                        d = kCsBins - 1 - 8 * lane - j;
                        found = true;
                    }
                    if (!found) run += t[j];
                }
                d = __shfl_sync(0xffffffffu, d, __ffs(hit) - 1);
                above = __shfl_sync(0xffffffffu, run, __ffs(hit) - 1);
            }
            theta |= d << shift;
            __syncwarp();
        }
        if (lane == 0) sh.range[0] = theta;
    }
    __syncthreads();
    theta_out = sh.range[0];
    return true;
}

// As radix_select, over the cluster.  COUNT: target = k.  Otherwise target = ceil(tp * kept mass), the kept mass
// being the total of level 0.  Returns theta (0 = keep everything: the k-th largest token has weight 0).
template <bool COUNT>
__device__ uint32_t cs_select(CsShared& sh, const uint32_t* keys, int plen, float zmax, uint32_t floor_key,
                              uint64_t k_target, float tp, uint32_t CS, uint32_t& gen) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    uint32_t theta = 0, d0 = 0;
    uint64_t above = 0, target = k_target;
    bool listed = false;
    for (int level = 0; level < 5; ++level) {
        const int shift = 32 - 8 * level;  // levels 1..4: 24, 16, 8, 0
        uint32_t* h = &sh.hist[gen & 1][0][0];
        for (int i = tid; i < 3 * kCsBins; i += kCsThreads) h[i] = 0;
        if (level == 1 && tid == 0) sh.ncand = 0;
        __syncthreads();
        if (tid == 0) sh.pick[0] = ~0ull;
        if (listed) {
            const int nc = (int)sh.ncand;
            for (int i = tid; i < nc; i += kCsThreads) {
                const uint32_t key = sh.cand[i];
                if ((key >> (shift + 8)) == (theta >> (shift + 8)))
                    cs_hist_add<COUNT>(h, (key >> shift) & 255u, key, zmax);
            }
        } else {
            const uint4* k4 = reinterpret_cast<const uint4*>(keys);
            const int n4 = plen >> 2;
            for (int c0 = warp * 32; c0 < n4; c0 += kCsThreads) {  // the same trip count in every lane of a warp
                const bool valid = c0 + lane < n4;
                const uint4 q = valid ? k4[c0 + lane] : make_uint4(0u, 0u, 0u, 0u);
                const uint32_t kk[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t key = kk[e];
                    uint32_t d = cs_digit0(key_to_float(key), zmax);
                    bool pass = valid && key >= floor_key;
                    if (level > 0) {
                        pass = pass && d == d0;
                        if (level == 1) {  // the tokens of the bin, appended with one atomic per warp
                            const unsigned m = __ballot_sync(0xffffffffu, pass);
                            if (m) {
                                uint32_t pos = 0;
                                if (lane == __ffs(m) - 1) pos = atomicAdd(&sh.ncand, (uint32_t)__popc(m));
                                pos = __shfl_sync(0xffffffffu, pos, __ffs(m) - 1) + __popc(m & ((1u << lane) - 1u));
                                if (pass && pos < (uint32_t)kCsCand) sh.cand[pos] = key;
                            }
                        } else {
                            pass = pass && (key >> (shift + 8)) == (theta >> (shift + 8));
                        }
                        d = (key >> shift) & 255u;
                    }
                    if (pass) cs_hist_add<COUNT>(h, d, key, zmax);
                }
            }
        }
        cluster_sync_all();
        if (level == 1) listed = sh.ncand <= (uint32_t)kCsCand;  // per CTA: the histograms are the same either way
        // thread t < 256 owns digit 255 - t: its total over the cluster, then a prefix sum from the top digit down
        uint64_t tot = 0;
        if (tid < kCsBins) {
            const uint32_t a = smem_u32(&h[kCsBins - 1 - tid]);
            uint32_t l0[kCsMaxCluster], l1[kCsMaxCluster], l2[kCsMaxCluster];  // all loads of the 215-cycle path in flight
#pragma unroll
            for (uint32_t r = 0; r < (uint32_t)kCsMaxCluster; ++r) {
                const uint32_t ra = map_to_rank(a, r < CS ? r : 0u);
                l0[r] = ld_cluster_u32(ra);
                l1[r] = COUNT ? 0u : ld_cluster_u32(ra + 4 * kCsBins);
                l2[r] = COUNT ? 0u : ld_cluster_u32(ra + 8 * kCsBins);
            }
#pragma unroll
            for (uint32_t r = 0; r < (uint32_t)kCsMaxCluster; ++r)
                if (r < CS) tot += (uint64_t)l0[r] + ((uint64_t)l1[r] << 16) + ((uint64_t)l2[r] << 32);
        }
        const uint32_t d = cs_cross(sh, tot, above, target, !COUNT && level == 0, tp);
        ++gen;
        if (level == 0) {
            d0 = d;
            if (d0 == 0) return 0u;  // the cut falls among tokens of weight 0: keeping all of them changes nothing
            if (cs_finish_on_list<COUNT>(sh, keys, plen, zmax, floor_key, d0, above, target, CS, gen, theta))
                return theta;
        } else {
            theta |= d << shift;
        }
    }
    return theta;
}

__global__ void __launch_bounds__(kCsThreads, 2) sample_tokens_cluster_kernel(const SampleParams p, const int slice) {
    extern __shared__ __align__(16) unsigned char cs_smem[];
    CsShared& sh = *reinterpret_cast<CsShared*>(cs_smem);
    uint32_t* keys = reinterpret_cast<uint32_t*>(cs_smem + ((sizeof(CsShared) + 15) & ~(size_t)15));
    const uint32_t rank = cluster_ctarank(), CS = cluster_nctarank();
    const int row = blockIdx.x / CS, V = p.vocab;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int lo = min(V, (int)rank * slice), len = min(V, lo + slice) - lo, plen = (len + 3) & ~3;
    // every per-row parameter is requested here, in front of the pass over HBM (each is a cold miss of its own)
    const float T = p.temperature ? p.temperature[row] : 1.f;
    const int k = p.top_k ? p.top_k[row] : 0;
    const float tp = p.top_p ? p.top_p[row] : 1.f;
    const uint64_t seed = p.seeds ? p.seeds[row] : 0ull, step = p.step ? *p.step : 0ull;
    const float inv_t = T > 0.f ? 1.f / T : 1.f;
    uint32_t gen = 0;

    // ---- the one pass over HBM: z -> key into shared memory; maximum and its lowest index as max of (key << 32 | ~i)
    uint64_t best = 0;
    auto put = [&](int i, float logit) -> uint32_t {  // i: index in the slice
        const uint32_t key = order_key(logit * inv_t);
        const uint64_t c = ((uint64_t)key << 32) | (uint32_t)(~(uint32_t)(lo + i));
        best = c > best ? c : best;
        return key;
    };
    if (!p.bf16) {
        const float* f = reinterpret_cast<const float*>(p.logits) + (size_t)row * p.row_stride + lo;
        if ((reinterpret_cast<uintptr_t>(f) & 15) == 0) {
            const float4* b = reinterpret_cast<const float4*>(f);
            const int n4 = len >> 2;
            for (int c0 = tid; c0 < n4; c0 += kCsLoads * kCsThreads) {
                float4 a[kCsLoads];
#pragma unroll
                for (int u = 0; u < kCsLoads; ++u)
                    if (c0 + u * kCsThreads < n4) a[u] = __ldcs(b + c0 + u * kCsThreads);
#pragma unroll
                for (int u = 0; u < kCsLoads; ++u) {
                    const int c = c0 + u * kCsThreads;
                    if (c < n4) {
                        uint4 k;
                        k.x = put(4 * c, a[u].x); k.y = put(4 * c + 1, a[u].y);
                        k.z = put(4 * c + 2, a[u].z); k.w = put(4 * c + 3, a[u].w);
                        reinterpret_cast<uint4*>(keys)[c] = k;
                    }
                }
            }
            for (int i = 4 * n4 + tid; i < len; i += kCsThreads) keys[i] = put(i, f[i]);
        } else {
            for (int i = tid; i < len; i += kCsThreads) keys[i] = put(i, f[i]);
        }
    } else {
        const __nv_bfloat16* hp = reinterpret_cast<const __nv_bfloat16*>(p.logits) + (size_t)row * p.row_stride + lo;
        if ((reinterpret_cast<uintptr_t>(hp) & 15) == 0) {
            const uint4* b = reinterpret_cast<const uint4*>(hp);
            const int n8 = len >> 3;
            for (int c0 = tid; c0 < n8; c0 += kCsLoads * kCsThreads) {
                uint4 a[kCsLoads];
#pragma unroll
                for (int u = 0; u < kCsLoads; ++u)
                    if (c0 + u * kCsThreads < n8) a[u] = __ldcs(b + c0 + u * kCsThreads);
#pragma unroll
                for (int u = 0; u < kCsLoads; ++u) {
                    const int c = c0 + u * kCsThreads;
                    if (c < n8) {
                        const uint32_t w[4] = {a[u].x, a[u].y, a[u].z, a[u].w};
                        uint32_t k[8];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            k[2 * j] = put(8 * c + 2 * j, __uint_as_float(w[j] << 16));
                            k[2 * j + 1] = put(8 * c + 2 * j + 1, __uint_as_float(w[j] & 0xffff0000u));
                        }
                        reinterpret_cast<uint4*>(keys)[2 * c] = make_uint4(k[0], k[1], k[2], k[3]);
                        reinterpret_cast<uint4*>(keys)[2 * c + 1] = make_uint4(k[4], k[5], k[6], k[7]);
                    }
                }
            }
            for (int i = 8 * n8 + tid; i < len; i += kCsThreads) keys[i] = put(i, __bfloat162float(hp[i]));
        } else {
            for (int i = tid; i < len; i += kCsThreads) keys[i] = put(i, __bfloat162float(hp[i]));
        }
    }
    if (tid < plen - len) keys[len + tid] = kKeyNegInf;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const uint64_t other = __shfl_xor_sync(0xffffffffu, best, o);
        best = other > best ? other : best;
    }
    if (lane == 0) sh.wred[warp] = best;
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int w = 1; w < kCsWarps; ++w) best = sh.wred[w] > best ? sh.wred[w] : best;
    }
    cs_allgather(sh, gen, best, CS);
    best = sh.gath[0];
    for (uint32_t r = 1; r < CS; ++r) best = sh.gath[r] > best ? sh.gath[r] : best;
    const int argmax = (int)(~(uint32_t)best);
    const float zmax = key_to_float((uint32_t)(best >> 32));

    if (!(T > 0.f)) {  // greedy (the same branch in every CTA of the cluster)
        if (rank == 0 && tid == 0) p.tokens[row] = argmax;
    } else {
        uint32_t floor_key = 0;
        if (k > 0 && k < V) floor_key = cs_select<true>(sh, keys, plen, zmax, 0u, (uint64_t)k, 0.f, CS, gen);
        if (tp > 0.f && tp < 1.f) floor_key = cs_select<false>(sh, keys, plen, zmax, floor_key, 0ull, tp, CS, gen);

        // ---- invert the running sum in index order; thread t owns tokens [t n, (t + 1) n) of the slice, n odd
        // (consecutive lanes on distinct banks)
        const int n = ((slice + kCsThreads - 1) / kCsThreads) | 1;
        const int i0 = min(plen, tid * n), i1 = min(plen, i0 + n);
        uint32_t sum_hi = 0, sum_lo = 0;  // n < 2^7 tokens: no overflow
#pragma unroll 8
        for (int j = 0; j < n; ++j) {
            const int i = i0 + j;
            const uint32_t key = i < i1 ? keys[i] : 0u;
            uint32_t wh, wl;
            cs_weight(key_to_float(key), zmax, wh, wl);
            if (i < i1 && key >= floor_key) {
                sum_hi += wh;
                sum_lo += wl;
            }
        }
        const uint64_t mine = ((uint64_t)sum_hi << 16) + sum_lo;
        uint64_t incl = warp_scan_u64(mine, lane);
        __syncthreads();  // wred may still be read (select or the maximum)
        if (lane == 31) sh.wred[warp] = incl;
        __syncthreads();
        uint64_t base = 0, cta_total = 0;
#pragma unroll
        for (int w = 0; w < kCsWarps; ++w) {
            const uint64_t t = sh.wred[w];
            if (w < warp) base += t;
            cta_total += t;
        }
        cs_allgather(sh, gen, cta_total, CS);
        uint64_t W = 0, before = 0;
        for (uint32_t r = 0; r < CS; ++r) {
            const uint64_t t = sh.gath[r];
            if (r < rank) before += t;
            W += t;
        }
        uint32_t c[4] = {(uint32_t)step, (uint32_t)(step >> 32), (uint32_t)row, 0u};
        philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
        const uint64_t target = __umul64hi(((uint64_t)c[0] << 32) | 0x80000000ull, W);
        const uint64_t run = before + base + incl - mine;
        if (W == 0 && rank == 0 && tid == 0) p.tokens[row] = argmax;  // cannot happen (the maximum weighs 2^32); guard
        // exactly one thread of the cluster owns the target; its warp scans that thread's tokens together
        const unsigned own = __ballot_sync(0xffffffffu, W != 0 && mine > 0 && run <= target && target < run + mine);
        if (own) {
            const int src = __ffs(own) - 1;
            const int b0 = __shfl_sync(0xffffffffu, i0, src), b1 = __shfl_sync(0xffffffffu, i1, src);
            uint64_t r0 = __shfl_sync(0xffffffffu, run, src);
            for (int base_i = b0; base_i < b1; base_i += 32) {
                const int i = base_i + lane;
                const uint32_t key = i < b1 ? keys[i] : 0u;
                uint32_t wh, wl;
                cs_weight(key_to_float(key), zmax, wh, wl);
                const uint64_t w = (i < b1 && key >= floor_key) ? ((uint64_t)wh << 16) + wl : 0ull;
                const uint64_t inc = warp_scan_u64(w, lane);
                const unsigned hit = __ballot_sync(0xffffffffu, w > 0 && r0 + inc > target);
                if (hit) {
                    if (lane == 0) p.tokens[row] = lo + base_i + __ffs(hit) - 1;
                    break;
                }
                r0 += __shfl_sync(0xffffffffu, inc, 31);
            }
        }
    }
    cluster_sync_all();  // no CTA leaves while a peer may still read its shared memory
}

__global__ void sample_advance_kernel(uint64_t* step) { *step += 1; }

}  // namespace mstar

extern "C" int mstar_sample_tokens(int32_t* tokens_out, const void* logits, int64_t row_stride, int32_t num_rows,
                                   int32_t vocab, const float* temperature, const int32_t* top_k, const float* top_p,
                                   const uint64_t* seeds, uint64_t* step, uint32_t flags, void* stream) {
    using namespace mstar;
    launch_count_reset();
    if (flags & ~(MSTAR_FLAG_LOGITS_BF16 | MSTAR_FLAG_SAMPLE_ADVANCE_STEP | MSTAR_FLAG_SAMPLE_ONE_CTA))
        return MSTAR_ERR_INVALID_ARG;
    if (num_rows < 0 || vocab <= 0 || row_stride < vocab) return MSTAR_ERR_INVALID_ARG;
    if (num_rows == 0) return MSTAR_OK;
    if (!tokens_out || !logits || !seeds || !step) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(tokens_out, 4) || !aligned(seeds, 8) || !aligned(step, 8)) return MSTAR_ERR_INVALID_ARG;
    const bool bf = (flags & MSTAR_FLAG_LOGITS_BF16) != 0;
    if (!aligned(logits, bf ? 2 : 4)) return MSTAR_ERR_INVALID_ARG;
    SampleParams p{};
    p.logits = logits;
    p.row_stride = row_stride;
    p.vocab = vocab;
    p.bf16 = bf ? 1 : 0;
    p.temperature = temperature;
    p.top_k = top_k;
    p.top_p = top_p;
    p.seeds = seeds;
    p.step = step;
    p.tokens = tokens_out;
    cudaStream_t st = (cudaStream_t)stream;
    // cluster size by vocabulary: slices of at most 4096 tokens up to 4 CTAs, then 8 CTAs with whatever slice results
    const int cs = vocab <= 4096 ? 1 : vocab <= 8192 ? 2 : vocab <= 16384 ? 4 : kCsMaxCluster;
    const int slice = ((vocab + cs - 1) / cs + 7) & ~7;
    if (!(flags & MSTAR_FLAG_SAMPLE_ONE_CTA) && slice <= kCsMaxSlice) {
        const size_t smem = ((sizeof(CsShared) + 15) & ~(size_t)15) + (size_t)slice * 4;
        static PerDeviceOnce once_cs;
        MSTAR_CUDA_OK(set_max_dynamic_smem(once_cs, sample_tokens_cluster_kernel,
                                           (int)(((sizeof(CsShared) + 15) & ~(size_t)15) + (size_t)kCsMaxSlice * 4)));
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)num_rows * cs);
        cfg.blockDim = dim3(kCsThreads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = cs;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        MSTAR_CUDA_OK(cudaLaunchKernelEx(&cfg, sample_tokens_cluster_kernel, p, slice));
    } else {
        static PerDeviceOnce once;
        MSTAR_CUDA_OK(set_max_dynamic_smem(once, sample_tokens_kernel, 16 * kSmpThreads * 8));
        sample_tokens_kernel<<<(unsigned)num_rows, kSmpThreads, 16 * kSmpThreads * 8, st>>>(p);
        MSTAR_CUDA_OK(cudaGetLastError());
    }
    launch_count_add(1);
    if (flags & MSTAR_FLAG_SAMPLE_ADVANCE_STEP) {
        sample_advance_kernel<<<1, 1, 0, st>>>(step);
        MSTAR_CUDA_OK(cudaGetLastError());
        launch_count_add(1);
    }
    return MSTAR_OK;
}
