// sampling.cu -- mstar_sample_tokens: CUDA-graph-compatible token sampling (last clause;
// PAPER.md:134 "a cuda-graph-compatible sampling plugin", :230; definition: DESIGN.md R28, oracle/sampling.py).
//
// One CTA per row of logits.  Everything after the exponential is INTEGER arithmetic, so the result does not depend on
// the order in which threads add: token weights are fixed-point, w_i = floor(2^32 * 2^((z_i - z_max) log2 e)), sums are
// 64-bit integers, the uniform number is the 64-bit fraction (x + 1/2) / 2^32 of a Philox4x32-10 word and the running
// sum is inverted in index order.  No state on the host: seeds and the step counter are device memory, so a replayed
// CUDA graph draws fresh numbers (MSTAR_FLAG_SAMPLE_ADVANCE_STEP adds 1 to the counter behind the sampling kernel).
//
// Passes over the row (all L2 hits after the first): maximum / argmax; [top-k: 8 radix-select passes on the order-
// preserving integer image of z, 4 bits each, counting]; total weight; [top-p: 8 radix-select passes, weighing; total
// weight of the nucleus]; weight per warp segment; scan of the one segment that holds the target.  A radix-select
// pass keeps one private 16-bin histogram per thread in shared memory (no atomics) and reduces it afterwards.
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

// order-preserving map float -> uint32 (larger float, larger key; -0 < +0)
__device__ __forceinline__ uint32_t order_key(float z) {
    const uint32_t b = __float_as_uint(z);
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

__global__ void sample_advance_kernel(uint64_t* step) { *step += 1; }

}  // namespace mstar

extern "C" int mstar_sample_tokens(int32_t* tokens_out, const void* logits, int64_t row_stride, int32_t num_rows,
                                   int32_t vocab, const float* temperature, const int32_t* top_k, const float* top_p,
                                   const uint64_t* seeds, uint64_t* step, uint32_t flags, void* stream) {
    using namespace mstar;
    launch_count_reset();
    if (flags & ~(MSTAR_FLAG_LOGITS_BF16 | MSTAR_FLAG_SAMPLE_ADVANCE_STEP)) return MSTAR_ERR_INVALID_ARG;
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
    static PerDeviceOnce once;
    MSTAR_CUDA_OK(set_max_dynamic_smem(once, sample_tokens_kernel, 16 * kSmpThreads * 8));
    sample_tokens_kernel<<<(unsigned)num_rows, kSmpThreads, 16 * kSmpThreads * 8, st>>>(p);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    if (flags & MSTAR_FLAG_SAMPLE_ADVANCE_STEP) {
        sample_advance_kernel<<<1, 1, 0, st>>>(step);
        MSTAR_CUDA_OK(cudaGetLastError());
        launch_count_add(1);
    }
    return MSTAR_OK;
}
