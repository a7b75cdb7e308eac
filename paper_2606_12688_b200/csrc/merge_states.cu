// merge_states.cu -- log-sum-exp merge of two normalised attention states (shared-prefix
// "cascade" decode for CFG branches: "three labels over a single paged KV pool ... by-reference").
// The branches of a request share the physical pages of their common prefix; a cascade reads those pages once:
//   pass A  one decode call over the shared prefix with the branches' queries stacked as extra grouped heads
//           (q row = [request][kv head][branch][g], so Hq' = B * Hq and the same kv-head map h div G' applies),
//   pass B  one decode call over each branch's private suffix (block table advanced past the prefix pages),
//   merge   out = (e^{lse_a - M} out_a + e^{lse_b - M} out_b) / (e^{lse_a - M} + e^{lse_b - M}), M = max(lse_a, lse_b),
//           lse = M + ln(...): the combine formula of step a3 with l = 1 (oracle: COMBINE).
// One warp per output row; fp32 states in (MSTAR_FLAG_OUT_F32 outputs of the two passes), bf16 or fp32 out.
#include <cuda_bf16.h>

#include "host_common.h"
#include "ptx.cuh"

namespace mstar {

template <int D>
__global__ void __launch_bounds__(128) merge_states_kernel(const float* __restrict__ out_a,
                                                           const float* __restrict__ lse_a,
                                                           const int32_t* __restrict__ row_map_a,
                                                           const float* __restrict__ out_b,
                                                           const float* __restrict__ lse_b, int64_t n_rows,
                                                           void* __restrict__ out, float* __restrict__ lse_out,
                                                           int32_t out_f32) {
    constexpr int VEC = D / 32;
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (row >= n_rows) return;
    const int64_t ra = row_map_a ? (int64_t)__ldg(row_map_a + row) : row;
    const float la = __ldg(lse_a + ra), lb = __ldg(lse_b + row);
    const float M = fmaxf(la, lb);
    // natural-log LSEs; an empty state has lse = -inf and weight 0
    const float wa = (la == -INFINITY) ? 0.f : __expf(la - M);
    const float wb = (lb == -INFINITY) ? 0.f : __expf(lb - M);
    const float z = wa + wb;
    const float inv = z > 0.f ? 1.f / z : 0.f;
    float acc[VEC];
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
        const float a = wa > 0.f ? __ldg(out_a + ra * D + lane * VEC + i) : 0.f;
        const float b = wb > 0.f ? __ldg(out_b + row * D + lane * VEC + i) : 0.f;
        acc[i] = (wa * a + wb * b) * inv;
    }
    if (out_f32) {
        float* o = reinterpret_cast<float*>(out) + row * D + lane * VEC;
#pragma unroll
        for (int i = 0; i < VEC; ++i) o[i] = acc[i];
    } else {
        __nv_bfloat16* o = reinterpret_cast<__nv_bfloat16*>(out) + row * D + lane * VEC;
#pragma unroll
        for (int i = 0; i < VEC; i += 2) *reinterpret_cast<uint32_t*>(o + i) = pack_bf16x2(acc[i], acc[i + 1]);
    }
    if (lse_out && lane == 0) lse_out[row] = z > 0.f ? M + __logf(z) : -INFINITY;
}

}  // namespace mstar

extern "C" int mstar_merge_attn_states(void* out, float* lse_out, const float* out_a, const float* lse_a,
                                       const int32_t* row_map_a, const float* out_b, const float* lse_b,
                                       int64_t num_rows, int32_t head_dim, uint32_t flags, void* stream) {
    using namespace mstar;
    launch_count_reset();
    if (flags & ~MSTAR_FLAG_OUT_F32) return MSTAR_ERR_INVALID_ARG;
    if (num_rows < 0 || (head_dim != 64 && head_dim != 128)) return MSTAR_ERR_INVALID_ARG;
    if (num_rows == 0) return MSTAR_OK;
    if (!out || !out_a || !lse_a || !out_b || !lse_b) return MSTAR_ERR_INVALID_ARG;
    if (!aligned(out, 16) || !aligned(out_a, 16) || !aligned(out_b, 16)) return MSTAR_ERR_INVALID_ARG;
    const unsigned blocks = (unsigned)((num_rows + 3) / 4);
    const int f32 = (flags & MSTAR_FLAG_OUT_F32) ? 1 : 0;
    if (head_dim == 128)
        merge_states_kernel<128><<<blocks, 128, 0, (cudaStream_t)stream>>>(out_a, lse_a, row_map_a, out_b, lse_b,
                                                                           num_rows, out, lse_out, f32);
    else
        merge_states_kernel<64><<<blocks, 128, 0, (cudaStream_t)stream>>>(out_a, lse_a, row_map_a, out_b, lse_b,
                                                                          num_rows, out, lse_out, f32);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}
