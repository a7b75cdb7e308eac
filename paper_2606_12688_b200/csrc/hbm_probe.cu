// hbm_probe.cu -- measurement aid: a read-only streaming kernel, the practical HBM-read ceiling that
// bench.py reports beside the decode kernel's rate.  Sums a buffer as 32-bit words with 16-byte streaming loads
// (ld.global.nc.L1::no_allocate), 8 loads in flight per thread, grid = 8 blocks of 256 threads per SM.
#include "host_common.h"

namespace mstar {

__global__ void __launch_bounds__(256) hbm_read_probe_kernel(const int4* __restrict__ src, int64_t n_vec,
                                                             unsigned long long* __restrict__ out) {
    constexpr int UNROLL = 8;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    unsigned int acc = 0;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < n_vec; i0 += stride * UNROLL) {
        int4 v[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int64_t i = i0 + u * stride;
            v[u] = make_int4(0, 0, 0, 0);
            if (i < n_vec)
                asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];"
                             : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w)
                             : "l"(src + i));
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) acc += (unsigned)v[u].x + (unsigned)v[u].y + (unsigned)v[u].z + (unsigned)v[u].w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0 && out) atomicAdd(out, (unsigned long long)acc);
}

}  // namespace mstar

extern "C" int mstar_hbm_read_probe(const void* buf, size_t bytes, unsigned long long* sum_out, void* stream) {
    using namespace mstar;
    launch_count_reset();
    if (!buf || !aligned(buf, 16) || bytes % 16) return MSTAR_ERR_INVALID_ARG;
    if (bytes == 0) return MSTAR_OK;
    const int blocks = device_sm_count() * 8;
    hbm_read_probe_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<const int4*>(buf),
                                                                   (int64_t)(bytes / 16), sum_out);
    MSTAR_CUDA_OK(cudaGetLastError());
    launch_count_add(1);
    return MSTAR_OK;
}
