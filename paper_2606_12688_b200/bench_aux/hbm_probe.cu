// hbm_probe.cu -- measurement aid, NOT part of the product library: built into its own
// libmstar_benchaux.so, which only bench.py loads.  A read-only streaming kernel, the practical HBM-read ceiling
// that bench.py reports beside the decode kernel's rate.  Sums a buffer as 32-bit words with 16-byte streaming loads
// (ld.global.nc.L1::no_allocate), 8 loads in flight per thread, grid = 8 blocks of 256 threads per SM.
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace mstar_benchaux {

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

}  // namespace mstar_benchaux

// Streams `bytes` bytes (multiple of 16, 16-B aligned, device) through 16-byte read-only loads and adds the wrapping
// sum of their 32-bit words to *sum_out (device, may be NULL; not zeroed).  0 = enqueued, -1 = bad argument, -4 = CUDA.
extern "C" int mstar_benchaux_hbm_read_probe(const void* buf, size_t bytes, unsigned long long* sum_out, void* stream) {
    if (!buf || (reinterpret_cast<uintptr_t>(buf) % 16) || bytes % 16) return -1;
    if (bytes == 0) return 0;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return -4;
    }
    mstar_benchaux::hbm_read_probe_kernel<<<sms * 8, 256, 0, (cudaStream_t)stream>>>(
        reinterpret_cast<const int4*>(buf), (int64_t)(bytes / 16), sum_out);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}
