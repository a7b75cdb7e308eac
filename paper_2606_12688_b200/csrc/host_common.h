// host_common.h -- host-side helpers shared by the launchers: status plumbing, launch counting,
// argument checks and the TMA tensor-map cache for the K/V pools.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/mstar_attn.h"

namespace mstar {

// thread-local count of kernels the current API call has enqueued
void launch_count_reset();
void launch_count_add(int n);

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// Validates the pool geometry common to all entry points.  Returns MSTAR_OK or a negative status.
int check_pool(const mstar_kv_pool* pool);
// The same for a quantised (one byte per element) pool: head_dim 128 only, strides multiples of 16.
int check_pool_fp8(const mstar_kv_pool* pool);

// One tensor map per pool tensor: 4-D view (D, page_size, Hkv, num_pages) of bf16 with a
// (64, page_size, 1, 1) box and 128-B swizzle, so that a (page, kv head, 64-column half) slab lands in
// shared memory as page_size rows of 128 B, conflict-free for ldmatrix.  Cached per
// (pointer, geometry); thread-safe.  A tensor map encodes a (unified) virtual address and a geometry, nothing of
// the device that owns the memory, so the cache needs no device key.
struct PoolMaps {
    CUtensorMap k;
    CUtensorMap v;
};
int get_pool_maps(const mstar_kv_pool* pool, PoolMaps* out);
// Quantised pool: 4-D view (D, page_size, Hkv, num_pages) of bytes with a (128, page_size, 1, 1) box and 128-B
// swizzle: a (page, kv head) slab lands as page_size rows of 128 B, one row per token.
int get_pool_maps_fp8(const mstar_kv_pool* pool, PoolMaps* out);

// 3-D view (D, Hq, total_rows) of a contiguous [rows][Hq][D] bf16 tensor with a (64, 1, box_rows) box,
// 128-B swizzle.  Not cached (cheap, pointer changes every call).
int make_rows_map(const void* base, int64_t rows, int32_t num_heads, int32_t head_dim, int32_t box_rows,
                  CUtensorMap* out);

// tcgen05 / TMEM prefill kernel (prefill_umma.cu); head_dim 128, or 64 on a bf16 pool
int launch_prefill_umma(const PoolMaps& maps, const void* q, int32_t total_q, const int32_t* cu_seqlens_q,
                        const int32_t* block_table, int64_t bt_stride, const int32_t* seq_lens, int32_t S,
                        int32_t Hq, int32_t Hkv, int32_t page_size, int32_t max_q_len, float scale, int32_t causal,
                        void* out, float* lse, int32_t out_f32, int32_t reuse_plan, void* workspace,
                        size_t workspace_bytes, cudaStream_t stream, int32_t kv_f16 = 0, int32_t head_dim = 128);
size_t prefill_umma_workspace_bytes(int32_t num_seqs, int32_t total_q, int32_t num_q_heads);

// Properties of the CURRENT device (cudaGetDevice), cached per device ordinal; thread-safe.
int device_sm_count();
int device_max_smem_optin();
int current_device();

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: one flag bit per device ordinal and kernel
// instantiation (devices >= 64 set the attribute on every call).
struct PerDeviceOnce {
    unsigned long long done = 0;
};
bool per_device_test(PerDeviceOnce& once, int dev);
void per_device_mark(PerDeviceOnce& once, int dev);
template <typename Kernel>
inline cudaError_t set_max_dynamic_smem(PerDeviceOnce& once, Kernel kernel, int bytes) {
    const int dev = current_device();
    if (per_device_test(once, dev)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) per_device_mark(once, dev);
    return e;
}

#define MSTAR_CUDA_OK(expr)                         \
    do {                                            \
        cudaError_t e__ = (expr);                   \
        if (e__ != cudaSuccess) {                   \
            (void)cudaGetLastError();               \
            return MSTAR_ERR_CUDA;                  \
        }                                           \
    } while (0)

}  // namespace mstar
