// host_common.cu -- status strings, pool validation, TMA tensor-map creation and cache.
#include <mutex>
#include <vector>

#include "host_common.h"

namespace mstar {

static thread_local int g_launches = 0;
void launch_count_reset() { g_launches = 0; }
void launch_count_add(int n) { g_launches += n; }

int check_pool(const mstar_kv_pool* pool) {
    if (!pool || !pool->k_pool || !pool->v_pool) return MSTAR_ERR_INVALID_ARG;
    if (pool->num_pages <= 0 || pool->num_kv_heads <= 0) return MSTAR_ERR_INVALID_ARG;
    if (pool->page_size != 16 && pool->page_size != 32) return MSTAR_ERR_UNSUPPORTED;
    if (pool->head_dim != 64 && pool->head_dim != 128) return MSTAR_ERR_UNSUPPORTED;
    if (!aligned(pool->k_pool, 128) || !aligned(pool->v_pool, 128)) return MSTAR_ERR_INVALID_ARG;
    if (pool->stride_page <= 0 || pool->stride_head <= 0 || pool->stride_token < pool->head_dim)
        return MSTAR_ERR_INVALID_ARG;
    if (pool->stride_page % 8 || pool->stride_head % 8 || pool->stride_token % 8) return MSTAR_ERR_INVALID_ARG;
    if (pool->num_pages * (int64_t)pool->num_kv_heads * pool->page_size >= (int64_t(1) << 31))
        return MSTAR_ERR_UNSUPPORTED;
    return MSTAR_OK;
}

int check_pool_fp8(const mstar_kv_pool* pool) {
    if (!pool || !pool->k_pool || !pool->v_pool) return MSTAR_ERR_INVALID_ARG;
    if (pool->num_pages <= 0 || pool->num_kv_heads <= 0) return MSTAR_ERR_INVALID_ARG;
    if (pool->page_size != 16 && pool->page_size != 32) return MSTAR_ERR_UNSUPPORTED;
    if (pool->head_dim != 128) return MSTAR_ERR_UNSUPPORTED;
    if (!aligned(pool->k_pool, 128) || !aligned(pool->v_pool, 128)) return MSTAR_ERR_INVALID_ARG;
    if (pool->stride_page <= 0 || pool->stride_head <= 0 || pool->stride_token < pool->head_dim)
        return MSTAR_ERR_INVALID_ARG;
    if (pool->stride_page % 16 || pool->stride_head % 16 || pool->stride_token % 16) return MSTAR_ERR_INVALID_ARG;
    if (pool->num_pages * (int64_t)pool->num_kv_heads * pool->page_size >= (int64_t(1) << 31))
        return MSTAR_ERR_UNSUPPORTED;
    return MSTAR_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            (void)cudaGetLastError();
    });
    return fn;
}

static int encode_pool_map(void* base, const mstar_kv_pool* pool, int elem_bytes, CUtensorMap* out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return MSTAR_ERR_CUDA;
    if (elem_bytes == 1) {
        cuuint64_t dims[4] = {(cuuint64_t)pool->head_dim, (cuuint64_t)pool->page_size,
                              (cuuint64_t)pool->num_kv_heads, (cuuint64_t)pool->num_pages};
        cuuint64_t strides[3] = {(cuuint64_t)pool->stride_token, (cuuint64_t)pool->stride_head,
                                 (cuuint64_t)pool->stride_page};
        cuuint32_t box[4] = {128, (cuuint32_t)pool->page_size, 1, 1};
        cuuint32_t estr[4] = {1, 1, 1, 1};
        CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, base, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        return r == CUDA_SUCCESS ? MSTAR_OK : MSTAR_ERR_INVALID_ARG;
    }
    cuuint64_t dims[4] = {(cuuint64_t)pool->head_dim, (cuuint64_t)pool->page_size, (cuuint64_t)pool->num_kv_heads,
                          (cuuint64_t)pool->num_pages};
    cuuint64_t strides[3] = {(cuuint64_t)pool->stride_token * 2, (cuuint64_t)pool->stride_head * 2,
                             (cuuint64_t)pool->stride_page * 2};
    cuuint32_t box[4] = {64, (cuuint32_t)pool->page_size, 1, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, base, dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? MSTAR_OK : MSTAR_ERR_INVALID_ARG;
}

struct CacheEntry {
    mstar_kv_pool key;
    int elem_bytes;
    PoolMaps maps;
};
static std::mutex g_cache_mu;
static std::vector<CacheEntry> g_cache;

static bool same_pool(const mstar_kv_pool& a, const mstar_kv_pool& b) {
    return a.k_pool == b.k_pool && a.v_pool == b.v_pool && a.num_pages == b.num_pages &&
           a.page_size == b.page_size && a.num_kv_heads == b.num_kv_heads && a.head_dim == b.head_dim &&
           a.stride_page == b.stride_page && a.stride_head == b.stride_head && a.stride_token == b.stride_token;
}

static int pool_maps(const mstar_kv_pool* pool, int elem_bytes, PoolMaps* out);
int get_pool_maps(const mstar_kv_pool* pool, PoolMaps* out) { return pool_maps(pool, 2, out); }
int get_pool_maps_fp8(const mstar_kv_pool* pool, PoolMaps* out) { return pool_maps(pool, 1, out); }

static int pool_maps(const mstar_kv_pool* pool, int elem_bytes, PoolMaps* out) {
    std::lock_guard<std::mutex> lock(g_cache_mu);
    for (const CacheEntry& e : g_cache)
        if (e.elem_bytes == elem_bytes && same_pool(e.key, *pool)) {
            *out = e.maps;
            return MSTAR_OK;
        }
    CacheEntry e;
    e.key = *pool;
    e.elem_bytes = elem_bytes;
    int rc = encode_pool_map(pool->k_pool, pool, elem_bytes, &e.maps.k);
    if (rc != MSTAR_OK) return rc;
    rc = encode_pool_map(pool->v_pool, pool, elem_bytes, &e.maps.v);
    if (rc != MSTAR_OK) return rc;
    if (g_cache.size() >= 64) g_cache.erase(g_cache.begin());
    g_cache.push_back(e);
    *out = e.maps;
    return MSTAR_OK;
}

int make_rows_map(const void* base, int64_t rows, int32_t num_heads, int32_t head_dim, int32_t box_rows,
                  CUtensorMap* out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return MSTAR_ERR_CUDA;
    cuuint64_t dims[3] = {(cuuint64_t)head_dim, (cuuint64_t)num_heads, (cuuint64_t)rows};
    cuuint64_t strides[2] = {(cuuint64_t)head_dim * 2, (cuuint64_t)head_dim * 2 * num_heads};
    cuuint32_t box[3] = {64, 1, (cuuint32_t)box_rows};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? MSTAR_OK : MSTAR_ERR_INVALID_ARG;
}

int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return dev;
}

static std::mutex g_dev_mu;
constexpr int kMaxCachedDevices = 64;

static int device_attr_cached(cudaDeviceAttr attr, int (&cache)[kMaxCachedDevices], int fallback) {
    const int dev = current_device();
    std::lock_guard<std::mutex> lock(g_dev_mu);
    if (dev >= 0 && dev < kMaxCachedDevices && cache[dev] > 0) return cache[dev];
    int v = 0;
    if (cudaDeviceGetAttribute(&v, attr, dev) != cudaSuccess || v <= 0) {
        (void)cudaGetLastError();
        return fallback;
    }
    if (dev >= 0 && dev < kMaxCachedDevices) cache[dev] = v;
    return v;
}

int device_sm_count() {
    static int cache[kMaxCachedDevices] = {};
    return device_attr_cached(cudaDevAttrMultiProcessorCount, cache, 148);
}

int device_max_smem_optin() {
    static int cache[kMaxCachedDevices] = {};
    return device_attr_cached(cudaDevAttrMaxSharedMemoryPerBlockOptin, cache, 227 * 1024);
}

bool per_device_test(PerDeviceOnce& once, int dev) {
    if (dev < 0 || dev >= 64) return false;
    std::lock_guard<std::mutex> lock(g_dev_mu);
    return (once.done >> dev) & 1ull;
}
void per_device_mark(PerDeviceOnce& once, int dev) {
    if (dev < 0 || dev >= 64) return;
    std::lock_guard<std::mutex> lock(g_dev_mu);
    once.done |= 1ull << dev;
}

}  // namespace mstar

extern "C" {

int32_t mstar_last_launch_count(void) { return mstar::g_launches; }

const char* mstar_status_string(int status) {
    switch (status) {
        case MSTAR_OK: return "MSTAR_OK";
        case MSTAR_ERR_INVALID_ARG: return "MSTAR_ERR_INVALID_ARG";
        case MSTAR_ERR_UNSUPPORTED: return "MSTAR_ERR_UNSUPPORTED";
        case MSTAR_ERR_WORKSPACE_TOO_SMALL: return "MSTAR_ERR_WORKSPACE_TOO_SMALL";
        case MSTAR_ERR_CUDA: return "MSTAR_ERR_CUDA";
        default: return "MSTAR_ERR_UNKNOWN";
    }
}

const char* mstar_version(void) { return "0.1.0"; }

}  // extern "C"
