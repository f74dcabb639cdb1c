// mm_runtime.cu — host-side plumbing shared by the entry points: the library's stream-ordered scratch pool and the
// TMA tensor-map encoder (driver entry point fetched at run time: libmm.so does not link libcuda).
#include <cuda.h>
#include <cuda_runtime.h>

#include <stdlib.h>

#include <mutex>
#include <string>

#include "mm_internal.h"

namespace {

// One CUDA memory pool per device, owned by the library.  Device calls take their scratch (the adjoint's split
// operand tiles, the forward's repacked volume) from it with cudaMallocFromPoolAsync on the caller's stream and give
// it back with cudaFreeAsync in stream order: no synchronisation, re-entrant across streams, and the memory stays in
// the pool between calls (release threshold = everything) until mm_workspace_release trims it.
constexpr int MAX_DEV = 64;
std::mutex g_pool_mu;
cudaMemPool_t g_pool[MAX_DEV] = {};

cudaError_t pool_for_current_device(cudaMemPool_t *out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pool[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        e = cudaMemPoolCreate(&g_pool[dev], &props);
        if (e != cudaSuccess) { g_pool[dev] = nullptr; return e; }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(g_pool[dev], cudaMemPoolAttrReleaseThreshold, &keep);
    }
    *out = g_pool[dev];
    return cudaSuccess;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static std::once_flag once;
    static EncodeTiledFn fn = nullptr;
    std::call_once(once, [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    });
    return fn;
}

}  // namespace

// MM_SCRATCH_MALLOC=1 (debugging/profiling only: ncu's kernel replay cannot save and restore pool memory): plain
// cudaMalloc / cudaFree, which synchronise.
static bool scratch_plain() { static const bool v = getenv("MM_SCRATCH_MALLOC") != nullptr; return v; }

cudaError_t mm_scratch_alloc(void **p, size_t bytes, cudaStream_t st)
{
    if (scratch_plain()) return cudaMalloc(p, bytes ? bytes : 16);
    cudaMemPool_t pool;
    cudaError_t e = pool_for_current_device(&pool);
    if (e != cudaSuccess) return e;
    return cudaMallocFromPoolAsync(p, bytes ? bytes : 16, pool, st);
}

cudaError_t mm_scratch_free(void *p, cudaStream_t st)
{
    if (!p) return cudaSuccess;
    if (scratch_plain()) { cudaStreamSynchronize(st); return cudaFree(p); }
    return cudaFreeAsync(p, st);
}

void mm_scratch_trim()
{
    std::lock_guard<std::mutex> lock(g_pool_mu);
    for (int d = 0; d < MAX_DEV; d++)
        if (g_pool[d]) cudaMemPoolTrimTo(g_pool[d], 0);
}

bool mm_tma_available() { return encode_tiled_fn() != nullptr; }

// fp32 tensor [n3][n2][n1][n0] (n0 innermost, dense), box [b3][b2][b1][b0]; out-of-bounds reads give 0.  swizzle = 0, 32,
// 64 or 128 bytes: the box lands in shared memory with that swizzle (the low log2(swizzle/16) bits of the 16-byte chunk
// index are XORed with the same number of bits of the 128-byte row index); swizzle must equal b0 * 4 here.
bool mm_tma_encode_4d_f32(void *tmap_out, const void *base, const unsigned long long n[4], const unsigned b[4], int swizzle)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[4] = {n[0], n[1], n[2], n[3]};
    cuuint64_t strides[3] = {n[0] * 4ull, n[0] * n[1] * 4ull, n[0] * n[1] * n[2] * 4ull};
    cuuint32_t box[4] = {b[0], b[1], b[2], b[3]};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = fn((CUtensorMap *)tmap_out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<void *>(base), dims, strides, box,
                          estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          swizzle == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                                         : swizzle == 32 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        mm_set_error("cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r));
        return false;
    }
    return true;
}
