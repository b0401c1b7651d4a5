// tma_utils.cuh -- mbarrier / TMA (cp.async.bulk.tensor) wrappers, tensor-map encoding and the strip decomposition
// shared by the TMA-staged K1 kernels (spin_stencil_tma.cu: one step per pass; spin_cheb2_tma.cu: two steps per pass).
// Product code: shares nothing with oracle/.
#pragma once
#include <atomic>
#include <cuda.h>
#include "common.cuh"

namespace tma {

constexpr int TXMAX = 60;          // strip width (sites); a row box holds 64 sites starting at xb - 2
constexpr int ROWD = 192;          // doubles per main row box of a 3-vector field (64 sites x 3)
constexpr int SIDED = 16;          // doubles per x-wrap side box (128 B)
constexpr int CROWD = 64;          // doubles per main row box of the scalar field c

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}

// first column of strip i (even, so that the 24-byte sites of a box start 16-byte aligned)
__host__ __device__ __forceinline__ int strip_x(int i, int Lx, int nsx) { return 2 * (int)(((long long)i * (Lx >> 1)) / nsx); }

// CTA that owns linearised strip-row idx when `total` strip-rows are split evenly over `grid` CTAs
__device__ __forceinline__ int cta_of(long long idx, long long total, int grid) {
    long long b = idx * grid / total;
    while (b + 1 < (long long)grid && (total * (b + 1)) / grid <= idx) ++b;
    while (b > 0 && (total * b) / grid > idx) --b;
    return (int)b;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn lookup_encode() {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
        return (EncodeTiledFn)f;
    return nullptr;
}
inline EncodeTiledFn get_encode() {
    static const EncodeTiledFn fn = lookup_encode();   // thread-safe one-time initialisation (moto_lowest_modes_batch runs host threads)
    return fn;
}

// field array [nvec][Ly][ncomp Lx] fp64 as a 3-D tensor; box = {inner doubles, rows, 1}
inline bool encode(CUtensorMap* map, const double* base, int Lx, int Ly, int nvec, int inner, int rows, int ncomp = 3) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t gdim[3] = {(cuuint64_t)ncomp * Lx, (cuuint64_t)Ly, (cuuint64_t)nvec};
    cuuint64_t gstr[2] = {(cuuint64_t)8 * ncomp * Lx, (cuuint64_t)8 * ncomp * Lx * Ly};
    cuuint32_t box[3] = {(cuuint32_t)inner, (cuuint32_t)rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) applies per device: remember which devices have it (one bit each),
// safe against the host threads of moto_lowest_modes_batch (setting it twice is harmless).
template <typename Kernel>
inline bool ensure_smem_attr(Kernel kernel, size_t bytes, std::atomic<unsigned long long>& seen) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    const unsigned long long bit = 1ull << (dev & 63);
    if (seen.load(std::memory_order_acquire) & bit) return true;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) return false;
    seen.fetch_or(bit, std::memory_order_release);
    return true;
}

}  // namespace tma
