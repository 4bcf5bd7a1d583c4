// Tensor-map (TMA) staging of y tiles: host-side descriptor construction and the device-side issue / wait wrappers.
//
// north_star item (3): "a y-axis FFT done as TMA-staged tile transposes".  Where it is used and why: pp_ypass.cuh,
// ypass_*_tma_kernel.  A tile of T double2 columns x N rows of one z plane is fetched by the copy engine as boxes of
// 256 rows x T*16 bytes straight into the CTA's shared-memory tile -- no load instruction, no L1 tag lookup per row
// segment, no address arithmetic in the threads.  The Makhoul permutation of the cosine / sine transforms
// is expressed in the descriptors themselves: one view of the array holds its even rows
// (row stride 2 * pitch), one its odd rows, so the permuted sequence lands as two ascending runs.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>

namespace pp {

// ---- host ---------------------------------------------------------------------------------------------------
typedef CUresult (*pp_encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                       const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                       CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point query: no link-time dependency on libcuda
inline pp_encode_tiled_fn tma_encode_fn() {
    static pp_encode_tiled_fn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return (pp_encode_tiled_fn)p;
    }();
    return fn;
}

// View of the spectral array w[nz][N][nxh] (double2) as a rank-3 tensor of doubles (x, row, plane) holding the rows
// row0, row0 + rstep, ... (nrows of them) of every plane; box = T double2 columns x box_rows rows x 1 plane.
inline bool tma_make_rows_map(CUtensorMap *map, const double2 *w, int nxh, int N, int nz, int row0, int rstep, int nrows,
                              int T, int box_rows) {
    pp_encode_tiled_fn enc = tma_encode_fn();
    if (!enc) return false;
    const cuuint64_t pitch = (cuuint64_t)nxh * sizeof(double2);
    const cuuint64_t dims[3] = {(cuuint64_t)nxh * 2, (cuuint64_t)nrows, (cuuint64_t)nz};
    const cuuint64_t strides[2] = {pitch * (cuuint64_t)rstep, pitch * (cuuint64_t)N};
    const cuuint32_t box[3] = {(cuuint32_t)(2 * T), (cuuint32_t)box_rows, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    void *base = (void *)(w + (size_t)row0 * nxh);
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// ---- device -------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned phase) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(a), "r"(phase) : "memory");
}
// box at coordinates (x in doubles, row of the view, plane) -> shared memory, completion counted on `bar`
__device__ __forceinline__ void tma_load_3d(void *smem_dst, const CUtensorMap *map, int x, int row, int plane, uint64_t *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::
                     "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(map), "r"(x), "r"(row), "r"(plane),
                 "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}

// shared memory -> box at the same coordinates (bulk async group of the issuing thread)
__device__ __forceinline__ void tma_store_3d(const CUtensorMap *map, int x, int row, int plane, const void *smem_src) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(map), "r"(x), "r"(row), "r"(plane),
                 "r"((unsigned)__cvta_generic_to_shared(smem_src))
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit_and_wait_read() {
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
// generic-proxy writes to shared memory made visible to the copy engine (every writing thread, before the barrier)
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace pp
