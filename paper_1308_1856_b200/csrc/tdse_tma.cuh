// tdse_tma.cuh -- TMA (cp.async.bulk.tensor), mbarrier and thread-block-cluster helpers of the sm_100a kernels, and the
// host side of the tensor maps (cuTensorMapEncodeTiled through the runtime's driver entry point: no link against
// libcuda).  Tensor maps are encoded on every launch and handed to the kernel BY VALUE (__grid_constant__), so that
// nothing is cached per pointer and a captured graph owns its copy.  Per-device one-time set-up (function attributes,
// constant tables) goes through DeviceOnce.
#pragma once
#include <cuda.h>

#include <atomic>

#include "tdse_device.cuh"

namespace tdse {

// true exactly once per CUDA device ordinal (< 64) for the object it guards; the caller then performs the set-up for the
// CURRENT device (cudaFuncSetAttribute and __constant__ uploads are per device)
struct DeviceOnce {
    std::atomic<unsigned long long> done{0};
    bool first() {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev > 63) return true;      // unknown: always set up
        const unsigned long long bit = 1ull << dev;
        return (done.fetch_or(bit) & bit) == 0;
    }
};

// ---- TMA (cp.async.bulk.tensor) + mbarrier helpers ---------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    unsigned ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
// 3-D tiled tensor load global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, unsigned long long *bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- thread-block cluster helpers (distributed shared memory) ----------------------------------------------------
__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned cluster_nctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ unsigned dsmem_addr(const void *p, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
    return r;
}
__device__ __forceinline__ double2 ld_dsmem2(unsigned addr) {
    double2 v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
// Cluster barrier, arrive side.  What crosses CTAs here is SHARED memory only (rows published with st.shared, read by
// the neighbouring CTA with ld.shared::cluster after its wait.acquire).  `barrier.cluster.arrive.release` is lowered to
// MEMBAR.ALL.GPU + ERRBAR (it must also cover global memory): 17 % of all stall samples of the CFG3 kernel
// (profiles/r02_README.md).  A CTA-scope fence is enough for the purpose: once the st.shared have been performed with
// respect to the CTA they ARE in the SM's shared-memory array, which is the only copy a remote ld.shared::cluster can
// read; the loads a thread did before arriving have returned their data by then.  CFG3 step: 78.2 -> 64.4 us.  Define
// TDSE_CLUSTER_RELEASE_STRICT for the textbook form.
#ifdef TDSE_CLUSTER_RELEASE_STRICT
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
#else
__device__ __forceinline__ void cluster_arrive() { asm volatile("fence.acq_rel.cta; barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
#endif
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}


__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, int c3,
                                            unsigned long long *bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

// cuTensorMapEncodeTiled through the runtime (no link against libcuda)
typedef CUresult (*TmaEncodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline TmaEncodeTiled tma_encode_fn() {
    static TmaEncodeTiled fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess && p &&
            qres == cudaDriverEntryPointSuccess)
            fn = (TmaEncodeTiled)p;
        cudaGetLastError();
    }
    return fn;
}


// State array seen as [rows = batch*n_l][n_r/8 groups][16 doubles], box = box_rows x box_cols/8 x 16, 128-byte swizzle
// (register-patch kernel: the per-thread patch reads at a 64-byte lane stride are then bank-conflict free).
inline bool tma_map_rows3d(CUtensorMap *m, const void *base, int n_r, int total_rows, int box_rows, int box_cols) {
    const TmaEncodeTiled encode = tma_encode_fn();
    if (!encode) return false;
    const cuuint64_t dims[3] = {16, (cuuint64_t)(n_r / 8), (cuuint64_t)total_rows};
    const cuuint64_t strides[2] = {128, (cuuint64_t)n_r * 16};          // bytes, dims 1 and 2
    const cuuint32_t box[3] = {16, (cuuint32_t)(box_cols / 8), (cuuint32_t)box_rows};
    const cuuint32_t estr[3] = {1, 1, 1};
    return encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// State array seen as [batch][n_l][n_r/8][16 doubles], box = 1 x box_rows x box_cols/8 x 16, no swizzle: everything
// outside a member's index box is zero-filled by the hardware (tile kernels).
inline bool tma_map_member4d(CUtensorMap *m, const void *base, int n_r, int n_l, int batch, int box_rows, int box_cols) {
    const TmaEncodeTiled encode = tma_encode_fn();
    if (!encode) return false;
    const cuuint64_t dims[4] = {16, (cuuint64_t)(n_r / 8), (cuuint64_t)n_l, (cuuint64_t)batch};
    const cuuint64_t strides[3] = {128, (cuuint64_t)n_r * 16, (cuuint64_t)n_r * 16 * (cuuint64_t)n_l};
    const cuuint32_t box[4] = {16, (cuuint32_t)(box_cols / 8), (cuuint32_t)box_rows, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void *>(base), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tdse
