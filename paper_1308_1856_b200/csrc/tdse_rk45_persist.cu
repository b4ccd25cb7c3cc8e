// Instantiations and launch of the persistent Dormand-Prince kernel (tdse_rk45_persist.cuh).
#include <cstdio>
#include "tdse_rk45_persist.cuh"
#include "tdse_tma.cuh"

namespace tdse {

template <int FD, bool VG>
static int rkp_launch(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    static DeviceOnce once;
    auto kern = rk45_persist_kernel<FD, VG>;
    if (once.first()) {
        if (cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kRkpMaxSmem) != cudaSuccess)
            return TDSE_ERR_CUDA;
    }
    // every CTA waits for its neighbours: the grid must be co-resident, which a cooperative launch guarantees (or refuses)
    void *args[] = {(void *)&a};
    const cudaError_t le = cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)p.G), dim3(kRkpThreads), args, (size_t)p.smem, s);
    if (le != cudaSuccess) { fprintf(stderr, "rkp launch: %s (G=%d smem=%d)\n", cudaGetErrorString(le), p.G, p.smem); return TDSE_ERR_CUDA; }
    return TDSE_OK;
}

int launch_rk45_persist(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    const bool vg = a.g.gauge == 1;
    if (a.g.fd == 3) return vg ? rkp_launch<3, true>(a, p, s) : rkp_launch<3, false>(a, p, s);
    return vg ? rkp_launch<5, true>(a, p, s) : rkp_launch<5, false>(a, p, s);
}

}  // namespace tdse
