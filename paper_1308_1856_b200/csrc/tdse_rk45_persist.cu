// Instantiations and launch of the persistent Dormand-Prince kernel (tdse_rk45_persist.cuh).
#include "tdse_rk45_persist.cuh"
#include "tdse_tma.cuh"

namespace tdse {

template <int FD, bool VG, bool KREG>
static int rkp_launch(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    static DeviceOnce once;
    auto kern = rk45_persist_kernel<FD, VG, KREG>;
    if (once.first()) {
        if (cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kRkpMaxSmem) != cudaSuccess)
            return TDSE_ERR_CUDA;
    }
    // every CTA waits for its neighbours: the grid must be co-resident, which a cooperative launch guarantees (or refuses)
    void *args[] = {(void *)&a};
    if (cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)p.G), dim3(kRkpThreads), args, (size_t)p.smem, s) !=
        cudaSuccess) {
        cudaGetLastError();
        return TDSE_ERR_CUDA;
    }
    return TDSE_OK;
}

template <int FD, bool VG>
static int rkp_launch_k(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    return p.kreg ? rkp_launch<FD, VG, true>(a, p, s) : rkp_launch<FD, VG, false>(a, p, s);
}

int launch_rk45_persist(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    const bool vg = a.g.gauge == 1;
    if (a.g.fd == 3) return vg ? rkp_launch_k<3, true>(a, p, s) : rkp_launch_k<3, false>(a, p, s);
    return vg ? rkp_launch_k<5, true>(a, p, s) : rkp_launch_k<5, false>(a, p, s);
}

}  // namespace tdse
