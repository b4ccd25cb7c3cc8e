// Instantiations and launch of the persistent Dormand-Prince kernel (tdse_rk45_persist.cuh).
#include "tdse_rk45_persist.cuh"
#include "tdse_tma.cuh"

namespace tdse {

template <int FD, bool VG, bool KREG, bool FIXED>
static int rkp_launch_f(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    static DeviceOnce once;
    auto kern = rk45_persist_kernel<FD, VG, KREG, FIXED>;
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

template <int FD, bool VG, bool KREG>
static int rkp_launch(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    if (a.fixed) return rkp_launch_f<FD, VG, KREG, true>(a, p, s);
    if (a.n_stage != 7) return TDSE_ERR_UNSUPPORTED;        // (the adaptive instantiation is Dormand-Prince's seven stages)
    return rkp_launch_f<FD, VG, KREG, false>(a, p, s);
}

// CTAs of this instantiation that can be resident at once on the current device (0: error)
template <int FD, bool VG, bool KREG>
static int rkp_resident(const RkpPlan &p) {
    auto kern = rk45_persist_kernel<FD, VG, KREG, false>;      // (the fixed-step instantiation needs no more than this one)
    if (cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kRkpMaxSmem) != cudaSuccess) return 0;
    int dev = 0, n_sm = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)kern, kRkpThreads, (size_t)p.smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return per_sm * n_sm;
}

template <int FD, bool VG>
static int rkp_launch_k(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    return p.kreg ? rkp_launch<FD, VG, true>(a, p, s) : rkp_launch<FD, VG, false>(a, p, s);
}

// can the grid of the plan be co-resident (what the hand-shakes between CTAs need)?  Else the caller runs stage by stage.
bool rk45_persist_fits(int fd, int gauge, const RkpPlan &p) {
    int n = 0;
    if (fd == 3) n = gauge == 1 ? (p.kreg ? rkp_resident<3, true, true>(p) : rkp_resident<3, true, false>(p))
                                : (p.kreg ? rkp_resident<3, false, true>(p) : rkp_resident<3, false, false>(p));
    else n = gauge == 1 ? (p.kreg ? rkp_resident<5, true, true>(p) : rkp_resident<5, true, false>(p))
                        : (p.kreg ? rkp_resident<5, false, true>(p) : rkp_resident<5, false, false>(p));
    return n >= p.G;
}

int launch_rk45_persist(const RkpArgs &a, const RkpPlan &p, cudaStream_t s) {
    const bool vg = a.g.gauge == 1;
    if (a.g.fd == 3) return vg ? rkp_launch_k<3, true>(a, p, s) : rkp_launch_k<3, false>(a, p, s);
    return vg ? rkp_launch_k<5, true>(a, p, s) : rkp_launch_k<5, false>(a, p, s);
}

}  // namespace tdse
