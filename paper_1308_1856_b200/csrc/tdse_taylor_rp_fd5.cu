// tdse_taylor_rp_fd5.cu -- the 5-point instantiations of the persistent register-patch kernel (own translation unit
// so that the library builds in parallel).
#include "tdse_taylor_rp.cuh"

namespace tdse {
int rp_init_fd5() { return rp_init_tables<5>(); }
int launch_taylor_rp_fd5(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                         const double *dtp, int order, cudaStream_t s, const RpObs *ob, int n_steps) {
    return launch_taylor_rp_fd<5>(g, p, in, out, ef, dtp, order, s, ob, n_steps);
}
}  // namespace tdse
