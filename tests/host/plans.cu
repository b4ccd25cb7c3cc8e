// Host-side test aid (CPU suite): prints the plans of the register-patch kernel and of the persistent Runge-Kutta kernel
// for the grids given on the command line (n_r n_l fd batch order persist, repeated).  No device is touched.
#include <cstdio>
#include <cstdlib>

#include "tdse_rk45_persist.cuh"
#include "tdse_taylor_rp_plan.h"

namespace tdse { bool tma_available() { return true; } }
using namespace tdse;

int main(int argc, char **argv) {
    for (int i = 1; i + 5 < argc; i += 6) {
        tdse_grid g{};
        g.n_r = atoi(argv[i]); g.dr = 0.1; g.n_l = atoi(argv[i + 1]); g.fd_order = atoi(argv[i + 2]); g.gauge = 0;
        g.z_nuc = 1.0; g.batch = atoi(argv[i + 3]);
        const int order = atoi(argv[i + 4]), persist = atoi(argv[i + 5]);
        const RpPlan p = rp_plan(g, order, 148, -1, -1, 0, persist);
        const RkpPlan q = rkp_plan(g, 148, kRkpMaxSmem);
        printf("%d %d %d %d %d %d %d %d %d %d %d %d %d %d %d %d %d %d %d\n", p.ok, p.variant, p.tma, p.cl, p.W, p.H, p.WT, p.n_tiles,
               p.n_items, p.grid, p.threads, p.persist, q.ok, q.G, q.Wc, q.R, q.pitch, q.smem, q.kreg);
    }
    return 0;
}
