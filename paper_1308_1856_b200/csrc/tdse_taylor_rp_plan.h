// tdse_taylor_rp_plan.h -- host-side plan of the persistent register-patch kernel (tdse_taylor_rp.cuh): which
// instantiation, tile geometry and grid a (grid, order) pair runs with.  Plain C++ (no device code) so that the API
// translation unit does not have to compile the kernels.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "tdse_device.cuh"

namespace tdse {

constexpr int kRpRows = 4;     // patch rows

struct RpVariant { int cp, nwr, nwc, minb; };
// instantiations: (patch columns, row-group warps, column-segment warps, min CTAs/SM); 16 points per thread
constexpr RpVariant kRpVariants[] = {
    {4, 1, 1, 8}, {4, 2, 1, 4}, {4, 4, 1, 2}, {4, 8, 1, 1},      // 128-column tiles, 4 / 8 / 16 / 32 rows
    {4, 4, 2, 1},                                                // 256-column tile (edge exchange between warps), 16 rows
    // 8 points per thread, 128-column tiles of two warps, 4 / 8 / 16 rows: only for the multi-step launches of small
    // grids (persist > 1), whose step time is the latency of one warp's sweep -- half the patch, about half the sweep
    {2, 1, 2, 4}, {2, 2, 2, 2}, {2, 4, 2, 1},
};
constexpr int kNumRpVariants = sizeof(kRpVariants) / sizeof(kRpVariants[0]);
// the instantiations that also exist as cluster kernels (16 rows per CTA)
constexpr bool rp_clusterable(int variant) { return variant == 2 || variant == 4; }
// ... and as fused-RK4 / imaginary-time kernels (one-warp-wide tiles)
constexpr bool rp_rk_capable(int variant) { return variant >= 0 && variant <= 3; }
// ... and those that exist only as multi-step (PERSIST) kernels
constexpr bool rp_persist_only(int variant) { return variant >= 5; }

// rk = kernel MODE (0 Taylor, 1 classic RK4, 2 imaginary time); cl: CTAs per cluster (1: none)
struct RpPlan { int ok, variant, tma, cl, rk, W, H, WT, n_tiles, n_items, grid, threads, persist; };     // persist: steps per launch (0: one)

bool tma_available();       // cuTensorMapEncodeTiled could be resolved (tdse_api.cu)

// use_tma: -1 heuristic, 0 never, 1 whenever the layout allows it (n_r % 8 == 0 and more than one tile)
// rk: plan the fused RK4 / imaginary-time step (only the one-warp-wide instantiations, full tiles)
// persist = k > 1: temporal blocking across steps: the halo covers k steps (H = k x order x hw), so one launch takes up to
// k steps with psi in registers (Taylor in real time, full tiles, direct loads, no cluster); kept only while the interior
// of a tile stays at least half of it
inline RpPlan rp_plan(const tdse_grid &g, int order, int n_sm, int force_variant, int use_tma, int rk = 0, int persist = 0) {
    if (persist > 1 && rk != 0) persist = 0;
    RpPlan best{};
    const int hw = (g.fd_order == 3) ? 1 : 2;
    double best_cost = 0.0;
    for (int i = 0; i < kNumRpVariants; ++i) {
        if (force_variant >= 0 && i != force_variant) continue;
        const RpVariant &v = kRpVariants[i];
        const int WT = 32 * v.cp * v.nwc;
        if (rk && (!rp_rk_capable(i) || g.n_r < WT)) continue;
        if (rp_persist_only(i) && persist <= 1) continue;
        int rows = kRpRows * v.nwr, cl = 1;
        if (persist > 1 && (rows < g.n_l || g.n_r <= WT)) continue;
        if (rows < g.n_l) {
            // more rows than one CTA holds: split them over a cluster of 2, 4 or 8 CTAs (16-row CTAs only)
            if (!rp_clusterable(i)) continue;
            while (cl < 8 && rows * cl < g.n_l) cl *= 2;
            if (rows * cl < g.n_l) continue;
            rows *= cl;
        }
        if (rows >= 2 * g.n_l && v.nwr > 1) continue;      // more than half of the rows would be padding
        for (int tma = 0; tma <= 1; ++tma) {
            const bool tma_ok = !(g.n_r & 7) && g.n_r > WT && tma_available();
            if (tma && (use_tma == 0 || !tma_ok || persist > 1)) continue;
            if (!tma && use_tma == 1 && tma_ok && persist <= 1) continue;
            int H = order * hw * (persist > 1 ? persist : 1);
            if (tma) H = (H + 7) & ~7;                      // tile starts on a 128-byte column group
            else if ((g.n_r & 1) == 0) H = (H + 1) & ~1;    // even halo: every patch row starts 32-byte aligned
            RpPlan p{};
            p.variant = i; p.tma = tma; p.cl = cl; p.rk = rk; p.H = H; p.WT = WT; p.threads = 32 * v.nwr * v.nwc;
            p.persist = persist > 1 ? persist : 0;
            if (g.n_r <= WT) { p.W = g.n_r; p.n_tiles = 1; }
            else {
                p.W = WT - 2 * H;
                if (p.W < (persist > 1 ? WT / 2 : WT / 4)) continue;
                p.n_tiles = (g.n_r + p.W - 1) / p.W;
            }
            p.n_items = p.n_tiles * g.batch;
            p.grid = std::min(p.n_items, n_sm * v.minb / cl);       // clusters (= CTAs when cl == 1)
            // a grid that is a multiple of n_tiles keeps every CTA on one radial tile (coefficients loaded once)
            if (p.n_tiles * 4 <= p.grid) p.grid = p.grid / p.n_tiles * p.n_tiles;
            p.grid *= cl;
            p.ok = 1;
            // cost ~ time: the points one CTA computes per item times the items an SM has to work through (at least
            // one: a small grid is bound by the serial work of a CTA, so more and smaller CTAs win).  Measured
            // penalties: tiles wider than one warp 1.4x (edge columns through shared memory, no work before the
            // barrier); cluster barriers 1.25x; the asynchronous tile fetch hides the load latency of the next item.
            const double n_ctas = (double)p.n_items * cl;
            double cost = (double)(rows / cl) * WT * std::max(1.0, n_ctas / n_sm);
            if (force_variant < 0 && v.nwc > 1) cost *= 1.4;
            if (persist > 1) cost *= v.cp / 4.0;            // latency-bound: the sweep of one warp scales with its patch
            if (cl > 1) cost *= 1.25;
            // (a state that stays in L2 gains less from the prefetch than it loses to the halo rounded up to 8 columns:
            // CFG3 62.1 us per step with direct loads, 88 interior columns, against 63.1 us with TMA tiles, 80)
            const bool l2_resident = 2.0 * 16.0 * (double)g.n_r * g.n_l * g.batch < 100e6;
            if (tma) cost *= l2_resident ? 0.93 : 0.85;
            if (!best.ok || cost < best_cost) { best = p; best_cost = cost; }
        }
    }
    return best;
}

// Observables fused into the last pass of a step (row a6; P:371 column list, "not performed asynchronously"):
// norm, the l / l+1 products of <z> (Eq. 34) and <z''> (Eq. 36) and up to kRpObsStates bound-state overlaps
// (Eq. 25) are reduced from the registers that hold psi(t + dt); one partial per work item (and cluster rank), the
// last CTA to finish adds them per member in a fixed order and writes the row.
constexpr int kRpObsStates = 4;
constexpr int kRpObsRed = 3 + 2 * kRpObsStates;
struct RpObs {
    const Ctl *ctl; const tdse_pulse *pulse;
    const double *phi; const int *l_of_state; int n_states;
    int step_off;                   // the step of the captured block this launch is
    double *partials;               // [n_items * cluster size][kRpObsRed]
    unsigned int *counter;          // zero before the launch; reset by the last CTA
    double *rows;                   // [rows][batch][3 + n_states]
};

// can the plan reduce the observable row in its own store phase (full tiles, real time, few bound states)?
inline bool rp_obs_capable(const RpPlan &p, const tdse_grid &g, int n_states) {
    return p.ok && p.rk != 2 && g.n_r >= p.WT && n_states <= kRpObsStates;
}
// doubles of partial sums the fused observables need
inline size_t rp_obs_partials(const RpPlan &p) { return (size_t)p.n_items * p.cl * kRpObsRed * (p.persist > 1 ? p.persist : 1); }

// defined in tdse_taylor_rp_fd3.cu / tdse_taylor_rp_fd5.cu
int rp_init_fd3();          // uploads the 1/k table of that translation unit to the current device (tdse_create)
int rp_init_fd5();
int launch_taylor_rp_fd3(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                         const double *dtp, int order, cudaStream_t s, const RpObs *ob, int n_steps);
int launch_taylor_rp_fd5(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                         const double *dtp, int order, cudaStream_t s, const RpObs *ob, int n_steps);

// n_steps > 1 only with a persistent plan (ef then holds n_steps x batch field values)
inline int launch_taylor_rp(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                            const double *dtp, int order, cudaStream_t s, const RpObs *ob = nullptr, int n_steps = 1) {
    return g.fd == 3 ? launch_taylor_rp_fd3(g, p, in, out, ef, dtp, order, s, ob, n_steps)
                     : launch_taylor_rp_fd5(g, p, in, out, ef, dtp, order, s, ob, n_steps);
}

}  // namespace tdse
