// tdse_taylor_rp.cuh -- temporally blocked Taylor step, v3: persistent CTAs on register patches.
//
// Method: Eq. 37 (reading R-G6): F(t+dt) = sum_{k=0..P} F^(k), F^(k) = (-i dt/k) H F^(k-1); all P orders of a
// step are applied in ONE pass over HBM (32 B/point/step; the paper launches one kernel per order).
//
// Work item = (member b, radial tile t).  A CTA is NWR x NWC warps; a warp owns 4 partial waves x 32*CP radial
// columns, a thread a patch of 4 rows x CP adjacent columns (CP = 2 or 4) whose current term u_k AND accumulator
// stay in registers for the whole step.  What differs from v2 (tdse_taylor_rt.cuh):
//   * no shared-memory tile: a thread loads its patch straight from global memory (CP*16 contiguous bytes per
//     row, 256-bit accesses when aligned; a warp reads 32*CP*16 contiguous bytes) and stores the result likewise;
//   * radial neighbours come from the adjacent LANES by warp shuffle; only the l-1 / l+1 rows (and, for NWC > 1,
//     the two edge lanes of a warp) go through a small double-buffered shared-memory exchange;
//   * CTAs are persistent (grid = resident CTAs, a multiple of the tile count so that a CTA stays on one radial
//     tile and keeps its per-column coefficients);
//   * the operator is applied as H' = H / c1 (c1 = first off-diagonal stencil weight), so the radial part is
//     (f_{j-1} + f_{j+1}) + d' f_j with no multiply on the neighbours; u'_k = H'^k psi and the accumulator takes
//     (-i)^k (dt c1)^k / k! u'_k -- the same polynomial as Eq. 37 in another rounding order.  The coupling weight
//     c_l E r_j / c1 of the (l, l+1) pair is formed once and used for both rows.  12.25 (3-point) / 16.25 (5-point)
//     FP64 instructions per point-update instead of 16.3 / 20.
#pragma once
#include "tdse_taylor_rp_plan.h"
#include "tdse_tma.cuh"

namespace tdse {

static __constant__ double kRpInvK[65];   // 1/k, k = 1..64 (filled by rp_init_tables)

template <int FD, int CP, int NWR, int NWC>
struct RpGeom {
    static constexpr int HW = (FD == 3) ? 1 : 2;
    static constexpr int NT = NWR * NWC * 32;
    static constexpr int WT = 32 * CP * NWC;           // tile columns
    static constexpr int ROWS = kRpRows * NWR;
    static_assert(HW <= CP, "radial halo wider than the patch");
};

// shared memory: vertical exchange [parity][warp][top,bottom][CP planes][32 lanes], radial edge exchange between
// the warps of a row group [parity][warp][left,right][4 rows][HW], row table
template <int FD, int CP, int NWR, int NWC, bool TMA, bool RK = false>
struct RpSmem {
    // TMA landing zone of the next item: [row][128-byte column group][8 columns], 128-byte swizzled; first member
    // so that it is 1024-byte aligned
    double2 stage[TMA ? kRpRows * NWR * 32 * CP * NWC : 1];
    unsigned long long mbar;                // completion of the TMA tile fetch
    unsigned long long cbar;                // CTA-wide split barrier of the order loop (arrive after publishing, wait before reading)
    double2 xch[2][NWR * NWC][2][CP][32];
    double2 edge[2][NWR * NWC][2][kRpRows][(FD == 3) ? 1 : 2];
    double2 zrow[CP][32];                   // zeros for ever: the rows above l = 0 and below the last row group
    double rowtab[NWR * kRpRows][4];        // {c_l, l(l+1), c_{l-1}, 0}
    double2 psi_s[RK ? kRpRows * CP : 1][NWR * NWC * 32];   // RK4: psi(t_n) of every thread's patch (private slots)
    double red[NWR * NWC][kRpObsRed];       // fused observables: per-warp partial sums
    int last_flag;
};

__device__ __forceinline__ double2 shfl_up2(double2 v) {
    return make_double2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ double2 shfl_dn2(double2 v) {
    return make_double2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ void ldg256(const double2 *p, double2 &a, double2 &b) {
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a.x), "=d"(a.y), "=d"(b.x), "=d"(b.y) : "l"(p));
}
__device__ __forceinline__ void stg256(double2 *p, const double2 &a, const double2 &b) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y) : "memory");
}

// tile start of tile t: interior [t*W, (t+1)*W) plus H halo columns per side, clamped so that a tile at a wall
// starts (ends) exactly at the wall: the zero beyond the tile IS the Dirichlet wall.
__device__ __forceinline__ int rp_start(int t, int W, int H, int N, int WT) {
    int start = t * W - H;
    if (start > N - WT) start = N - WT;
    if (start < 0) start = 0;
    return start;
}

// grid = persistent CTAs, block = NT.  n_l <= 4*NWR.  H = halo columns per side (>= order * HW; even when n_r is
// even so that every patch row is 32-byte aligned).  MASK: n_r < WT (single tile, columns >= n_r held at zero).
// TMA: the next item's tile is fetched by one cp.async.bulk.tensor (3-D view [row][n_r/8][8 columns], 128-byte
// swizzle so that the per-thread patch reads are bank-conflict free) while the current item is computed; needs
// n_r % 8 == 0, H % 8 == 0, W % 8 == 0 and n_r >= WT.
// CLUSTER: the n_l rows are split over the CTAs of a thread-block cluster (rank = row block of 4*NWR rows); the
// l-1 / l+1 rows at a CTA boundary are read from the neighbouring CTA's shared memory (DSMEM) and the per-order
// barrier is a cluster barrier.
// RK: classic RK4 (Eq. 38) instead of Taylor: four sweeps with the field at t_n, t_n + h/2 (twice),
// t_n + h (ef[stage*batch + b]); sweep i forms k_i = -i H g_i, the next stage vector g_{i+1} = psi + a_i h k_i (psi
// re-read from this thread's private shared-memory slots) and psi_new += b_i h k_i: 32 B/point/step over HBM instead
// of 272 for one kernel per stage.
// MODE: 0 Taylor in real time, 1 classic RK4 (above), 2 Taylor in IMAGINARY time (-i -> 1, weights
// (-dt c1)^k / k!; the caller re-normalises).
// OBS: the observable sums of the row logged after this step are reduced in the store phase (RpObs above).
// PERSIST: temporal blocking ACROSS steps: the halo H covers n_steps x order x hw columns, so a tile can take n_steps
// whole steps with psi in registers (field value ef[step * batch + b]; after each step the sum becomes the next input;
// one observable partial per logged step) and touches HBM once per launch -- small grids are bound by the serial work of
// a CTA instead of by one launch per step (NS: "so small grids are not launch-bound", hard part 4).
// CUT: some points of the patch are HELD at zero (centrifugal inner cut-off g.j0; columns >= n_r of a grid narrower than
// the tile): a separate instantiation, because the extra control flow costs the plain kernel its register allocation.
template <int FD, int CP, int NWR, int NWC, bool MASK, int MINB, bool TMA, bool CLUSTER, int MODE = 0, bool OBS = false,
          bool PERSIST = false, bool CUT = false>
__global__ void __launch_bounds__(NWR * NWC * 32, MINB)
taylor_rp_kernel(GridDev g, const double2 *__restrict__ in, double2 *__restrict__ out, const double *__restrict__ ef,
                 const double *__restrict__ dtp, int order, int W, int H, int n_tiles, int n_items,
                 const __grid_constant__ CUtensorMap tmap, const RpObs ob, int n_steps) {
    static_assert(!(OBS && MODE == 2), "fused observables: real-time propagation");
    static_assert(!(OBS && MASK), "fused observables: unmasked instantiations");
    static_assert(!(PERSIST && (MASK || TMA || CLUSTER || MODE != 0)), "several steps per launch: full tiles, direct loads, Taylor");
    static_assert(!(TMA && MASK), "the TMA path needs a full tile");
    static_assert(NWC > 1 || CP == 4, "one-warp-wide tiles use the edge-weight trick, which needs 4-column patches");
    using G = RpGeom<FD, CP, NWR, NWC>;
    constexpr int RP = kRpRows, WT = G::WT, HW = G::HW;
    extern __shared__ __align__(1024) unsigned char rp_smem_raw[];
    constexpr bool RK = (MODE == 1), IMAG = (MODE == 2);
    using Smem = RpSmem<FD, CP, NWR, NWC, TMA, RK>;
    Smem &sm = *reinterpret_cast<Smem *>(rp_smem_raw);     // dynamic shared memory starts 1024-byte aligned
    if (TMA && (smem_u32(rp_smem_raw) & 1023u)) __trap();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wr = warp / NWC, wc = warp - wr * NWC;
    const int L = g.n_l, N = g.n_r;
    const int crank = CLUSTER ? (int)cluster_ctarank() : 0, csize = CLUSTER ? (int)cluster_nctarank() : 1;
    const int rbase = crank * NWR * RP;                        // global row of this CTA's row 0
    const int cid = CLUSTER ? (int)blockIdx.x / csize : (int)blockIdx.x, ncl = CLUSTER ? (int)gridDim.x / csize : (int)gridDim.x;
    const int r0 = wr * RP, c0 = (wc * 32 + lane) * CP;
    const int gr0 = rbase + r0;                                // global row of this thread's patch row 0
    const double2 z2 = make_double2(0.0, 0.0);
    const bool al32 = !MASK && ((N & 1) == 0) && ((H & 1) == 0) && ((W & 1) == 0) && N >= WT;
    const bool ragged_rows = (csize * NWR * RP != L);

    for (int r = threadIdx.x; r < NWR * RP; r += G::NT) {
        const int l = rbase + r;
        sm.rowtab[r][0] = (l + 1 < L) ? __ldg(g.cl + l) : 0.0;
        sm.rowtab[r][1] = (double)l * (double)(l + 1);
        sm.rowtab[r][2] = (l >= 1 && l < L) ? __ldg(g.cl + l - 1) : 0.0;
        sm.rowtab[r][3] = 0.0;
    }
    for (int i = threadIdx.x; i < CP * 32; i += G::NT) sm.zrow[i / 32][i % 32] = make_double2(0.0, 0.0);
    __syncthreads();

    const double dt = *dtp;
    // fused observables: is the step a logged one, which row, at what time (uniform over the grid)
    bool obs_now = false;
    long long obs_row = 0;
    double obs_t = 0.0;
    // (the control block is read once: its loads must not sit in front of every step of a multi-step launch)
    const long long obs_base = OBS ? ob.ctl->step_base + ob.step_off + 1 : 0;
    const int obs_every = OBS ? ob.ctl->obs_every : 0;
    const double obs_t0 = OBS ? ob.ctl->t0 : 0.0, obs_dt = OBS ? ob.ctl->dt : 0.0;
    auto obs_setup = [&](const int step) {
        const long long n = obs_base + step;
        obs_now = obs_every > 0 && (n % obs_every) == 0;
        obs_row = obs_now ? n / obs_every - 1 : 0;
        obs_t = time_at(obs_t0, (double)n, obs_dt);
    };
    if (OBS) obs_setup(0);
    bool any_obs = obs_now;                                  // some step of this launch is a logged one
    const bool obs_direct = (n_tiles * csize == 1);         // the CTA owns the whole member: it writes the row itself
    // (with_field = false: the -E(t) term of <z''> is added afterwards by add_field, many rows at a time)
    auto write_row = [&](const int bb, const double (&s)[kRpObsRed], const bool with_field) {
        double *o = ob.rows + ((size_t)obs_row * g.batch + bb) * (3 + ob.n_states);
        o[0] = g.dr * s[0];
        o[1] = 2.0 * g.dr * s[1];
        const double acc = 2.0 * g.z * g.dr * s[2];
        o[2] = with_field ? -pulse_E(ob.pulse[bb], obs_t) - acc : -acc;
        for (int si = 0; si < ob.n_states && si < kRpObsStates; ++si) {
            const double ar = g.dr * s[3 + 2 * si], ai = g.dr * s[4 + 2 * si];
            o[3 + si] = ar * ar + ai * ai;
        }
    };
    const double inv_c1 = 1.0 / g.c1;
    const double kappa = dt * g.c1;                 // u'_k = (H/c1)^k psi  ->  weight (dt c1)^k / k!
    const double c2p = g.c2 * inv_c1;               // 5-point: second off-diagonal weight / c1 (= -1/16)
    // radial exchange across warps: lane 0 reads the right edge of warp wc-1, lane 31 the left edge of warp wc+1
    const bool is_edge = (NWC > 1) && (lane == 0 || lane == 31);
    const bool has_nb = (NWC > 1) && ((lane == 0 && wc > 0) || (lane == 31 && wc < NWC - 1));
    const int nb_warp = has_nb ? ((lane == 0) ? warp - 1 : warp + 1) : warp;
    const int nb_side = (lane == 0) ? 1 : 0, my_side = (lane == 0) ? 0 : 1;

    constexpr unsigned kStageBytes = (unsigned)(sizeof(double2) * RP * NWR * WT);
    unsigned tma_phase = 0;
    if (threadIdx.x == 0) {
        mbar_init(&sm.mbar, 1);
        mbar_init(&sm.cbar, G::NT);
    }
    __syncthreads();
    unsigned cphase = 0;
    bool armed = false;                      // a barrier arrival of this thread has not been waited for yet
    auto bar_arrive = [&]() {
        if (CLUSTER) cluster_arrive(); else mbar_arrive(&sm.cbar);
        armed = true;
    };
    auto bar_wait = [&]() {
        if (CLUSTER) cluster_wait();
        else { mbar_wait(&sm.cbar, cphase); cphase ^= 1u; }
        armed = false;
    };
    // tile of work item `it` -> stage (one thread; the stage must have been consumed by every thread)
    auto fetch_tile = [&](const int fb, const int ft) {
        if (TMA && threadIdx.x == 0) {
            fence_proxy_async_smem();
            mbar_expect_tx(&sm.mbar, kStageBytes);
            tma_load_3d(sm.stage, &tmap, 0, rp_start(ft, W, H, N, WT) >> 3, fb * L + rbase, &sm.mbar);
        }
    };
    const int db = ncl / n_tiles, dtile = ncl - db * n_tiles;
    int b = cid / n_tiles, t = cid - b * n_tiles;
    if (cid < n_items) fetch_tile(b, t);

    const double wl = (lane == 0) ? 0.0 : 1.0, wrt = (lane == 31) ? 0.0 : 1.0;
    // l-1 / l+1 rows of the neighbouring row groups (or the zero row); the parity offset is 0 for the zero row
    constexpr int kParStride = (int)(sizeof(sm.xch[0]) / sizeof(double2));
    const double2 *lo_base = (wr > 0) ? &sm.xch[0][wr > 0 ? warp - NWC : 0][1][0][lane] : &sm.zrow[0][lane];
    const double2 *up_base = (wr < NWR - 1) ? &sm.xch[0][wr < NWR - 1 ? warp + NWC : 0][0][0][lane] : &sm.zrow[0][lane];
    const int lo_par = (wr > 0) ? kParStride : 0, up_par = (wr < NWR - 1) ? kParStride : 0;
    // CLUSTER: the row groups at the CTA boundary read the neighbouring CTA's exchange buffer through DSMEM
    const bool lo_remote = CLUSTER && wr == 0 && crank > 0, up_remote = CLUSTER && wr == NWR - 1 && crank < csize - 1;
    unsigned lo_dsm = 0, up_dsm = 0;
    if (CLUSTER) {
        if (lo_remote) lo_dsm = dsmem_addr(&sm.xch[0][(NWR - 1) * NWC + wc][1][0][lane], (unsigned)(crank - 1));
        if (up_remote) up_dsm = dsmem_addr(&sm.xch[0][wc][0][0][lane], (unsigned)(crank + 1));
    }

    int t_cur = -1;
    double ef_cur = (cid < n_items) ? __ldg(ef + b) : 0.0, ef_next = 0.0;
    double Dq[CP], Cq[CP], Eq[CP];
    bool dom[CP];
#pragma unroll
    for (int q = 0; q < CP; ++q) { Dq[q] = 0.0; Cq[q] = 0.0; dom[q] = true; }

    for (int item = cid; item < n_items; item += ncl) {
        const int start = rp_start(t, W, H, N, WT);
        const double2 *src_g = in + ((size_t)b * L + rbase) * N + start + c0;
        // ---- own patch straight from global memory -------------------------------------------------------------
        double2 T[RP][CP], A[RP][CP];
        if (TMA) {
            if (order < 2 && item != cid) {      // no second order whose barrier could have covered the refill
                if (armed) bar_wait();
                fetch_tile(b, t);
            }
            mbar_wait(&sm.mbar, tma_phase);
            tma_phase ^= 1u;
            const int gidx = (wc * 32 + lane) * CP / 8, chunk0 = ((wc * 32 + lane) * CP) & 7;
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    const double2 v = sm.stage[((r0 + r) * (WT / 8) + gidx) * 8 + ((chunk0 + q) ^ (gidx & 7))];
                    T[r][q] = (gr0 + r < L) ? v : z2;
                }
        } else {
#pragma unroll
        for (int r = 0; r < RP; ++r) {
            const double2 *p = src_g + (size_t)(r0 + r) * N;
            if (gr0 + r < L) {
                if (al32) {
#pragma unroll
                    for (int q = 0; q < CP; q += 2) ldg256(p + q, T[r][q], T[r][q + 1]);
                } else {
#pragma unroll
                    for (int q = 0; q < CP; ++q) T[r][q] = (!MASK || start + c0 + q < N) ? __ldg(p + q) : z2;
                }
            } else {
#pragma unroll
                for (int q = 0; q < CP; ++q) T[r][q] = z2;
            }
        }
        }
        // ---- centrifugal cut-off (tdse_set_cutoff): the held points of this patch read as zero and stay zero ---------
        // (a grid narrower than the tile of an unmasked instantiation -- the persistent kernel -- holds its columns >= n_r
        // at zero the same way)
        const bool cut_item = CUT && ((g.j0 != nullptr && start < g.j0_max) || (!MASK && N < start + WT));   // (uniform over the CTA)
        unsigned held_bits = 0u;
        if (cut_item) {
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int q = 0; q < CP; ++q)
                    if (held_pt(g, gr0 + r, start + c0 + q) || start + c0 + q >= N) { held_bits |= 1u << (r * CP + q); T[r][q] = z2; }
        }
        // ---- per-column coefficients (scaled by 1/c1): reloaded only when the radial tile changes ----------------
        if (t != t_cur) {
            t_cur = t;
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                const int j = start + c0 + q;
                dom[q] = !MASK || j < N;
                const int jj = (dom[q] && j < N) ? j : 0;
                Dq[q] = inv_c1 * __ldg(g.vj + jj);
                Cq[q] = inv_c1 * __ldg(g.cen + jj);
            }
        }
        // coupling weights E r_j / c1 for the field value of this step (Taylor) or of RK stage `st`
        auto set_field = [&](const int st) {
            const double es = inv_c1 * (((RK || st) ? __ldg(ef + st * g.batch + b) : ef_cur) * g.dr);
#pragma unroll
            for (int q = 0; q < CP; ++q) Eq[q] = es * (double)(dom[q] ? start + c0 + q + 1 : 1);
        };
        // interior columns of the tile and valid rows (what is stored and what enters the observables); recomputed where
        // needed so that nothing of it is live across the order loop
        auto interior = [&](bool (&in_c)[CP], bool (&row_ok)[RP]) {
            const int lo_c = t * W - start;                  // first interior column (tile coordinates)
            int wint = N - t * W;
            if (wint > W) wint = W;
#pragma unroll
            for (int q = 0; q < CP; ++q) in_c[q] = c0 + q >= lo_c && c0 + q < lo_c + wint;
#pragma unroll
            for (int r = 0; r < RP; ++r) row_ok[r] = !ragged_rows || gr0 + r < L;
        };
        const int n_rep = PERSIST ? n_steps : 1;
        for (int step = 0; step < n_rep; ++step) {          // (PERSIST: psi stays in registers between the steps)
        if (PERSIST && step > 0) {
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int q = 0; q < CP; ++q) T[r][q] = A[r][q];
            if (OBS) { obs_setup(step); any_obs = any_obs || obs_now; }
        }
        set_field(0);
        if (RK) {       // psi(t_n) is needed again when the stage vectors g_2..g_4 are formed
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int q = 0; q < CP; ++q) sm.psi_s[r * CP + q][threadIdx.x] = T[r][q];
        }
        // publish u_0: rows 0 and RP-1 for the warps above / below, edge columns for the warps left / right
        // (after every thread has finished reading the previous item's last exchange)
        if (armed) bar_wait();
#pragma unroll
        for (int q = 0; q < CP; ++q) {
            sm.xch[0][warp][0][q][lane] = T[0][q];
            sm.xch[0][warp][1][q][lane] = T[RP - 1][q];
        }
        if (is_edge) {
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int h = 0; h < HW; ++h) sm.edge[0][warp][my_side][r][h] = (lane == 0) ? T[r][h] : T[r][CP - 1 - h];
        }
        bar_arrive();

        // One row of one order: To[r] = (H' Ti)[r], A[r] += weight * To[r].  dn / up = rows l-1 / l+1, alo / aup =
        // their coupling weights c_{l-1} E r / c1 and c_l E r / c1; ev1 / ev2 = edge columns of the neighbouring warp.
        auto do_row = [&](const double2 (&Ti)[RP][CP], double2 (&To)[RP][CP], const int r, const double2 (&dn)[CP],
                          const double2 (&up)[CP], const double (&alo)[CP], const double (&aup)[CP], const double ll1,
                          const int pr, const bool odd, const bool first, const double s, const bool want_out,
                          const double cg) {
            double2 lf1 = shfl_up2(Ti[r][CP - 1]);       // column c0 - 1 from lane - 1
            double2 rg1 = shfl_dn2(Ti[r][0]);            // column c0 + CP from lane + 1
            double2 lf2 = z2, rg2 = z2;
            if (FD == 5) {
                lf2 = shfl_up2(Ti[r][CP - 2]);
                rg2 = shfl_dn2(Ti[r][1]);
            }
            if (NWC > 1) {      // NWC == 1: the tile edge is zero through the weights wl / wrt below
                double2 ev1 = z2, ev2 = z2;
                if (has_nb) {
                    ev1 = sm.edge[pr][nb_warp][nb_side][r][0];
                    if (FD == 5) ev2 = sm.edge[pr][nb_warp][nb_side][r][HW - 1];
                }
                if (lane == 0) { lf1 = ev1; lf2 = ev2; }
                if (lane == 31) { rg1 = ev1; rg2 = ev2; }
            }
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                const double2 f = Ti[r][q];
                const double2 m1 = (q > 0) ? Ti[r][q > 0 ? q - 1 : 0] : lf1;
                const double2 p1 = (q < CP - 1) ? Ti[r][q < CP - 1 ? q + 1 : 0] : rg1;
                const double d = fma(ll1, Cq[q], Dq[q]);
                // lanes 0 / 31 of a one-warp-wide tile got their own value back from the shuffle: weight 0
                double hx, hy;
                if (NWC == 1 && q == 0) { hx = fma(wl, m1.x, p1.x); hy = fma(wl, m1.y, p1.y); }
                else if (NWC == 1 && q == CP - 1) { hx = fma(wrt, p1.x, m1.x); hy = fma(wrt, p1.y, m1.y); }
                else { hx = m1.x + p1.x; hy = m1.y + p1.y; }
                if (FD == 5) {
                    const double2 m2 = (q > 1) ? Ti[r][q > 1 ? q - 2 : 0] : ((q == 1) ? lf1 : lf2);
                    const double2 p2 = (q < CP - 2) ? Ti[r][q < CP - 2 ? q + 2 : 0] : ((q == CP - 2) ? rg1 : rg2);
                    double sx, sy;
                    if (NWC == 1 && q <= 1) { sx = fma(wl, m2.x, p2.x); sy = fma(wl, m2.y, p2.y); }
                    else if (NWC == 1 && q >= CP - 2) { sx = fma(wrt, p2.x, m2.x); sy = fma(wrt, p2.y, m2.y); }
                    else { sx = m2.x + p2.x; sy = m2.y + p2.y; }
                    hx = fma(c2p, sx, hx);
                    hy = fma(c2p, sy, hy);
                }
                hx = fma(d, f.x, hx);
                hy = fma(d, f.y, hy);
                hx = fma(aup[q], up[q].x, hx);
                hy = fma(aup[q], up[q].y, hy);
                hx = fma(alo[q], dn[q].x, hx);
                hy = fma(alo[q], dn[q].y, hy);
                if (MASK && !dom[q]) { hx = 0.0; hy = 0.0; }
                if (!RK) To[r][q] = make_double2(hx, hy);
                else if (want_out) {            // g_{i+1} = psi + a_i h k_i,  k_i = -i H g_i = c1 (hy - i hx)
                    const double2 p0 = first ? f : sm.psi_s[r * CP + q][threadIdx.x];
                    To[r][q] = make_double2(fma(cg, hy, p0.x), fma(-cg, hx, p0.y));
                }
                // acc += (-i)^k (dt c1)^k / k! * u'_k; s carries the sign: odd k: -+i, even k: -+1
                // (order 1 starts the sum from psi itself: A = u_0 + ..., no separate copy)
                if (first && odd) { A[r][q].x = fma(s, hy, f.x); A[r][q].y = fma(-s, hx, f.y); }
                else if (first) { A[r][q].x = fma(s, hx, f.x); A[r][q].y = fma(s, hy, f.y); }
                else if (odd) { A[r][q].x = fma(s, hy, A[r][q].x); A[r][q].y = fma(-s, hx, A[r][q].y); }
                else { A[r][q].x = fma(s, hx, A[r][q].x); A[r][q].y = fma(s, hy, A[r][q].y); }
            }
            if (cut_item) {     // P H P: the new term (stage vector) vanishes at the held points (A is cleared at the end)
#pragma unroll
                for (int q = 0; q < CP; ++q)
                    if ((held_bits >> (r * CP + q)) & 1u) To[r][q] = z2;
            }
        };

        // One order.  The rows that need nothing from other warps (1 and 2 of a one-warp-wide tile) are computed
        // BEFORE waiting on the barrier that publishes the other warps' rows; then rows 0 and 3, then this warp's
        // outer rows are published and the barrier is signalled (split arrive / wait).  The order loop below is
        // unrolled by two with the roles of T and U swapped, so that the new term is written where the term before
        // last lived and no register copies are needed at the loop back-edge.
        auto sweep = [&](const double2 (&Ti)[RP][CP], double2 (&To)[RP][CP], const int k, const bool odd, const bool first, const double s,
                         const double cg) {
            const bool want_out = k < order;
            const int pr = (k - 1) & 1, pw = k & 1;
            double cup[RP], ll1[RP];
#pragma unroll
            for (int r = 0; r < RP; ++r) {
                const double2 rt = *reinterpret_cast<const double2 *>(&sm.rowtab[r0 + r][0]);
                cup[r] = rt.x; ll1[r] = rt.y;
            }
            double a0[CP], a1[CP], a2[CP], a3[CP], ac[CP];
            if (NWC == 1) {
#pragma unroll
                for (int q = 0; q < CP; ++q) { a0[q] = cup[0] * Eq[q]; a1[q] = cup[1] * Eq[q]; a2[q] = cup[2] * Eq[q]; }
                do_row(Ti, To, 1, Ti[0], Ti[2], a0, a1, ll1[1], pr, odd, first, s, want_out, cg);
                do_row(Ti, To, 2, Ti[1], Ti[3], a1, a2, ll1[2], pr, odd, first, s, want_out, cg);
            }
            bar_wait();
            // every value of the stage was consumed by the arithmetic of order 1: fetch the next item (and its field value)
            if (TMA && k == 2 && item + ncl < n_items) {
                int nb = b + db, nt = t + dtile;
                if (nt >= n_tiles) { nt -= n_tiles; ++nb; }
                fetch_tile(nb, nt);
            }
            if (!RK && k == 1) {
                if (PERSIST && step + 1 < n_rep) ef_next = __ldg(ef + (size_t)(step + 1) * g.batch + b);
                else if (item + ncl < n_items) ef_next = __ldg(ef + b + db + ((t + dtile >= n_tiles) ? 1 : 0));
            }
            double2 lo[CP], below[CP];
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                if (CLUSTER && lo_remote) lo[q] = ld_dsmem2(lo_dsm + (unsigned)((pr * kParStride + q * 32) * sizeof(double2)));
                else lo[q] = lo_base[pr * lo_par + q * 32];
            }
            const double clo = sm.rowtab[r0][2];
            if (NWC == 1) {
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    if (CLUSTER && up_remote) below[q] = ld_dsmem2(up_dsm + (unsigned)((pr * kParStride + q * 32) * sizeof(double2)));
                    else below[q] = up_base[pr * up_par + q * 32];
                }
#pragma unroll
                for (int q = 0; q < CP; ++q) { ac[q] = clo * Eq[q]; a3[q] = cup[3] * Eq[q]; }
                do_row(Ti, To, 0, lo, Ti[1], ac, a0, ll1[0], pr, odd, first, s, want_out, cg);
                do_row(Ti, To, 3, Ti[2], below, a2, a3, ll1[3], pr, odd, first, s, want_out, cg);
            } else {
                // tiles wider than a warp: every row needs the neighbouring warp's edge columns, so all rows come after
                // the barrier, in order, with the coupling weights of one row pair formed at a time (register budget)
#pragma unroll
                for (int q = 0; q < CP; ++q) { ac[q] = clo * Eq[q]; a0[q] = cup[0] * Eq[q]; }
                do_row(Ti, To, 0, lo, Ti[1], ac, a0, ll1[0], pr, odd, first, s, want_out, cg);
#pragma unroll
                for (int q = 0; q < CP; ++q) a1[q] = cup[1] * Eq[q];
                do_row(Ti, To, 1, Ti[0], Ti[2], a0, a1, ll1[1], pr, odd, first, s, want_out, cg);
#pragma unroll
                for (int q = 0; q < CP; ++q) a2[q] = cup[2] * Eq[q];
                do_row(Ti, To, 2, Ti[1], Ti[3], a1, a2, ll1[2], pr, odd, first, s, want_out, cg);
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    if (CLUSTER && up_remote) below[q] = ld_dsmem2(up_dsm + (unsigned)((pr * kParStride + q * 32) * sizeof(double2)));
                    else below[q] = up_base[pr * up_par + q * 32];
                    a3[q] = cup[3] * Eq[q];
                }
                do_row(Ti, To, 3, Ti[2], below, a2, a3, ll1[3], pr, odd, first, s, want_out, cg);
            }
            if (k < order) {
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    sm.xch[pw][warp][0][q][lane] = To[0][q];
                    sm.xch[pw][warp][1][q][lane] = To[RP - 1][q];
                }
                if (is_edge) {
#pragma unroll
                    for (int r = 0; r < RP; ++r)
#pragma unroll
                        for (int h = 0; h < HW; ++h)
                            sm.edge[pw][warp][my_side][r][h] = (lane == 0) ? To[r][h] : To[r][CP - 1 - h];
                }
            }
            bar_arrive();
        };

        double2 U[RP][CP];
        if (RK) {
            // classic RK4: a = (1/2, 1/2, 1), b = (1/6, 1/3, 1/3, 1/6); kappa = h c1 carries k_i's factor c1
            sweep(T, U, 1, true, true, kappa * (1.0 / 6.0), 0.5 * kappa);
            set_field(1);
            sweep(U, T, 2, true, false, kappa * (1.0 / 3.0), 0.5 * kappa);
            set_field(2);
            sweep(T, U, 3, true, false, kappa * (1.0 / 3.0), kappa);
            set_field(3);
            sweep(U, T, 4, true, false, kappa * (1.0 / 6.0), 0.0);
        } else if (IMAG) {
            double sk = -kappa;                                   // every order is "even": real weights (-kappa)^k / k!
            sweep(T, U, 1, false, true, sk, 0.0);
            int k = 2;
            for (; k + 1 <= order; k += 2) {
                sk = sk * (-kappa * kRpInvK[k]);
                sweep(U, T, k, false, false, sk, 0.0);
                sk = sk * (-kappa * kRpInvK[k + 1]);
                sweep(T, U, k + 1, false, false, sk, 0.0);
            }
            if (k <= order) {
                sk = sk * (-kappa * kRpInvK[k]);
                sweep(U, T, k, false, false, sk, 0.0);
            }
        } else {
            double sk = kappa;
            sweep(T, U, 1, true, true, sk, 0.0);                  // order 1: -i
            int k = 2;
            for (; k + 1 <= order; k += 2) {
                sk = sk * (kappa * kRpInvK[k]);
                sweep(U, T, k, false, false, (k & 2) ? -sk : sk, 0.0);
                sk = sk * (kappa * kRpInvK[k + 1]);
                sweep(T, U, k + 1, true, false, ((k + 1) & 2) ? -sk : sk, 0.0);
            }
            if (k <= order) {
                sk = sk * (kappa * kRpInvK[k]);
                sweep(U, T, k, false, false, (k & 2) ? -sk : sk, 0.0);
            }
        }
        // the barrier signalled by the last order is waited for before the next item publishes (or at the end)
        if (cut_item) {
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int q = 0; q < CP; ++q)
                    if ((held_bits >> (r * CP + q)) & 1u) A[r][q] = z2;
        }

        // ---- end of the step: absorber, observables of the logged row ---------------------------------------------
        {
            if (MODE != 2 && g.mask != nullptr) {            // absorbing boundary: psi *= exp(-i W dt) (Eq. 18)
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    const int jj = start + c0 + q;
                    const double m = (jj < N) ? __ldg(g.mask + jj) : 0.0;
#pragma unroll
                    for (int r = 0; r < RP; ++r) { A[r][q].x *= m; A[r][q].y *= m; }
                }
            }
            // (the fused observables come BEFORE the stores: the release fences of their exchange would otherwise wait
            // for the stores to drain)
            if (OBS && obs_now) {
                bool in_c[CP], row_ok[RP];
                interior(in_c, row_ok);
                // row l-1 of psi(t + dt) for this thread's row 0: one more exchange through the buffer of the order loop
                if (armed) bar_wait();
#pragma unroll
                for (int q = 0; q < CP; ++q) sm.xch[0][warp][1][q][lane] = A[RP - 1][q];
                bar_arrive();
                double red[kRpObsRed];
#pragma unroll
                for (int i = 0; i < kRpObsRed; ++i) red[i] = 0.0;
                // the sums that need nothing from other warps are formed between arrive and wait
                double szc[CP];
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    double nn = 0.0, sz = 0.0;
#pragma unroll
                    for (int r = 0; r < RP; ++r) {
                        const double2 a = A[r][q];
                        if (row_ok[r]) nn += a.x * a.x + a.y * a.y;
                        if (r > 0 && row_ok[r]) {
                            const double2 pv = A[r > 0 ? r - 1 : 0][q];
                            sz = fma(sm.rowtab[r0 + r][2], pv.x * a.x + pv.y * a.y, sz);     // c_{l-1} Re(conj f_{l-1} f_l)
                        }
                    }
                    szc[q] = sz;
                    if (in_c[q]) red[0] += nn;
                }
                bar_wait();
                const double c_lo = sm.rowtab[r0][2];
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    double2 lo;
                    if (CLUSTER && lo_remote) lo = ld_dsmem2(lo_dsm + (unsigned)(q * 32 * sizeof(double2)));
                    else lo = lo_base[q * 32];
                    const double sz = fma(c_lo, lo.x * A[0][q].x + lo.y * A[0][q].y, szc[q]);
                    if (in_c[q]) {
                        const double rj = g.dr * (double)(start + c0 + q + 1);
                        red[1] = fma(rj, sz, red[1]);
                        red[2] += sz / (rj * rj);
                    }
                }
                bar_arrive();                   // (waited for before the next item publishes into the buffer)
#pragma unroll
                for (int si = 0; si < kRpObsStates; ++si) {          // (compile-time indices: red[] stays in registers)
                    if (si >= ob.n_states) continue;
                    const int lr = __ldg(ob.l_of_state + si) - gr0;
                    if (lr < 0 || lr >= RP) continue;
#pragma unroll
                    for (int q = 0; q < CP; ++q) {
                        if (!in_c[q]) continue;
                        const double w = __ldg(ob.phi + (size_t)si * N + start + c0 + q);
                        double2 a = A[0][q];
#pragma unroll
                        for (int r = 1; r < RP; ++r) if (lr == r) a = A[r][q];
                        red[3 + 2 * si] = fma(w, a.x, red[3 + 2 * si]);
                        red[4 + 2 * si] = fma(w, a.y, red[4 + 2 * si]);
                    }
                }
#pragma unroll
                for (int i = 0; i < kRpObsRed; ++i) {
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) red[i] += __shfl_down_sync(0xffffffffu, red[i], off);
                }
                if (lane == 0) {
#pragma unroll
                    for (int i = 0; i < kRpObsRed; ++i) sm.red[warp][i] = red[i];
                }
                __syncthreads();
                if (obs_direct) {
                    if (threadIdx.x == 0) {
                        double sred[kRpObsRed];
#pragma unroll
                        for (int i = 0; i < kRpObsRed; ++i) {
                            double v = 0.0;
                            for (int w2 = 0; w2 < NWR * NWC; ++w2) v += sm.red[w2][i];
                            sred[i] = v;
                        }
                        write_row(b, sred, true);
                    }
                    __syncthreads();            // sm.red is free again (the next step may come soon)
                } else if (threadIdx.x < kRpObsRed) {
                    double v = 0.0;
                    for (int w2 = 0; w2 < NWR * NWC; ++w2) v += sm.red[w2][threadIdx.x];
                    ob.partials[(((size_t)step * n_items + item) * csize + crank) * kRpObsRed + threadIdx.x] = v;
                }
            }
        }
        if (PERSIST && step + 1 < n_rep) ef_cur = ef_next;
        }   // step
        // ---- psi(t + dt): interior columns of the tile straight from registers ---------------------------------
        {
            double2 *dst_g = out + ((size_t)b * L + rbase + r0) * N + start + c0;
            bool in_c[CP], row_ok[RP];
            interior(in_c, row_ok);
            double2 *prow[RP];
#pragma unroll
            for (int r = 0; r < RP; ++r) prow[r] = dst_g + (size_t)r * N;
            if (al32) {                                      // interior bounds are even: in_c[q] == in_c[q + 1]
#pragma unroll
                for (int r = 0; r < RP; ++r)
#pragma unroll
                    for (int q = 0; q < CP; q += 2)
                        if (in_c[q] && row_ok[r]) stg256(prow[r] + q, A[r][q], A[r][q + 1]);
            } else {
#pragma unroll
                for (int r = 0; r < RP; ++r)
#pragma unroll
                    for (int q = 0; q < CP; ++q)
                        if (in_c[q] && row_ok[r]) prow[r][q] = A[r][q];
            }
        }
        b += db; t += dtile;
        if (t >= n_tiles) { t -= n_tiles; ++b; }
        ef_cur = ef_next;
    }
    if (armed) bar_wait();     // (cluster: no CTA may exit while a neighbour can still read its shared memory)
    if (OBS && !obs_direct) {
        // (uniform over the grid: every CTA took the same steps)
        if (PERSIST) { for (int st = 0; st < n_steps; ++st) { obs_setup(st); any_obs = any_obs || obs_now; } }
        if (!any_obs) return;
        // the last CTA to sign off adds the partials of every member in a fixed order and writes the row
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            const unsigned int ticket = atomicAdd(ob.counter, 1u);
            sm.last_flag = (ticket == gridDim.x - 1);
        }
        __syncthreads();
        if (!sm.last_flag) return;
        __threadfence();
        const int per = n_tiles * csize;
        const int n_st = PERSIST ? n_steps : 1;
        if (per <= 16) {
            // few partials per member (small grids): one THREAD per (step, member) adds them in a fixed order and
            // writes the row, field value included -- no barriers, every row of the launch at the same time
            for (int idx = threadIdx.x; idx < n_st * g.batch; idx += G::NT) {
                const int st = idx / g.batch, bb = idx - st * g.batch;
                obs_setup(st);
                if (!obs_now) continue;
                double s[kRpObsRed];
#pragma unroll
                for (int j = 0; j < kRpObsRed; ++j) s[j] = 0.0;
                const double *pp = ob.partials + ((size_t)st * n_items * csize + (size_t)bb * per) * kRpObsRed;
                for (int i = 0; i < per; ++i) {
#pragma unroll
                    for (int j = 0; j < kRpObsRed; ++j) s[j] += __ldcg(pp + (size_t)i * kRpObsRed + j);
                }
                write_row(bb, s, true);
            }
            if (threadIdx.x == 0) *ob.counter = 0u;
            return;
        }
        for (int st = 0; st < n_st; ++st) {
        obs_setup(st);
        if (!obs_now) continue;
        constexpr int NW = NWR * NWC;
        // many members: one warp per member; few members (a single wavefunction): the whole CTA per member
        const bool by_warp = g.batch >= NW;
        for (int bb = by_warp ? warp : 0; bb < g.batch; bb += by_warp ? NW : 1) {
            double s[kRpObsRed];
#pragma unroll
            for (int i = 0; i < kRpObsRed; ++i) s[i] = 0.0;
            const double *pp = ob.partials + ((size_t)st * n_items * csize + (size_t)bb * per) * kRpObsRed;
            const int first = by_warp ? lane : (int)threadIdx.x, stride = by_warp ? 32 : G::NT;
#pragma unroll 4
            for (int i = first; i < per; i += stride) {
#pragma unroll
                for (int j = 0; j < kRpObsRed; ++j) s[j] += __ldcg(pp + (size_t)i * kRpObsRed + j);
            }
#pragma unroll
            for (int j = 0; j < kRpObsRed; ++j) {
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) s[j] += __shfl_down_sync(0xffffffffu, s[j], off);
            }
            if (by_warp) {
                if (lane == 0) write_row(bb, s, false);
            } else {
                __syncthreads();
                if (lane == 0) {
#pragma unroll
                    for (int j = 0; j < kRpObsRed; ++j) sm.red[warp][j] = s[j];
                }
                __syncthreads();
                if (threadIdx.x == 0) {
#pragma unroll
                    for (int j = 0; j < kRpObsRed; ++j) {
                        double v = 0.0;
                        for (int w2 = 0; w2 < NW; ++w2) v += sm.red[w2][j];
                        s[j] = v;
                    }
                    write_row(bb, s, false);
                }
            }
        }
        }   // step of the launch
        // <z''> = -E(t) - ...: the field values of all rows of the launch, one (step, member) per thread -- a serial
        // evaluation per row (three divisions, a sine and a cosine in one thread) would cost more than the sums
        __syncthreads();
        for (int idx = threadIdx.x; idx < n_st * g.batch; idx += G::NT) {
            const int st = idx / g.batch, bb = idx - st * g.batch;
            obs_setup(st);
            if (!obs_now) continue;
            double *o = ob.rows + ((size_t)obs_row * g.batch + bb) * (3 + ob.n_states);
            o[2] = o[2] - pulse_E(ob.pulse[bb], obs_t);
        }
        if (threadIdx.x == 0) *ob.counter = 0u;
    }
}

// ------------------------------------------------------------------------------------------------------
// Host side: launchers of the instantiations of ONE stencil (FD), compiled in tdse_taylor_rp_fd3.cu / _fd5.cu
// ------------------------------------------------------------------------------------------------------
// (one copy of the constant table per translation unit, hence per FD)
template <int FD>
inline int rp_init_tables() {
    static DeviceOnce once;
    if (!once.first()) return TDSE_OK;
    double h[65];
    h[0] = 0.0;
    for (int k = 1; k <= 64; ++k) h[k] = 1.0 / (double)k;
    return cudaMemcpyToSymbol(kRpInvK, h, sizeof(h)) == cudaSuccess ? TDSE_OK : TDSE_ERR_CUDA;
}

template <class K>
inline int rp_launch_kernel(K kern, DeviceOnce *once, int smem, const RpPlan &p, cudaStream_t s, const GridDev &g,
                            const double2 *in, double2 *out, const double *ef, const double *dtp, int order,
                            const CUtensorMap &tm, const RpObs &ob, int n_steps = 1) {
    if (once->first()) {
        if (cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
            return TDSE_ERR_CUDA;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.grid); cfg.blockDim = dim3(p.threads); cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = p.cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = (p.cl > 1) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, g, in, out, ef, dtp, order, p.W, p.H, p.n_tiles, p.n_items, tm, ob, n_steps) == cudaSuccess
               ? TDSE_OK : TDSE_ERR_CUDA;
}

// the four full-tile instantiations (direct / TMA) x (CTA / cluster) of one (MODE, OBS) pair
template <int FD, int CP, int NWR, int NWC, int MINB, bool CLUSTERABLE, int MODE, bool OBS, bool CUT = false>
inline int rp_launch_full(const GridDev &g, const RpPlan &p, const CUtensorMap &tm, const double2 *in, double2 *out,
                          const double *ef, const double *dtp, int order, cudaStream_t s, const RpObs &ob) {
    static DeviceOnce once[4];
    constexpr bool RK = (MODE == 1);
    const int sm_t = (int)sizeof(RpSmem<FD, CP, NWR, NWC, true, RK>), sm_n = (int)sizeof(RpSmem<FD, CP, NWR, NWC, false, RK>);
    if (p.cl > 1) {
        if (!CLUSTERABLE) return TDSE_ERR_UNSUPPORTED;
        constexpr bool kCl = CLUSTERABLE;
        if (p.tma) return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, false, MINB, true, kCl, MODE, OBS, false, CUT>, &once[3], sm_t, p, s, g, in, out, ef, dtp, order, tm, ob);
        return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, false, MINB, false, kCl, MODE, OBS, false, CUT>, &once[2], sm_n, p, s, g, in, out, ef, dtp, order, tm, ob);
    }
    if (p.tma) return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, false, MINB, true, false, MODE, OBS, false, CUT>, &once[1], sm_t, p, s, g, in, out, ef, dtp, order, tm, ob);
    return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, false, MINB, false, false, MODE, OBS, false, CUT>, &once[0], sm_n, p, s, g, in, out, ef, dtp, order, tm, ob);
}

// MODE 1 / 2 instantiations exist only for the one-warp-wide variants (RKABLE) and full tiles; fused observables (ob)
// for full tiles in real time (MODE 0 / 1)
// up to p.persist steps per launch (halo sized for them)
template <int FD, int CP, int NWR, int NWC, int MINB>
inline int rp_launch_persist(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                             const double *dtp, int order, cudaStream_t s, const RpObs *ob, int n_steps) {
    const bool mask = g.n_r < 32 * CP * NWC;
    if (!p.persist || mask || p.tma || p.cl > 1 || p.rk != 0 || n_steps > p.persist || g.j0 != nullptr) return TDSE_ERR_UNSUPPORTED;
    static DeviceOnce once[2];
    const CUtensorMap no_map{};
    const RpObs no_obs{};
    const int smem = (int)sizeof(RpSmem<FD, CP, NWR, NWC, false>);
    if (ob) return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, false, MINB, false, false, 0, true, true>, &once[0], smem, p, s, g, in, out, ef, dtp, order, no_map, *ob, n_steps);
    return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, false, MINB, false, false, 0, false, true>, &once[1], smem, p, s, g, in, out, ef, dtp, order, no_map, no_obs, n_steps);
}

template <int FD, int CP, int NWR, int NWC, int MINB, bool CLUSTERABLE, bool RKABLE>
inline int rp_launch_one(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                         const double *dtp, int order, cudaStream_t s, const RpObs *ob, int n_steps) {
    const bool mask = g.n_r < 32 * CP * NWC;
    if (p.persist) return rp_launch_persist<FD, CP, NWR, NWC, MINB>(g, p, in, out, ef, dtp, order, s, ob, n_steps);
    if (n_steps != 1) return TDSE_ERR_UNSUPPORTED;
    CUtensorMap tmap{};
    if (p.tma) {
        if (mask) return TDSE_ERR_UNSUPPORTED;
        if (!tma_map_rows3d(&tmap, in, g.n_r, g.batch * g.n_l, kRpRows * NWR, 32 * CP * NWC)) return TDSE_ERR_CUDA;
    }
    const RpObs none{};
    if (mask) {
        if (p.rk != 0 || p.cl > 1 || ob) return TDSE_ERR_UNSUPPORTED;
        static DeviceOnce once;
        return rp_launch_kernel(taylor_rp_kernel<FD, CP, NWR, NWC, true, MINB, false, false, 0, false, false, true>, &once,
                                (int)sizeof(RpSmem<FD, CP, NWR, NWC, false>), p, s, g, in, out, ef, dtp, order, tmap, none);
    }
    const bool cut = g.j0 != nullptr;            // centrifugal cut-off: the CUT instantiations (no fused rows, no imaginary time)
    if (p.rk == 2) {
        if (!RKABLE || ob || cut) return TDSE_ERR_UNSUPPORTED;
        return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, RKABLE ? 2 : 0, false>(g, p, tmap, in, out, ef, dtp, order, s, none);
    }
    if (cut && ob) return TDSE_ERR_UNSUPPORTED;
    if (p.rk == 1) {
        if (!RKABLE) return TDSE_ERR_UNSUPPORTED;
        if (cut) return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, RKABLE ? 1 : 0, false, true>(g, p, tmap, in, out, ef, dtp, order, s, none);
        if (ob) return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, RKABLE ? 1 : 0, true>(g, p, tmap, in, out, ef, dtp, order, s, *ob);
        return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, RKABLE ? 1 : 0, false>(g, p, tmap, in, out, ef, dtp, order, s, none);
    }
    if (cut) return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, 0, false, true>(g, p, tmap, in, out, ef, dtp, order, s, none);
    if (ob) return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, 0, true>(g, p, tmap, in, out, ef, dtp, order, s, *ob);
    return rp_launch_full<FD, CP, NWR, NWC, MINB, CLUSTERABLE, 0, false>(g, p, tmap, in, out, ef, dtp, order, s, none);
}

template <int FD>
inline int launch_taylor_rp_fd(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                               const double *dtp, int order, cudaStream_t s, const RpObs *ob, int n_steps) {
    if (!p.ok) return TDSE_ERR_UNSUPPORTED;
#define TDSE_RP_CASE(I, CP, NWR, NWC, MINB) \
    case I: return rp_launch_one<FD, CP, NWR, NWC, MINB, rp_clusterable(I), rp_rk_capable(I)>(g, p, in, out, ef, dtp, order, s, ob, n_steps);
    switch (p.variant) {
        TDSE_RP_CASE(0, 4, 1, 1, 8)
        TDSE_RP_CASE(1, 4, 2, 1, 4)
        TDSE_RP_CASE(2, 4, 4, 1, 2)
        TDSE_RP_CASE(3, 4, 8, 1, 1)
        TDSE_RP_CASE(4, 4, 4, 2, 1)
        case 5: return rp_launch_persist<FD, 2, 1, 2, 4>(g, p, in, out, ef, dtp, order, s, ob, n_steps);
        case 6: return rp_launch_persist<FD, 2, 2, 2, 2>(g, p, in, out, ef, dtp, order, s, ob, n_steps);
        case 7: return rp_launch_persist<FD, 2, 4, 2, 1>(g, p, in, out, ef, dtp, order, s, ob, n_steps);
    }
#undef TDSE_RP_CASE
    return TDSE_ERR_UNSUPPORTED;
}

}  // namespace tdse
