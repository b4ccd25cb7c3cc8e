// tdse_taylor_rt.cuh -- temporally blocked Taylor step on REGISTER tiles: all orders of one step in one pass over
// HBM (32 B/point/step), with the current Taylor term AND the accumulator of every point held in registers.
//
// Method: Eq. 37 (reading R-G6): F(t+dt) = sum_{k=0..P} F^(k), F^(k) = (-i dt/k) H F^(k-1).  NS asks for the
// orders to be "temporally blocked in shared memory ... shrinking halo"; the paper launches one kernel per order
// (P:458).  Here a CTA owns all n_l partial waves of WT = CP*NCG radial columns; a thread owns a patch of RP rows x
// CP adjacent columns.  Per order a thread reads from shared memory only the values of OTHER threads that its
// patch touches (radial neighbours left/right, l-1 above, l+1 below) and publishes only its own boundary values.
// The real symmetric H acts on re and im separately, so the term kept is u_k = (dt H)^k psi (coefficients
// pre-multiplied by dt once per step) and the factor (-i)^k/k! is applied when u_k is added to the accumulator:
// the same polynomial as Eq. 37 in another rounding order.
//
// Shared-memory tile: two buffers [ROWS + 2][CP planes][PLP] complex128; column c lives in plane c % CP, slot
// c / CP + 1; slots 0 and NCG + 1 and the rows 0 and ROWS + 1 are zero for ever: they are the Dirichlet walls
// and the truncation f_{-1} = f_L = 0.  PLP = 8/CP (mod 8) makes the coalesced fill, the patch loads and
// the neighbour loads bank-conflict free.  A tile at a wall starts exactly at the wall (the zero pad IS the wall),
// so no thread needs a domain predicate unless the whole grid is narrower than one tile (MASK).
#pragma once
#include <algorithm>

#include "tdse_device.cuh"

namespace tdse {

template <int FD, int RP, int CP, int NRG, int NCG>
struct RtGeom {
    static constexpr int HW = (FD == 3) ? 1 : 2;
    static constexpr int RPT = RP, CPT = CP;
    static constexpr int ROWS = RP * NRG;               // rows held by the CTA (>= n_l)
    static constexpr int WT = CP * NCG;                 // tile columns
    static constexpr int NT = NRG * NCG;                // threads
    static constexpr int PAD = (CP == 4) ? 2 : 4;
    static constexpr int PLP = NCG + PAD;               // plane pitch (slots); NCG % 8 == 0
    static constexpr int ROWP = CP * PLP;               // row pitch (double2)
    static constexpr int BUF = (ROWS + 2) * ROWP;       // one buffer (double2)
    static constexpr size_t SMEM = (size_t)2 * BUF * sizeof(double2) + (size_t)ROWS * 4 * sizeof(double);
    static_assert(NCG % 8 == 0, "NCG must be a multiple of 8");
    static_assert(HW <= CP, "radial halo wider than the patch");
};

// element (row, column c) of a buffer; row in [-1, ROWS], c in [-CP, WT + CP)
template <class G>
__device__ __forceinline__ int rt_off(int row, int c) {
    return (row + 1) * G::ROWP + (c & (G::CPT - 1)) * G::PLP + (c / G::CPT) + 1;
}

// grid = (n_tiles, batch), block = NT, dynamic shared = G::SMEM.  W = interior columns per tile = WT - 2*order*HW.
template <int FD, int RP, int CP, int NRG, int NCG, bool MASK, int MINB>
__global__ void __launch_bounds__(NRG *NCG, MINB)
taylor_rt_kernel(GridDev g, const double2 *__restrict__ in, double2 *__restrict__ out, const double *__restrict__ ef,
                 const double *__restrict__ dtp, int order, int W) {
    using G = RtGeom<FD, RP, CP, NRG, NCG>;
    constexpr int HW = G::HW, ROWS = G::ROWS, WT = G::WT, NT = G::NT, PLP = G::PLP, ROWP = G::ROWP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2 *buf0 = reinterpret_cast<double2 *>(smem_raw);
    double2 *buf1 = buf0 + G::BUF;
    double *rowtab = reinterpret_cast<double *>(buf1 + G::BUF);     // [ROWS][4] = {c_{l-1}, c_l, l(l+1), 0}

    const int tid = threadIdx.x;
    const int L = g.n_l, N = g.n_r;
    const int b = blockIdx.y, t = blockIdx.x;
    const int H = order * HW;
    // tile start: interior [t*W, (t+1)*W) needs H halo columns per side unless the side is a wall
    int start = t * W - H;
    if (start > N - WT) start = N - WT;
    if (start < 0) start = 0;
    const double2 *src_g = in + (size_t)b * L * N;
    const double2 z2 = make_double2(0.0, 0.0);

    // ---- zero pads (both buffers), coefficient table, tile fill -----------------------------------------------
    for (int i = tid; i < 2 * G::BUF; i += NT) {
        const int e = i % G::BUF, row = e / ROWP, sl = (e % ROWP) % PLP;
        if (row == 0 || row == ROWS + 1 || sl == 0 || sl > NCG || row > L) buf0[i] = z2;   // buf1 follows buf0
    }
    for (int r = tid; r < ROWS; r += NT) {
        rowtab[4 * r + 0] = (r >= 1 && r < L) ? __ldg(g.cl + r - 1) : 0.0;
        rowtab[4 * r + 1] = (r + 1 < L) ? __ldg(g.cl + r) : 0.0;
        rowtab[4 * r + 2] = (double)(r * (r + 1));
        rowtab[4 * r + 3] = 0.0;
    }
    {
        const int total = L * WT;
#pragma unroll 4
        for (int i = tid; i < total; i += NT) {
            const int row = i / WT, c = i - row * WT;
            const int j = start + c;
            double2 v = z2;
            if (!MASK || j < N) v = __ldg(src_g + (size_t)row * N + j);
            buf0[rt_off<G>(row, c)] = v;
        }
    }
    __syncthreads();

    // ---- per-thread patch ------------------------------------------------------------------------------------
    const int cgi = tid % NCG, rgi = tid / NCG;
    const int r0 = rgi * RP, c0 = cgi * CP;
    const double dt = *dtp;
    const double e_b = __ldg(ef + b);
    const double c1 = dt * g.c1, c2 = dt * g.c2;
    double Dq[CP], Cq[CP], Eq[CP];
    bool dom[CP];
#pragma unroll
    for (int q = 0; q < CP; ++q) {
        const int j = start + c0 + q;
        dom[q] = !MASK || j < N;
        const int jj = dom[q] ? j : 0;
        Dq[q] = dt * __ldg(g.vj + jj);
        Cq[q] = dt * __ldg(g.cen + jj);
        Eq[q] = dt * (e_b * (g.dr * (double)(jj + 1)));
    }
    // own patch: slot cgi + 1 of plane q, rows r0 .. r0 + RP - 1
    const int own = (r0 + 1) * ROWP + cgi + 1;
    double2 T[RP][CP], A[RP][CP];
#pragma unroll
    for (int r = 0; r < RP; ++r)
#pragma unroll
        for (int q = 0; q < CP; ++q) {
            T[r][q] = buf0[own + r * ROWP + q * PLP];
            A[r][q] = T[r][q];
        }

    double inv_fact = 1.0;
    for (int k = 1; k <= order; ++k) {
        const double2 *src = (k & 1) ? buf0 : buf1;
        double2 *dst = (k & 1) ? buf1 : buf0;
        const double2 *so = src + own;
        double2 *dn = dst + own;
        inv_fact = inv_fact / (double)k;

        double2 prev[CP];                                   // old values of the row above the one being updated
#pragma unroll
        for (int q = 0; q < CP; ++q) prev[q] = so[-ROWP + q * PLP];
#pragma unroll
        for (int r = 0; r < RP; ++r) {
            const double2 rc = *reinterpret_cast<const double2 *>(rowtab + 4 * (r0 + r));   // {c_{l-1}, c_l}
            const double ll1 = rowtab[4 * (r0 + r) + 2];                                     // l(l+1)
            double2 below[CP];
            if (r == RP - 1) {
#pragma unroll
                for (int q = 0; q < CP; ++q) below[q] = so[RP * ROWP + q * PLP];
            }
            const double2 lf1 = so[r * ROWP + (CP - 1) * PLP - 1];          // column c0 - 1
            const double2 rg1 = so[r * ROWP + 1];                            // column c0 + CP
            double2 lf2 = z2, rg2 = z2;
            if (FD == 5) {
                lf2 = so[r * ROWP + (CP - 2) * PLP - 1];                     // column c0 - 2
                rg2 = so[r * ROWP + PLP + 1];                                // column c0 + CP + 1
            }
            double2 nw[CP];
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                const double2 f = T[r][q];
                const double2 m1 = (q > 0) ? T[r][q > 0 ? q - 1 : 0] : lf1;
                const double2 p1 = (q < CP - 1) ? T[r][q < CP - 1 ? q + 1 : 0] : rg1;
                const double2 lo = prev[q];
                const double2 up = (r < RP - 1) ? T[r < RP - 1 ? r + 1 : 0][q] : below[q];
                const double d = fma(ll1, Cq[q], Dq[q]);
                double hx = c1 * (m1.x + p1.x), hy = c1 * (m1.y + p1.y);
                if (FD == 5) {
                    const double2 m2 = (q > 1) ? T[r][q > 1 ? q - 2 : 0] : ((q == 1) ? lf1 : lf2);
                    const double2 p2 = (q < CP - 2) ? T[r][q < CP - 2 ? q + 2 : 0] : ((q == CP - 2) ? rg1 : rg2);
                    hx = fma(c2, m2.x + p2.x, hx);
                    hy = fma(c2, m2.y + p2.y, hy);
                }
                hx = fma(d, f.x, hx);
                hy = fma(d, f.y, hy);
                const double wx = fma(rc.y, up.x, rc.x * lo.x), wy = fma(rc.y, up.y, rc.x * lo.y);
                hx = fma(Eq[q], wx, hx);
                hy = fma(Eq[q], wy, hy);
                nw[q] = make_double2(hx, hy);
                if (MASK && !dom[q]) nw[q] = z2;
            }
#pragma unroll
            for (int q = 0; q < CP; ++q) { prev[q] = T[r][q]; T[r][q] = nw[q]; }
            if (k < order) {
                // publish what other threads read: the HW outermost columns of every row, all columns of the
                // first and the last row of the patch
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    const bool edge_col = (q < HW) || (q >= CP - HW);
                    const bool edge_row = (r == 0) || (r == RP - 1);
                    if (edge_col || edge_row) dn[r * ROWP + q * PLP] = nw[q];
                }
            }
        }
        // acc += (-i)^k / k! * u_k
        const double s = inv_fact;
        switch (k & 3) {
            case 0:
#pragma unroll
                for (int r = 0; r < RP; ++r)
#pragma unroll
                    for (int q = 0; q < CP; ++q) { A[r][q].x = fma(s, T[r][q].x, A[r][q].x); A[r][q].y = fma(s, T[r][q].y, A[r][q].y); }
                break;
            case 1:   // -i (x + i y) = y - i x
#pragma unroll
                for (int r = 0; r < RP; ++r)
#pragma unroll
                    for (int q = 0; q < CP; ++q) { A[r][q].x = fma(s, T[r][q].y, A[r][q].x); A[r][q].y = fma(-s, T[r][q].x, A[r][q].y); }
                break;
            case 2:
#pragma unroll
                for (int r = 0; r < RP; ++r)
#pragma unroll
                    for (int q = 0; q < CP; ++q) { A[r][q].x = fma(-s, T[r][q].x, A[r][q].x); A[r][q].y = fma(-s, T[r][q].y, A[r][q].y); }
                break;
            default:  // +i (x + i y) = -y + i x
#pragma unroll
                for (int r = 0; r < RP; ++r)
#pragma unroll
                    for (int q = 0; q < CP; ++q) { A[r][q].x = fma(-s, T[r][q].y, A[r][q].x); A[r][q].y = fma(s, T[r][q].x, A[r][q].y); }
                break;
        }
        __syncthreads();
    }

    // ---- psi(t + dt): park the sums in buf0 (free after the last barrier: the last order read buf[(P-1)&1] and
    // wrote nothing), then store the interior columns coalesced along r
    double2 *stage = (order & 1) ? buf1 : buf0;            // the buffer NOT read by the last order
#pragma unroll
    for (int r = 0; r < RP; ++r)
#pragma unroll
        for (int q = 0; q < CP; ++q) stage[own + r * ROWP + q * PLP] = A[r][q];
    __syncthreads();
    {
        const int lo_c = t * W - start;                      // first interior column (tile coordinates)
        int wint = N - t * W;
        if (wint > W) wint = W;
        double2 *dst_g = out + (size_t)b * L * N + (size_t)t * W;
        const int total = L * wint;
        for (int i = tid; i < total; i += NT) {
            const int row = i / wint, cc = i - row * wint;
            dst_g[(size_t)row * N + cc] = stage[rt_off<G>(row, lo_c + cc)];
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// Host side: choice of the instantiation and launch.
// ------------------------------------------------------------------------------------------------------
struct RtPlan { int ok, variant, W, WT, n_tiles, threads; size_t smem; };

struct RtVariant { int rp, cp, nrg, ncg, minb; };
// instantiations (RP, CP, NRG, NCG, min CTAs/SM); rows = RP*NRG must cover n_l
constexpr RtVariant kRtVariants[] = {
    {4, 4, 2, 64, 2},   // n_l <= 8 : 128 threads, 256 columns
    {4, 4, 4, 32, 2},   // n_l <= 16: 128 threads, 128 columns
    {4, 4, 4, 64, 1},   // n_l <= 16: 256 threads, 256 columns, one CTA per SM
    {4, 4, 8, 32, 1},   // n_l <= 32: 256 threads, 128 columns
    {4, 4, 8, 16, 2},   // n_l <= 32: 128 threads,  64 columns
};
constexpr int kNumRtVariants = sizeof(kRtVariants) / sizeof(kRtVariants[0]);

inline size_t rt_smem(const RtVariant &v) {
    const int pad = (v.cp == 4) ? 2 : 4;
    const size_t buf = (size_t)(v.rp * v.nrg + 2) * v.cp * (v.ncg + pad);
    return 2 * buf * sizeof(double2) + (size_t)v.rp * v.nrg * 4 * sizeof(double);
}

// pick the variant that computes the fewest columns in total (halo redundancy + ragged last tile), preferring
// two CTAs per SM on ties
inline RtPlan rt_plan(const tdse_grid &g, int order, int force_variant) {
    RtPlan best{};
    const int hw = (g.fd_order == 3) ? 1 : 2, H = order * hw;
    double best_cost = 0.0;
    for (int i = 0; i < kNumRtVariants; ++i) {
        if (force_variant >= 0 && i != force_variant) continue;
        const RtVariant &v = kRtVariants[i];
        if (v.rp * v.nrg < g.n_l) continue;
        if (v.rp * v.nrg >= 2 * g.n_l && v.nrg > 2) continue;          // more than half of the rows would be padding
        const int WT = v.cp * v.ncg;
        int W = WT - 2 * H, n_tiles = 1;
        if (g.n_r <= WT) {
            W = g.n_r;                                                  // the whole radial box in one tile: walls on both sides
        } else {
            if (W < WT / 4 || W < 2) continue;
            n_tiles = (g.n_r + W - 1) / W;
        }
        double cost = (double)n_tiles * WT * (v.rp * v.nrg);
        if (v.minb < 2) cost *= 1.15;                                  // exposed load/store phases with one CTA per SM
        if (!best.ok || cost < best_cost) {
            best_cost = cost;
            best.ok = 1; best.variant = i; best.W = W; best.WT = WT; best.n_tiles = n_tiles;
            best.threads = v.nrg * v.ncg; best.smem = rt_smem(v);
        }
    }
    return best;
}

template <int FD, int RP, int CP, int NRG, int NCG, int MINB>
inline int rt_launch_one(const GridDev &g, const RtPlan &p, const double2 *in, double2 *out, const double *ef,
                         const double *dtp, int order, cudaStream_t s) {
    using G = RtGeom<FD, RP, CP, NRG, NCG>;
    static bool attr_set[2] = {false, false};
    const bool mask = g.n_r < G::WT;
    if (!attr_set[mask]) {
        cudaError_t e = mask ? cudaFuncSetAttribute(taylor_rt_kernel<FD, RP, CP, NRG, NCG, true, MINB>,
                                                    cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM)
                             : cudaFuncSetAttribute(taylor_rt_kernel<FD, RP, CP, NRG, NCG, false, MINB>,
                                                    cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM);
        if (e != cudaSuccess) return TDSE_ERR_CUDA;
        e = mask ? cudaFuncSetAttribute(taylor_rt_kernel<FD, RP, CP, NRG, NCG, true, MINB>,
                                        cudaFuncAttributePreferredSharedMemoryCarveout, 100)
                 : cudaFuncSetAttribute(taylor_rt_kernel<FD, RP, CP, NRG, NCG, false, MINB>,
                                        cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) return TDSE_ERR_CUDA;
        attr_set[mask] = true;
    }
    dim3 grid(p.n_tiles, g.batch);
    if (mask)
        taylor_rt_kernel<FD, RP, CP, NRG, NCG, true, MINB><<<grid, G::NT, G::SMEM, s>>>(g, in, out, ef, dtp, order, p.W);
    else
        taylor_rt_kernel<FD, RP, CP, NRG, NCG, false, MINB><<<grid, G::NT, G::SMEM, s>>>(g, in, out, ef, dtp, order, p.W);
    return cudaGetLastError() == cudaSuccess ? TDSE_OK : TDSE_ERR_CUDA;
}

inline int launch_taylor_rt(const GridDev &g, const RtPlan &p, const double2 *in, double2 *out, const double *ef,
                            const double *dtp, int order, cudaStream_t s) {
    if (!p.ok) return TDSE_ERR_UNSUPPORTED;
#define TDSE_RT_CASE(I, RP, CP, NRG, NCG, MINB)                                                          \
    case I:                                                                                              \
        return (g.fd == 3) ? rt_launch_one<3, RP, CP, NRG, NCG, MINB>(g, p, in, out, ef, dtp, order, s)  \
                           : rt_launch_one<5, RP, CP, NRG, NCG, MINB>(g, p, in, out, ef, dtp, order, s);
    switch (p.variant) {
        TDSE_RT_CASE(0, 4, 4, 2, 64, 2)
        TDSE_RT_CASE(1, 4, 4, 4, 32, 2)
        TDSE_RT_CASE(2, 4, 4, 4, 64, 1)
        TDSE_RT_CASE(3, 4, 4, 8, 32, 1)
        TDSE_RT_CASE(4, 4, 4, 8, 16, 2)
    }
#undef TDSE_RT_CASE
    return TDSE_ERR_UNSUPPORTED;
}

}  // namespace tdse
