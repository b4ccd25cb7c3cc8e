// tdse_taylor_rp.cuh -- temporally blocked Taylor step, v3: persistent CTAs on register patches.
//
// Method: Eq. 37 (reading R-G6): F(t+dt) = sum_{k=0..P} F^(k), F^(k) = (-i dt/k) H F^(k-1); all P orders of a
// step are applied in ONE pass over HBM (32 B/point/step; the paper launches one kernel per order).
//
// Work item = (member b, radial tile t).  A warp owns 4 partial waves x 128 radial columns of the tile, a thread a
// patch of 4 rows x 4 adjacent columns whose current term u_k AND accumulator stay in registers for the whole
// step.  What differs from v2 (tdse_taylor_rt.cuh):
//   * no shared-memory tile: a thread loads its patch straight from global memory (64 contiguous bytes per row,
//     a warp reads 2 KB contiguous) and stores the result the same way;
//   * radial neighbours (columns c0-1, c0+4 [, c0-2, c0+5]) come from the adjacent LANES by warp shuffle;
//     only the l-1 / l+1 rows cross warps, through a small double-buffered shared-memory exchange
//     (lane-contiguous, conflict free) -- 16 instead of 28 shared-memory accesses per thread and order;
//   * CTAs are persistent (grid = resident CTAs), the zero rows / coefficient table are set up once, and the next
//     work item is prefetched into L2 (cp.async.bulk.prefetch.L2) while the current one is being computed;
//   * the operator is applied as H' = H / c1 (c1 = first off-diagonal stencil weight), so the radial part is
//     (f_{j-1} + f_{j+1}) + d' f_j with no multiply on the neighbours; u'_k = H'^k psi and the accumulator takes
//     (-i)^k (dt c1)^k / k! u'_k -- the same polynomial as Eq. 37 in another rounding order.  The coupling weight
//     c_l E r_j / c1 of the (l, l+1) pair is formed once and used for both rows.  12.25 (3-point) / 16.25 (5-point)
//     FP64 instructions per point-update instead of 16.3 / 20.
#pragma once
#include <algorithm>

#include "tdse_device.cuh"

namespace tdse {

constexpr int kRpRows = 4, kRpCols = 4, kRpWT = 128;     // patch rows, patch columns, tile columns (32 lanes x 4)

// shared memory: exchange buffers [2 parities][NW warps][2 (top,bottom)][4 planes][32 lanes] double2, row table
template <int NW>
struct RpSmem {
    double2 xch[2][NW][2][kRpCols][32];
    double rowtab[NW * kRpRows][4];        // {c_{l-1}, c_l, l(l+1), 0}
};

__device__ __forceinline__ double2 shfl_up2(double2 v) {
    return make_double2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ double2 shfl_dn2(double2 v) {
    return make_double2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ void l2_prefetch_bulk(const void *p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// tile start of tile t: interior [t*W, (t+1)*W) plus H halo columns per side, clamped so that a tile at a wall
// starts (ends) exactly at the wall: the zero beyond the tile IS the Dirichlet wall.
__device__ __forceinline__ int rp_start(int t, int W, int H, int N) {
    int start = t * W - H;
    if (start > N - kRpWT) start = N - kRpWT;
    if (start < 0) start = 0;
    return start;
}

// grid = persistent CTAs, block = NW*32.  n_l <= 4*NW.  MASK: n_r < 128 (single tile, columns >= n_r held at zero).
template <int FD, int NW, bool MASK, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB)
taylor_rp_kernel(GridDev g, const double2 *__restrict__ in, double2 *__restrict__ out, const double *__restrict__ ef,
                 const double *__restrict__ dtp, int order, int W, int n_tiles, int n_items) {
    constexpr int RP = kRpRows, CP = kRpCols, WT = kRpWT, HW = (FD == 3) ? 1 : 2;
    extern __shared__ __align__(16) unsigned char rp_smem_raw[];
    RpSmem<NW> &sm = *reinterpret_cast<RpSmem<NW> *>(rp_smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = g.n_l, N = g.n_r;
    const int H = order * HW;
    const int r0 = warp * RP, c0 = lane * CP;
    const double2 z2 = make_double2(0.0, 0.0);

    for (int r = threadIdx.x; r < NW * RP; r += NW * 32) {
        sm.rowtab[r][0] = (r >= 1 && r < L) ? __ldg(g.cl + r - 1) : 0.0;
        sm.rowtab[r][1] = (r + 1 < L) ? __ldg(g.cl + r) : 0.0;
        sm.rowtab[r][2] = (double)(r * (r + 1));
        sm.rowtab[r][3] = 0.0;
    }
    __syncthreads();

    const double dt = *dtp;
    const double inv_c1 = 1.0 / g.c1;
    const double kappa = dt * g.c1;                 // u'_k = (H/c1)^k psi  ->  weight (dt c1)^k / k!
    const double c2p = g.c2 * inv_c1;               // 5-point: second off-diagonal weight / c1 (= -1/16)

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int b = item / n_tiles, t = item - b * n_tiles;
        const int start = rp_start(t, W, H, N);
        const double2 *src_g = in + (size_t)b * L * N + start;
        // ---- prefetch the next item of this CTA into L2 (one lane per row) ------------------------------------
        {
            const int nitem = item + gridDim.x;
            if (nitem < n_items && threadIdx.x < L) {
                const int nb = nitem / n_tiles, nt = nitem - nb * n_tiles;
                const int ns = rp_start(nt, W, H, N);
                const int ncols = (N < WT) ? N : WT;
                l2_prefetch_bulk(in + ((size_t)nb * L + threadIdx.x) * N + ns, (unsigned)(ncols * sizeof(double2)));
            }
        }
        // ---- per-column coefficients (scaled by 1/c1) ----------------------------------------------------------
        const double e_b = __ldg(ef + b);
        double Dq[CP], Cq[CP], Eq[CP];
        bool dom[CP];
#pragma unroll
        for (int q = 0; q < CP; ++q) {
            const int j = start + c0 + q;
            dom[q] = !MASK || j < N;
            const int jj = dom[q] ? j : 0;
            Dq[q] = inv_c1 * __ldg(g.vj + jj);
            Cq[q] = inv_c1 * __ldg(g.cen + jj);
            Eq[q] = inv_c1 * (e_b * (g.dr * (double)(jj + 1)));
        }
        // ---- own patch straight from global memory -------------------------------------------------------------
        double2 T[RP][CP], A[RP][CP];
#pragma unroll
        for (int r = 0; r < RP; ++r)
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                double2 v = z2;
                if (r0 + r < L && dom[q]) v = __ldg(src_g + (size_t)(r0 + r) * N + c0 + q);
                T[r][q] = v;
                A[r][q] = v;
            }
        // publish rows 0 and RP-1 of u_0 for the neighbouring warps
#pragma unroll
        for (int q = 0; q < CP; ++q) {
            sm.xch[0][warp][0][q][lane] = T[0][q];
            sm.xch[0][warp][1][q][lane] = T[RP - 1][q];
        }
        __syncthreads();

        double sk = 1.0;
        for (int k = 1; k <= order; ++k) {
            const int pr = (k - 1) & 1, pw = k & 1;
            sk = sk * (kappa / (double)k);
            double2 lo[CP], below[CP];
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                lo[q] = (warp > 0) ? sm.xch[pr][warp > 0 ? warp - 1 : 0][1][q][lane] : z2;
                below[q] = (warp < NW - 1) ? sm.xch[pr][warp < NW - 1 ? warp + 1 : 0][0][q][lane] : z2;
            }
            double alo[CP];
            {
                const double clo = sm.rowtab[r0][0];
#pragma unroll
                for (int q = 0; q < CP; ++q) alo[q] = clo * Eq[q];
            }
#pragma unroll
            for (int r = 0; r < RP; ++r) {
                const double cup = sm.rowtab[r0 + r][1];
                const double ll1 = sm.rowtab[r0 + r][2];
                double2 lf1 = shfl_up2(T[r][CP - 1]);       // column c0 - 1 from lane - 1
                double2 rg1 = shfl_dn2(T[r][0]);            // column c0 + CP from lane + 1
                if (lane == 0) lf1 = z2;
                if (lane == 31) rg1 = z2;
                double2 lf2 = z2, rg2 = z2;
                if (FD == 5) {
                    lf2 = shfl_up2(T[r][CP - 2]);
                    rg2 = shfl_dn2(T[r][1]);
                    if (lane == 0) lf2 = z2;
                    if (lane == 31) rg2 = z2;
                }
                double2 nw[CP];
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    const double2 f = T[r][q];
                    const double2 m1 = (q > 0) ? T[r][q > 0 ? q - 1 : 0] : lf1;
                    const double2 p1 = (q < CP - 1) ? T[r][q < CP - 1 ? q + 1 : 0] : rg1;
                    const double2 up = (r < RP - 1) ? T[r < RP - 1 ? r + 1 : 0][q] : below[q];
                    const double d = fma(ll1, Cq[q], Dq[q]);
                    const double aup = cup * Eq[q];
                    double hx = m1.x + p1.x, hy = m1.y + p1.y;
                    if (FD == 5) {
                        const double2 m2 = (q > 1) ? T[r][q > 1 ? q - 2 : 0] : ((q == 1) ? lf1 : lf2);
                        const double2 p2 = (q < CP - 2) ? T[r][q < CP - 2 ? q + 2 : 0] : ((q == CP - 2) ? rg1 : rg2);
                        hx = fma(c2p, m2.x + p2.x, hx);
                        hy = fma(c2p, m2.y + p2.y, hy);
                    }
                    hx = fma(d, f.x, hx);
                    hy = fma(d, f.y, hy);
                    hx = fma(aup, up.x, hx);
                    hy = fma(aup, up.y, hy);
                    hx = fma(alo[q], lo[q].x, hx);
                    hy = fma(alo[q], lo[q].y, hy);
                    nw[q] = make_double2(hx, hy);
                    if (MASK && !dom[q]) nw[q] = z2;
                    alo[q] = aup;                           // c_l E r / c1 couples row l+1 back to row l
                }
#pragma unroll
                for (int q = 0; q < CP; ++q) { lo[q] = T[r][q]; T[r][q] = nw[q]; }
            }
            if (k < order) {
#pragma unroll
                for (int q = 0; q < CP; ++q) {
                    sm.xch[pw][warp][0][q][lane] = T[0][q];
                    sm.xch[pw][warp][1][q][lane] = T[RP - 1][q];
                }
            }
            // acc += (-i)^k (dt c1)^k / k! * u'_k
            const double s = sk;
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

        // ---- psi(t + dt): interior columns of the tile straight from registers ---------------------------------
        {
            const int lo_c = t * W - start;                  // first interior column (tile coordinates)
            int wint = N - t * W;
            if (wint > W) wint = W;
            double2 *dst_g = out + (size_t)b * L * N + start;
#pragma unroll
            for (int q = 0; q < CP; ++q) {
                const int c = c0 + q;
                if (c >= lo_c && c < lo_c + wint) {
#pragma unroll
                    for (int r = 0; r < RP; ++r)
                        if (r0 + r < L) dst_g[(size_t)(r0 + r) * N + c] = A[r][q];
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------------------
struct RpPlan { int ok, nw, W, n_tiles, n_items, grid, minb; };

inline RpPlan rp_plan(const tdse_grid &g, int order, int n_sm) {
    RpPlan p{};
    if (g.n_l > 32) return p;
    const int hw = (g.fd_order == 3) ? 1 : 2, H = order * hw;
    p.nw = (g.n_l <= 4) ? 1 : (g.n_l <= 8) ? 2 : (g.n_l <= 16) ? 4 : 8;
    p.minb = 8 / p.nw;
    if (g.n_r <= kRpWT) { p.W = g.n_r; p.n_tiles = 1; }
    else {
        p.W = kRpWT - 2 * H;
        if (p.W < kRpWT / 4) return p;
        p.n_tiles = (g.n_r + p.W - 1) / p.W;
    }
    p.n_items = p.n_tiles * g.batch;
    p.grid = std::min(p.n_items, n_sm * p.minb);
    p.ok = 1;
    return p;
}

template <int FD, int NW, int MINB>
inline int rp_launch_one(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                         const double *dtp, int order, cudaStream_t s) {
    const bool mask = g.n_r < kRpWT;
    const int smem = (int)sizeof(RpSmem<NW>);
    static bool attr_set[2] = {false, false};
    if (!attr_set[mask]) {
        cudaError_t e = mask ? cudaFuncSetAttribute(taylor_rp_kernel<FD, NW, true, MINB>,
                                                    cudaFuncAttributeMaxDynamicSharedMemorySize, smem)
                             : cudaFuncSetAttribute(taylor_rp_kernel<FD, NW, false, MINB>,
                                                    cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return TDSE_ERR_CUDA;
        attr_set[mask] = true;
    }
    if (mask)
        taylor_rp_kernel<FD, NW, true, MINB><<<p.grid, NW * 32, smem, s>>>(g, in, out, ef, dtp, order, p.W, p.n_tiles, p.n_items);
    else
        taylor_rp_kernel<FD, NW, false, MINB><<<p.grid, NW * 32, smem, s>>>(g, in, out, ef, dtp, order, p.W, p.n_tiles, p.n_items);
    return cudaGetLastError() == cudaSuccess ? TDSE_OK : TDSE_ERR_CUDA;
}

inline int launch_taylor_rp(const GridDev &g, const RpPlan &p, const double2 *in, double2 *out, const double *ef,
                            const double *dtp, int order, cudaStream_t s) {
    if (!p.ok) return TDSE_ERR_UNSUPPORTED;
#define TDSE_RP_CASE(NW, MINB)                                                                     \
    case NW:                                                                                       \
        return (g.fd == 3) ? rp_launch_one<3, NW, MINB>(g, p, in, out, ef, dtp, order, s)          \
                           : rp_launch_one<5, NW, MINB>(g, p, in, out, ef, dtp, order, s);
    switch (p.nw) {
        TDSE_RP_CASE(1, 8)
        TDSE_RP_CASE(2, 4)
        TDSE_RP_CASE(4, 2)
        TDSE_RP_CASE(8, 1)
    }
#undef TDSE_RP_CASE
    return TDSE_ERR_UNSUPPORTED;
}

}  // namespace tdse
