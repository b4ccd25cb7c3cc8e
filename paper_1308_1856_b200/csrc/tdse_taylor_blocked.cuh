// tdse_taylor_blocked.cuh -- temporally blocked Taylor step: ALL orders of one step in a single pass over HBM.
//
// NS: "successive Taylor orders are temporally blocked in shared memory (term_k = (-i dt/k) H term_{k-1},
// acc += term_k, shrinking halo) so HBM traffic per step drops by about the order".  P:456 Eq. 37 defines the
// recursion; the paper launches one kernel per order, i.e. 64 B/point/order of traffic; here a CTA keeps
// a tile of ALL n_l partial waves x (W + 2*order*HW) radial points resident in shared memory (two term buffers),
// the accumulator in registers, and reads psi once / writes psi once per step: 32 B/point/step.
//
// Tile: because every partial wave is resident the l+-1 coupling needs no halo; the radial halo is order*HW
// points per side and shrinks by HW per order.  Thread (cg, rg) owns 2 adjacent columns x RPT rows; the two
// columns live in separate "planes" (even / odd columns) so that every shared-memory access of a warp is a
// run of consecutive 16-byte words (no bank conflicts) while the thread still gets one radial neighbour of each
// column for free from its own registers.
#pragma once
#include <algorithm>

#include "tdse_device.cuh"

namespace tdse {

struct BlockedCfg {
    int fd = 0, n_l = 0, n_r = 0, batch = 0;
    int rpt = 0, nrg = 0;            // rows per thread, row groups
    int width_override = 0;          // option "taylor_block_width" (0 = heuristic)
    int smem_limit = 0;              // opt-in shared memory per CTA
    int n_sm = 148;
};

struct BlockedPlan { int ok, W, WT, NCG, NT, threads; size_t smem; };

inline int blocked_configure(BlockedCfg *cfg, const tdse_grid &g) {
    cfg->fd = g.fd_order; cfg->n_l = g.n_l; cfg->n_r = g.n_r; cfg->batch = g.batch;
    cfg->rpt = (g.n_l <= 16) ? 4 : 8;
    cfg->nrg = (g.n_l + cfg->rpt - 1) / cfg->rpt;
    int dev = 0, lim = 0, sm = 148;
    if (cudaGetDevice(&dev) != cudaSuccess) return TDSE_ERR_CUDA;
    if (cudaDeviceGetAttribute(&lim, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return TDSE_ERR_CUDA;
    cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
    cfg->smem_limit = lim; cfg->n_sm = sm;
    return TDSE_OK;
}

// shared bytes of a tile of WT columns: two term buffers [n_l][2*(NCG+2)] complex128 + the c_l table
inline size_t blocked_smem(const BlockedCfg &c, int WT) {
    const int PL = WT / 2 + 2;
    return (size_t)2 * c.n_l * 2 * PL * sizeof(double2) + (size_t)(c.n_l + 1) * sizeof(double);
}

inline BlockedPlan blocked_plan(const BlockedCfg &c, int order) {
    BlockedPlan p{};
    if (c.n_l > 64 || c.nrg < 1) return p;                    // accumulator registers: rows are split over <= 8 groups
    const int hw = (c.fd == 3) ? 1 : 2, H = order * hw;
    const int wt_threads = (512 / c.nrg) * 2;                 // NT = (WT/2) * nrg <= 512
    auto wt_fit = [&](size_t budget) {
        int wt = (int)((budget - (c.n_l + 1) * 8) / ((size_t)c.n_l * 64)) * 2 - 4;
        if (wt > wt_threads) wt = wt_threads;
        return wt & ~1;
    };
    int W = 0;
    if (c.width_override > 0) {
        W = c.width_override & ~1;
    } else {
        const int w2 = wt_fit((size_t)c.smem_limit / 2 - 1024) - 2 * H;   // two CTAs per SM
        const int w1 = wt_fit((size_t)c.smem_limit) - 2 * H;              // one CTA per SM
        if (w2 >= 6 * H) W = w2;
        else if (w1 >= 2 * H) W = w1;
        else return p;
        // small problems: keep at least ~2 tiles per SM
        const long long want = ((long long)c.n_r * c.batch + 2LL * c.n_sm - 1) / (2LL * c.n_sm);
        int wmin = (int)std::max<long long>(4LL * H, (want + 1) & ~1LL);
        if (wmin < 16) wmin = 16;
        if (W > wmin) W = wmin;
        if (W > ((c.n_r + 1) & ~1)) W = (c.n_r + 1) & ~1;
        if (W < 2) W = 2;
        // equal tiles: the last tile of a row should not be mostly empty
        const int nt = (c.n_r + W - 1) / W;
        W = (((c.n_r + nt - 1) / nt) + 1) & ~1;
    }
    const int WT = W + 2 * H;
    if (W < 2 || WT > wt_threads || blocked_smem(c, WT) > (size_t)c.smem_limit) return p;
    p.ok = 1; p.W = W; p.WT = WT; p.NCG = WT / 2; p.NT = p.NCG * c.nrg;
    p.threads = (p.NT + 31) & ~31; p.smem = blocked_smem(c, WT);
    return p;
}

inline bool blocked_supported(const BlockedCfg &c, int order) { return blocked_plan(c, order).ok != 0; }

// grid = (ceil(n_r / W), batch); block = plan.threads; dynamic shared = plan.smem
template <int FD, int RPT>
__global__ void __launch_bounds__(512) taylor_blocked_kernel(GridDev g, const double2 *__restrict__ in,
                                                             double2 *__restrict__ out, const double *__restrict__ ef,
                                                             const double *__restrict__ dtp, int order, int W, int NCG,
                                                             int NRG) {
    constexpr int HW = (FD == 3) ? 1 : 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L = g.n_l, H = order * HW, WT = W + 2 * H;
    const int PL = NCG + 2, PITCH = 2 * PL;                 // per row: even plane [PL], odd plane [PL]
    double2 *buf0 = reinterpret_cast<double2 *>(smem_raw);
    double2 *buf1 = buf0 + (size_t)L * PITCH;
    double *cls = reinterpret_cast<double *>(buf1 + (size_t)L * PITCH);    // cls[l+1] = c_l, cls[0] = 0

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int b = blockIdx.y, j0 = blockIdx.x * W;
    const double2 *src_g = in + (size_t)b * L * g.n_r;

    // ---- stage psi (zero outside the radial box); tile column c <-> plane (c+2)&1, slot (c+2)>>1
    for (int i = tid; i < L * WT; i += nthr) {
        const int r = i / WT, c = i - r * WT;
        const int j = j0 - H + c;
        double2 v = make_double2(0.0, 0.0);
        if (j >= 0 && j < g.n_r) v = __ldg(src_g + (size_t)r * g.n_r + j);
        buf0[r * PITCH + ((c + 2) & 1) * PL + ((c + 2) >> 1)] = v;
    }
    for (int i = tid; i < L * 4; i += nthr) {               // pad slots 0 and PL-1 of both planes, both buffers
        const int r = i >> 2, q = i & 3;
        const int off = r * PITCH + (q & 1) * PL + ((q >> 1) ? (PL - 1) : 0);
        buf0[off] = make_double2(0.0, 0.0);
        buf1[off] = make_double2(0.0, 0.0);
    }
    for (int i = tid; i <= L; i += nthr) cls[i] = (i == 0) ? 0.0 : __ldg(g.cl + i - 1);
    __syncthreads();

    const int cg = tid % NCG, rg = tid / NCG;
    const bool worker = rg < NRG;
    const int r0 = rg * RPT;
    const int c0 = 2 * cg;                                   // tile columns c0 (even plane) and c0 + 1 (odd plane)
    const int jA = j0 - H + c0, jB = jA + 1;
    const bool domA = jA >= 0 && jA < g.n_r, domB = jB >= 0 && jB < g.n_r;
    const bool intA = domA && c0 >= H && c0 < H + W, intB = domB && (c0 + 1) >= H && (c0 + 1) < H + W;
    const int slot = cg + 1;
    const double dt = *dtp;
    const double e_b = __ldg(ef + b);
    double vjA = 0.0, cenA = 0.0, erA = 0.0, vjB = 0.0, cenB = 0.0, erB = 0.0;
    if (domA) { vjA = __ldg(g.vj + jA); cenA = __ldg(g.cen + jA); erA = e_b * (g.dr * (double)(jA + 1)); }
    if (domB) { vjB = __ldg(g.vj + jB); cenB = __ldg(g.cen + jB); erB = e_b * (g.dr * (double)(jB + 1)); }

    double2 accA[RPT], accB[RPT];
#pragma unroll
    for (int rr = 0; rr < RPT; ++rr) {
        accA[rr] = make_double2(0.0, 0.0); accB[rr] = make_double2(0.0, 0.0);
        if (worker && r0 + rr < L) {
            accA[rr] = buf0[(r0 + rr) * PITCH + slot];
            accB[rr] = buf0[(r0 + rr) * PITCH + PL + slot];
        }
    }

    double2 *src = buf0, *dst = buf1;
    for (int k = 1; k <= order; ++k) {
        const int lo_k = k * HW, hi_k = WT - k * HW;
        const bool vA = c0 >= lo_k && c0 < hi_k, vB = (c0 + 1) >= lo_k && (c0 + 1) < hi_k;
        if (worker && (vA || vB)) {
            // fold the Taylor factor s = dt/k into the coefficients: term_k = (-i s) H term_{k-1}   (Eq. 37)
            const double s = dt / (double)k;
            const double sc1 = s * g.c1, sc2 = s * g.c2;
            const double svA = s * vjA, scA = s * cenA, seA = s * erA;
            const double svB = s * vjB, scB = s * cenB, seB = s * erB;
            const double2 *eS = src + slot, *oS = src + PL + slot;        // own even / odd column of row 0
            double2 *eD = dst + slot, *oD = dst + PL + slot;
            const double2 z = make_double2(0.0, 0.0);
            double2 loA = z, loB = z;
            if (r0 > 0) { loA = eS[(r0 - 1) * PITCH]; loB = oS[(r0 - 1) * PITCH]; }
            double2 fA = eS[r0 * PITCH], fB = oS[r0 * PITCH];
#pragma unroll
            for (int rr = 0; rr < RPT; ++rr) {
                const int r = r0 + rr;
                if (r < L) {
                    double2 upA = z, upB = z;
                    if (r + 1 < L) { upA = eS[(r + 1) * PITCH]; upB = oS[(r + 1) * PITCH]; }
                    const double2 l1 = oS[r * PITCH - 1];                 // column c0 - 1
                    const double2 r1 = eS[r * PITCH + 1];                 // column c0 + 2
                    const double ll1 = (double)(r * (r + 1));
                    const double cm = cls[r], cp = cls[r + 1];
                    const double dA = fma(ll1, scA, svA), dB = fma(ll1, scB, svB);
                    const double cmA = seA * cm, cpA = seA * cp, cmB = seB * cm, cpB = seB * cp;
                    double hAx = fma(cpA, upA.x, cmA * loA.x), hAy = fma(cpA, upA.y, cmA * loA.y);
                    double hBx = fma(cpB, upB.x, cmB * loB.x), hBy = fma(cpB, upB.y, cmB * loB.y);
                    if (FD == 5) {
                        const double2 l2 = eS[r * PITCH - 1];             // column c0 - 2
                        const double2 r2 = oS[r * PITCH + 1];             // column c0 + 3
                        hAx = fma(sc2, l2.x + r1.x, hAx); hAy = fma(sc2, l2.y + r1.y, hAy);
                        hBx = fma(sc2, l1.x + r2.x, hBx); hBy = fma(sc2, l1.y + r2.y, hBy);
                    }
                    hAx = fma(sc1, l1.x + fB.x, hAx); hAy = fma(sc1, l1.y + fB.y, hAy);
                    hBx = fma(sc1, fA.x + r1.x, hBx); hBy = fma(sc1, fA.y + r1.y, hBy);
                    hAx = fma(dA, fA.x, hAx); hAy = fma(dA, fA.y, hAy);
                    hBx = fma(dB, fB.x, hBx); hBy = fma(dB, fB.y, hBy);
                    // (-i)(x + i y) = y - i x
                    const double2 tA = domA ? make_double2(hAy, -hAx) : z;
                    const double2 tB = domB ? make_double2(hBy, -hBx) : z;
                    if (intA) { accA[rr].x += tA.x; accA[rr].y += tA.y; }
                    if (intB) { accB[rr].x += tB.x; accB[rr].y += tB.y; }
                    if (k < order) {
                        if (vA) eD[r * PITCH] = tA;
                        if (vB) oD[r * PITCH] = tB;
                    } else {
                        eD[r * PITCH] = accA[rr];                        // last order: park the sum for the coalesced store
                        oD[r * PITCH] = accB[rr];
                    }
                    loA = fA; loB = fB; fA = upA; fB = upB;
                }
            }
        }
        __syncthreads();
        double2 *t = src; src = dst; dst = t;
    }
    // ---- psi(t + dt): interior columns of the buffer written last (now `src`), coalesced along r
    double2 *dst_g = out + (size_t)b * L * g.n_r;
    for (int i = tid; i < L * W; i += nthr) {
        const int r = i / W, cc = i - r * W;
        const int j = j0 + cc, c = H + cc;
        if (j < g.n_r) dst_g[(size_t)r * g.n_r + j] = src[r * PITCH + ((c + 2) & 1) * PL + ((c + 2) >> 1)];
    }
}

inline int launch_taylor_blocked(const BlockedCfg &cfg, const GridDev &g, const double2 *in, double2 *out,
                                 const double *ef, const double *dtp, int order, cudaStream_t s) {
    const BlockedPlan p = blocked_plan(cfg, order);
    if (!p.ok) return TDSE_ERR_UNSUPPORTED;
    dim3 grid((g.n_r + p.W - 1) / p.W, g.batch);
#define TDSE_LAUNCH_BLOCKED(FDV, RPTV)                                                                             \
    do {                                                                                                           \
        static size_t set_smem = 0;                                                                                \
        if (set_smem < p.smem) {                                                                                   \
            if (cudaFuncSetAttribute(taylor_blocked_kernel<FDV, RPTV>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                     (int)cfg.smem_limit) != cudaSuccess)                                          \
                return TDSE_ERR_CUDA;                                                                              \
            set_smem = cfg.smem_limit;                                                                             \
        }                                                                                                          \
        taylor_blocked_kernel<FDV, RPTV><<<grid, p.threads, p.smem, s>>>(g, in, out, ef, dtp, order, p.W, p.NCG,   \
                                                                        cfg.nrg);                                  \
    } while (0)
    if (cfg.fd == 3 && cfg.rpt == 4) TDSE_LAUNCH_BLOCKED(3, 4);
    else if (cfg.fd == 3) TDSE_LAUNCH_BLOCKED(3, 8);
    else if (cfg.rpt == 4) TDSE_LAUNCH_BLOCKED(5, 4);
    else TDSE_LAUNCH_BLOCKED(5, 8);
#undef TDSE_LAUNCH_BLOCKED
    return cudaGetLastError() == cudaSuccess ? TDSE_OK : TDSE_ERR_CUDA;
}

}  // namespace tdse
