// tdse_tile_tma.cuh -- H.psi on (l, r) tiles fetched by TMA: the single-source variant of tile_kernel for grids with
// n_r % 8 == 0 (row a1: tdse_apply_H).
//
// tile_kernel stages its tile through registers (ld.global -> st.shared): at 5 CTAs per SM the loads in flight per
// SM are bounded by registers and the LSU pipe carries every byte twice (66 % busy on CFG4, profiles/).  Here a
// persistent CTA asks the TMA unit for the whole (8 + 2 rows) x (128 + 16 columns) box of the NEXT two work items
// while it computes the current one: the state array is described as a 4-D tensor [member][l][n_r/8][8 columns] so
// that everything outside the index box of a member (the rows l = -1 and l = n_l, the columns beyond the walls) is
// zero-filled by the hardware -- the Dirichlet walls of P:138-144 and the truncation f_{-1} = f_L = 0 cost nothing.
// The compute phase and the epilogue interface are those of tile_kernel.
#pragma once
#include "tdse_kernels.cuh"
#include "tdse_tma.cuh"            // mbarrier / TMA helpers, tensor maps

namespace tdse {

// measured on CFG4 / CFG5 (us): (stages, CTAs/SM, rows) = (2,3,8) 31.3 / 45.7; (3,3,8) 31.5 / 47.6; (2,4,8) 31.5 / 47.3;
// (2,2,16) 31.9 / 47.0; (4,2,8) 33.4 / 49.0; (3,2,16) 37.3 / 51.0
constexpr int kTtTW = 128, kTtTL = 8, kTtHalo = 8, kTtCols = kTtTW + 2 * kTtHalo, kTtRows = kTtTL + 2, kTtStages = 2;
constexpr int kTtMinB = 3;
constexpr unsigned kTtStageBytes = (unsigned)(kTtRows * kTtCols * sizeof(double2));

// grid = persistent CTAs, block = 256, dynamic shared = kTtStages * kTtStageBytes + 64.
// items = batch x l-tiles x r-tiles (r fastest).  Epi must have NRED == 0 and a plain input.
template <int FD, class Epi, bool VG = false>
__global__ void __launch_bounds__(256, kTtMinB)
tile_tma_kernel(GridDev g, Epi epi_in, const __grid_constant__ CUtensorMap tmap, int tiles_r, int tiles_l, int n_items) {
    static_assert(Epi::NRED == 0 && !Epi::CUSTOM_LOAD && !Epi::TWO_IN && !Epi::SCALED, "single-source epilogues only");
    constexpr int HW = (FD == 3) ? 1 : 2, COLS = kTtCols;
    extern __shared__ __align__(1024) unsigned char tt_smem[];
    double2 *st = reinterpret_cast<double2 *>(tt_smem);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(tt_smem + kTtStages * kTtStageBytes);
    Epi epi = epi_in;
    epi.begin();
    if (epi.skip_all()) return;
    const int tid = threadIdx.x;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kTtStages; ++s) mbar_init(&bars[s], 1);
    }
    __syncthreads();
    auto fetch = [&](const int item, const int s) {
        if (tid == 0 && item < n_items) {
            const int tr = item % tiles_r, rest = item / tiles_r, tl = rest % tiles_l, b = rest / tiles_l;
            fence_proxy_async_smem();
            mbar_expect_tx(&bars[s], kTtStageBytes);
            tma_load_4d(st + (size_t)s * kTtRows * COLS, &tmap, 0, tr * (kTtTW / 8) - kTtHalo / 8, tl * kTtTL - 1, b, &bars[s]);
        }
    };
#pragma unroll
    for (int s = 0; s < kTtStages; ++s) fetch(blockIdx.x + s * gridDim.x, s);

    const int tx = tid % kTtTW, ty = tid / kTtTW;
    unsigned phase = 0;          // bit s = parity of stage s
    int k = 0;
    double red[1] = {0.0};
    for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++k) {
        const int s = k % kTtStages;
        const int tr = item % tiles_r, rest = item / tiles_r, tl = rest % tiles_l, b = rest / tiles_l;
        const int j = tr * kTtTW + tx, l0 = tl * kTtTL;
        // per-column coefficients first: their latency overlaps the wait for the tile
        const double vj = (j < g.n_r) ? __ldg(g.vj + j) : 0.0, cen = (j < g.n_r) ? __ldg(g.cen + j) : 0.0;
        mbar_wait(&bars[s], (phase >> s) & 1u);
        phase ^= 1u << s;
        const bool cut_tile = g.j0 != nullptr && tr * kTtTW - kTtHalo < g.j0_max;       // the tile touches held points
        if (cut_tile) {          // centrifugal cut-off: held points read as zero (P H P)
            double2 *tile_s = st + (size_t)s * kTtRows * COLS;
            for (int i = tid; i < kTtRows * COLS; i += 256) {
                const int rr = i / COLS, cc = i - rr * COLS;
                if (held_pt(g, tl * kTtTL - 1 + rr, tr * kTtTW - kTtHalo + cc)) tile_s[i] = make_double2(0.0, 0.0);
            }
            __syncthreads();
        }
        if (j < g.n_r && epi.member_active(b)) {
            const double afield = epi.efield(b), rinv = 1.0 / (g.dr * (double)(j + 1));
            const double er = afield * (g.dr * (double)(j + 1));
            const int r0 = ty * (kTtTL / 2);
            const double2 *col = st + (size_t)s * kTtRows * COLS + (r0 + 1) * COLS + kTtHalo + tx;
            double2 lo = col[-COLS], f = col[0];
#pragma unroll
            for (int rr = 0; rr < kTtTL / 2; ++rr) {
                const int l = l0 + r0 + rr;
                if (l >= g.n_l) break;
                const double2 *c = col + rr * COLS;
                const double2 up = c[COLS];
                const double2 fm1 = c[-1], fp1 = c[1];
                double2 fm2 = fm1, fp2 = fp1;
                if (FD == 5) { fm2 = c[-2]; fp2 = c[2]; }
                const double d = fma((double)(l * (l + 1)), cen, vj);
                const double cm = (l > 0) ? __ldg(g.cl + l - 1) : 0.0;
                const double cp = __ldg(g.cl + l);
                double2 h = h_point<FD>(g, d, VG ? 0.0 : er, cm, cp, f, fm1, fp1, fm2, fp2, lo, up);
                if (VG) vg_couple<FD>(g, c, COLS, l, rinv, cm, cp, afield, lo, up, h);
                if (cut_tile && held_pt(g, l, j)) h = make_double2(0.0, 0.0);
                epi.point(b, l, j, ((size_t)b * g.n_l + l) * g.n_r + j, f, h, red);
                lo = f; f = up;
            }
        }
        __syncthreads();                                   // every thread is done with stage s
        fetch(item + kTtStages * gridDim.x, s);
    }
}

// 4-D tensor map of a state array for these kernels (by value; tdse_tma.cuh)
inline bool tile_tensor_map(CUtensorMap *m, const void *base, int n_r, int n_l, int batch) {
    return tma_map_member4d(m, base, n_r, n_l, batch, kTtRows, kTtCols);
}

}  // namespace tdse

namespace tdse {

// ------------------------------------------------------------------------------------------------------
// The fused Lanczos pass (EpiLanczosF, tdse_kernels.cuh) with TMA-fetched sources: the vector v_p is formed from up to
// three arrays (g_{p-1}, v_{p-1}, v_{p-2}); each source's box lands in its own raw buffer, the CTA combines them
// into the tile (halo included; zero-filled raw data combine to zero, so the walls stay exact), and as soon as the
// raw buffers are consumed the NEXT item's three boxes are requested -- they arrive during the H application,
// the epilogue and the other resident CTA's phases.  One partial of the two fused reductions per work item; a CTA
// signs off once (grid_finish).  grid = persistent CTAs, block = 256, 2 CTAs per SM (92 KB of shared memory each).
// ------------------------------------------------------------------------------------------------------
constexpr int kTt3Smem = 4 * (int)kTtStageBytes + 256;

template <int FD, class Epi, bool VG = false>
__global__ void __launch_bounds__(256, 2)
tile_tma3_kernel(GridDev g, Epi epi_in, RedCtx rc, const __grid_constant__ CUtensorMap tm0,
                 const __grid_constant__ CUtensorMap tm1, const __grid_constant__ CUtensorMap tm2, int tiles_r, int tiles_l,
                 int n_items) {
    static_assert(Epi::CUSTOM_LOAD && Epi::NRED > 0, "multi-source epilogues with fused reductions");
    constexpr int HW = (FD == 3) ? 1 : 2, COLS = kTtCols, ELEMS = kTtRows * kTtCols, NR = Epi::NRED;
    (void)HW;
    extern __shared__ __align__(1024) unsigned char t3_smem[];
    double2 *raw = reinterpret_cast<double2 *>(t3_smem);                       // [3][ELEMS]
    double2 *tile = raw + 3 * ELEMS;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(t3_smem + 4 * kTtStageBytes);
    double *red_s = reinterpret_cast<double *>(t3_smem + 4 * kTtStageBytes + 16);   // NR * 8 doubles
    int *flag = reinterpret_cast<int *>(t3_smem + 4 * kTtStageBytes + 16 + sizeof(double) * NR * 8);
    Epi epi = epi_in;
    epi.begin();
    if (epi.skip_all()) return;
    const int tid = threadIdx.x;
    if (tid == 0) mbar_init(bar, 1);
    __syncthreads();
    const int per_member = tiles_r * tiles_l;
    const bool has1 = epi.src(1) != nullptr, has2 = epi.src(2) != nullptr;
    auto fetch = [&](const int item) {
        if (tid == 0 && item < n_items) {
            const int b = item / per_member;
            if (!epi.member_active(b)) return;
            const int rest = item - b * per_member, tl = rest / tiles_r, tr = rest - tl * tiles_r;
            const int c1 = tr * (kTtTW / 8) - kTtHalo / 8, c2 = tl * kTtTL - 1;
            fence_proxy_async_smem();
            mbar_expect_tx(bar, kTtStageBytes * (1u + (has1 ? 1u : 0u) + (has2 ? 1u : 0u)));
            tma_load_4d(raw, &tm0, 0, c1, c2, b, bar);
            if (has1) tma_load_4d(raw + ELEMS, &tm1, 0, c1, c2, b, bar);
            if (has2) tma_load_4d(raw + 2 * ELEMS, &tm2, 0, c1, c2, b, bar);
        }
    };
    fetch(blockIdx.x);

    const int tx = tid % kTtTW, ty = tid / kTtTW;
    unsigned phase = 0;
    const double2 z2 = make_double2(0.0, 0.0);
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int b = item / per_member, rest = item - b * per_member, tl = rest / tiles_r, tr = rest - tl * tiles_r;
        double red[NR];
#pragma unroll
        for (int r = 0; r < NR; ++r) red[r] = 0.0;
        if (epi.member_active(b)) {
            epi.prepare(b);
            // per-column coefficients first: their latency overlaps the wait for the sources
            const int jc = tr * kTtTW + tx;
            const double vj = (jc < g.n_r) ? __ldg(g.vj + jc) : 0.0, cen = (jc < g.n_r) ? __ldg(g.cen + jc) : 0.0;
            mbar_wait(bar, phase);
            phase ^= 1u;
            const bool cut_tile = g.j0 != nullptr && tr * kTtTW - kTtHalo < g.j0_max;   // the tile touches held points
            for (int i = tid; i < ELEMS; i += 256) {
                double2 v = epi.combine(raw[i], has1 ? raw[ELEMS + i] : z2, has2 ? raw[2 * ELEMS + i] : z2);
                if (cut_tile) {      // centrifugal cut-off: held points read as zero (P H P)
                    const int rr = i / COLS, cc = i - rr * COLS;
                    if (held_pt(g, tl * kTtTL - 1 + rr, tr * kTtTW - kTtHalo + cc)) v = z2;
                }
                tile[i] = v;
            }
            __syncthreads();                               // tile complete, raw buffers consumed
            fetch(item + gridDim.x);
            const int j = tr * kTtTW + tx, l0 = tl * kTtTL;
            if (j < g.n_r) {
                const double afield = epi.efield(b), rinv = 1.0 / (g.dr * (double)(j + 1));
                const double er = afield * (g.dr * (double)(j + 1));
                const int r0 = ty * (kTtTL / 2);
                const double2 *col = tile + (r0 + 1) * COLS + kTtHalo + tx;
                double2 lo = col[-COLS], f = col[0];
#pragma unroll
                for (int rr = 0; rr < kTtTL / 2; ++rr) {
                    const int l = l0 + r0 + rr;
                    if (l >= g.n_l) break;
                    const double2 *c = col + rr * COLS;
                    const double2 up = c[COLS];
                    const double2 fm1 = c[-1], fp1 = c[1];
                    double2 fm2 = fm1, fp2 = fp1;
                    if (FD == 5) { fm2 = c[-2]; fp2 = c[2]; }
                    const double d = fma((double)(l * (l + 1)), cen, vj);
                    const double cm = (l > 0) ? __ldg(g.cl + l - 1) : 0.0;
                    const double cp = __ldg(g.cl + l);
                    double2 h = h_point<FD>(g, d, VG ? 0.0 : er, cm, cp, f, fm1, fp1, fm2, fp2, lo, up);
                    if (VG) vg_couple<FD>(g, c, COLS, l, rinv, cm, cp, afield, lo, up, h);
                    if (cut_tile && held_pt(g, l, j)) h = z2;
                    epi.point(b, l, j, ((size_t)b * g.n_l + l) * g.n_r + j, f, h, red);
                    lo = f; f = up;
                }
            }
        } else {
            fetch(item + gridDim.x);
        }
        grid_store_partial<256, NR>(red, rc, (size_t)item, red_s);    // (its barriers also fence the tile for the next item)
    }
    grid_finish<256, NR>(rc, gridDim.x, g.batch, epi, red_s, flag);
}

}  // namespace tdse
