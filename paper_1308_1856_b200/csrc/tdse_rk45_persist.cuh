// Adaptive Dormand-Prince 5(4) as ONE persistent kernel for grids that fit the shared memory of the machine (row a3 of
// SURVEY section 8; the stage loop of P:469-478 with the embedded error estimate of P:825 and the controller of reading
// R-C4).  The paper separates the stages into kernels because a kernel boundary was the only global synchronisation its
// devices offered; here the CTAs of a co-resident (cooperative) grid synchronise themselves:
//
//   * CTA c owns the radial columns [c Wc, (c+1) Wc) of EVERY row (member, l): the l +- 1 coupling never leaves the CTA;
//     psi, k_1..k_7 and two copies of the stage vector (read / being formed) of the owned points stay in shared memory for
//     the whole run.
//   * a stage needs the HW edge columns of the two neighbouring CTAs.  They travel as self-validating packets: every
//     8-byte word carries 4 bytes of data and the 4-byte sequence number of the exchange (an aligned 8-byte store is
//     single-copy atomic), so the receiver polls the data itself: one trip through L2 per stage, no fence, no separate
//     flag, no grid-wide barrier inside a step.  The owner of an edge point sends it the moment it is formed.
//   * the error norm needs every CTA: per-member partial sums travel the same way, and EVERY CTA adds all of them in the
//     same fixed order, so that all CTAs take the same accept / reject decision and the same next step without a second
//     exchange.  CTA 0 keeps the logs and writes the control block back at the end.
//
// The arithmetic per point (the order of the axpy sums, h_point / vg_couple) is that of the stage kernels
// (tile_kernel<EpiRK>): only the order of the reductions differs.  No host interaction between t0 and t_end.
#pragma once

#include <type_traits>

#include "tdse_device.cuh"

namespace tdse {

constexpr int kRkpThreads = 512;
constexpr int kRkpMaxPT = 4;            // owned points per thread (k_1..k_7 in shared memory)
constexpr int kRkpRegPT = 2;            // ... with psi and k_1..k_7 of the owned points in REGISTERS (the faster form)
constexpr int kRkpMaxB = 32;            // members
constexpr int kRkpMaxSmem = 224 * 1024; // dynamic shared memory of a CTA (the kernel has about 1 KB of static data besides)

struct RkpPlan { int ok, G, Wc, R, pitch, smem, kreg; size_t halo_bytes, part_bytes; };

inline int rkp_smem_bytes(int R, int Wc, int pitch, int B, int G, int kreg) {
    const int NW = kRkpThreads / 32;
    const size_t P = (size_t)R * Wc;
    return (int)(sizeof(double2) * (2 * (size_t)(R + 2) * pitch + (kreg ? 1 : 9) * P) +
                 sizeof(double) * (7 * B + 56 + 2 * (NW > B ? NW : B) + 2 * B + 2 * (size_t)G * B));
}

// columns per CTA so that at most n_sm CTAs cover n_r, every CTA (the last one too) owns at least HW columns, and the
// owned points fit the threads and the shared memory of one CTA
inline RkpPlan rkp_plan(const tdse_grid &g, int n_sm, int max_smem) {
    RkpPlan p{};
    const int HW = (g.fd_order == 3) ? 1 : 2;
    if (g.batch > kRkpMaxB || g.n_r < 2 * HW) return p;
    const long R = (long)g.batch * g.n_l;
    if (R > 4096) return p;
    int Wc = (g.n_r + n_sm - 1) / n_sm;
    if (Wc < 4) Wc = 4;
    for (;; ++Wc) {
        if (Wc > g.n_r) Wc = g.n_r;
        const int G = (g.n_r + Wc - 1) / Wc;
        const int last = g.n_r - (G - 1) * Wc;
        if (last >= HW || G == 1) {
            p.G = G; p.Wc = Wc;
            break;
        }
        if (Wc == g.n_r) return p;
    }
    p.R = (int)R;
    p.pitch = p.Wc + 2 * HW;
    if (R * p.Wc > (long)kRkpThreads * kRkpMaxPT) return p;
    p.kreg = R * p.Wc <= (long)kRkpThreads * kRkpRegPT;
    p.smem = rkp_smem_bytes(p.R, p.Wc, p.pitch, g.batch, p.G, p.kreg);
    if (p.smem > max_smem) return p;
    p.halo_bytes = (size_t)32 * 2 * p.G * 2 * p.R * HW;        // a complex value = 4 packets of 8 bytes
    p.part_bytes = (size_t)16 * 2 * p.G * g.batch * 2;         // a real value = 2 packets
    p.ok = 1;
    return p;
}

struct RkpArgs {
    GridDev g;
    double2 *psi;                 // the state, advanced in place
    Ctl *ctl;                     // read at the start, written back by CTA 0 at the end
    const tdse_pulse *pulse;
    const double *replay;
    double *dt_log, *err_log;
    unsigned long long *halo;     // [2][G][2 sides][R][HW][4] packets: edge columns of the stage vectors (zero before the launch)
    unsigned long long *part;     // [2][G][B][2][2] packets: error-norm partial sums (zero before the launch)
    int G, Wc, R, pitch;
    double a[7][7];               // a[s][j], j < s: stage vector g_{s+1} (the last row = the b row: psi_new)
    double d_err[7];              // b_j - bhat_j
    // Every explicit method runs here as an FSAL scheme: its last stage vector is psi_new, whose k is the k_1 of the next
    // step (Dormand-Prince is one by construction, n_stage = 7; classic RK4 becomes one with n_stage = 5, row 4 = b).
    int n_stage;                  // k vectors of a step, the closing one included (2..7)
    // FIXED-step mode (tdse_step_rk4): n_fixed steps of ctl->dt, every one accepted, no error estimate, no exchange of
    // sums; the field values of all stage times come from e_tab[step][n_stage][batch] (field_table_rk_kernel)
    int fixed;
    long long n_fixed;
    const double *e_tab;
};

// ---- self-validating packets: {32 bits of data, 32-bit sequence number} per aligned 8-byte word -------------------------
__device__ __forceinline__ void ll_send(unsigned long long *dst, double v, unsigned int seq) {
    const unsigned long long hi = (unsigned long long)seq << 32;
    const unsigned long long w0 = hi | (unsigned int)__double2loint(v), w1 = hi | (unsigned int)__double2hiint(v);
    asm volatile("st.volatile.global.v2.u64 [%0], {%1, %2};" ::"l"(dst), "l"(w0), "l"(w1) : "memory");
}
__device__ __forceinline__ void ll_peek(const unsigned long long *src, unsigned long long &w0, unsigned long long &w1) {
    asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(w0), "=l"(w1) : "l"(src) : "memory");
}
// the value of a packet pair that was peeked at earlier (polls again while the sequence number is not the expected one)
__device__ __forceinline__ double ll_finish(const unsigned long long *src, unsigned int seq, unsigned long long w0,
                                            unsigned long long w1) {
    while ((unsigned int)(w0 >> 32) != seq || (unsigned int)(w1 >> 32) != seq) ll_peek(src, w0, w1);
    return __hiloint2double((int)(unsigned int)w1, (int)(unsigned int)w0);
}
__device__ __forceinline__ double ll_recv(const unsigned long long *src, unsigned int seq) {
    unsigned long long w0, w1;
    do {
        asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(w0), "=l"(w1) : "l"(src) : "memory");
    } while ((unsigned int)(w0 >> 32) != seq || (unsigned int)(w1 >> 32) != seq);
    return __hiloint2double((int)(unsigned int)w1, (int)(unsigned int)w0);
}

template <int N> using RkpI = std::integral_constant<int, N>;

// KREG: at most kRkpRegPT points per thread; psi and k_1..k_7 of a thread's points stay in its registers, shared memory
// holds only the two copies of the stage vector (whose neighbours other threads read).
// FIXED: the fixed-step mode with any stage count (a separate instantiation: the adaptive Dormand-Prince run keeps its
// seven stages and its control flow as compile-time facts).
template <int FD, bool VG, bool KREG, bool FIXED>
__global__ void __launch_bounds__(kRkpThreads, 1) rk45_persist_kernel(const __grid_constant__ RkpArgs a) {
    constexpr int HW = (FD == 3) ? 1 : 2;
    constexpr int NT = kRkpThreads, NW = NT / 32, PT = KREG ? kRkpRegPT : kRkpMaxPT;
    extern __shared__ __align__(16) unsigned char rkp_smem[];
    const GridDev &g = a.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x, G = a.G, R = a.R, pitch = a.pitch, B = g.batch, L = g.n_l;
    const int c0 = cta * a.Wc, wc = min(a.Wc, g.n_r - c0), P = R * wc, Pcap = R * a.Wc, TS = (R + 2) * pitch;
    double2 *tile = reinterpret_cast<double2 *>(rkp_smem);          // [2][(R + 2)][pitch]: zero rows above and below
    double2 *psi_s = tile + 2 * (size_t)TS;                         // [P]   (slot p belongs to one thread)     } not with
    double2 *k_s = psi_s + (KREG ? 0 : Pcap);                       // [7][P]                                   } KREG
    double2 *ev = k_s + (KREG ? 0 : 7 * (size_t)Pcap);              // [P] (|Delta|^2, |psi_new|^2), row-major over the owned block
    double2 kr[KREG ? 7 : 1][PT], pr[PT];                           // KREG: k_1..k_7 and psi of this thread's points
    double *etab = reinterpret_cast<double *>(ev + Pcap);           // [7][B] field values of the stages
    double *coef = etab + 7 * B;                                    // [7][7] h a_{sj}, then [7] h (b_j - bhat_j)
    double *csum = coef + 56;                                       // [max(NW, B)][2] chunk sums
    double *msum = csum + 2 * (NW > B ? NW : B);                    // [B][2] member sums over all CTAs
    double *gath = msum + 2 * B;                                    // [G][B][2] partial sums of every CTA
    __shared__ struct {
        double t, h, t_end, rtol, dt_max;
        int done, last, after_reject, replay, stop;
        long long n_accept, n_reject, n_attempt, n_replay, max_log;
        int accept;
    } c;

    // ---- the owned points of this thread (edge columns first: they are formed and sent first) and their coefficients ---
    const int ec = min(wc, 2 * HW), nE = R * ec, wi = wc - ec, per = R * HW;
    int tix[PT], bb[PT], nix[PT], sl[PT], sr[PT];
    size_t gix[PT];
    double dd[PT], rj[PT], cm[PT], cp[PT];
    bool own[PT], held[PT], edge[PT];
#pragma unroll
    for (int i = 0; i < PT; ++i) {
        const int p = tid + i * NT;
        own[i] = p < P;
        edge[i] = p < nE;                   // its stencil reaches into a neighbouring CTA's columns
        int row = 0, col = 0;
        if (own[i]) {
            if (p < nE) { row = p / ec; const int e = p - row * ec; col = (e < HW) ? e : wc - (ec - e); }
            else { const int q = p - nE; row = q / wi; col = HW + (q - row * wi); }
        }
        const int b = row / L, l = row - b * L, j = c0 + col;
        bb[i] = b;
        tix[i] = (row + 1) * pitch + HW + col;
        nix[i] = row * wc + col;
        sl[i] = (own[i] && cta > 0 && col < HW) ? row * HW + col : -1;                       // my left edge -> CTA c - 1
        sr[i] = (own[i] && cta < G - 1 && col >= wc - HW) ? row * HW + col - (wc - HW) : -1;  // my right edge -> CTA c + 1
        gix[i] = ((size_t)b * L + l) * g.n_r + j;
        dd[i] = fma((double)(l * (l + 1)), __ldg(g.cen + j), __ldg(g.vj + j));
        rj[i] = g.dr * (double)(j + 1);
        cm[i] = (l > 0) ? __ldg(g.cl + l - 1) : 0.0;
        cp[i] = (l + 1 < L) ? __ldg(g.cl + l) : 0.0;       // (the row after a member's last one belongs to the next member)
        held[i] = held_pt(g, l, j);
    }
    for (int i = tid; i < 2 * TS; i += NT) tile[i] = make_double2(0.0, 0.0);
    if (tid == 0) {
        const Ctl &s = *a.ctl;
        c.t = s.t; c.h = s.h; c.t_end = s.t_end; c.rtol = s.rtol; c.dt_max = s.dt_max;
        c.done = s.done; c.last = s.last; c.after_reject = s.after_reject; c.replay = s.replay; c.stop = 0;
        c.n_accept = s.n_accept; c.n_reject = s.n_reject; c.n_attempt = s.n_attempt; c.n_replay = s.n_replay;
        c.max_log = s.max_log; c.accept = 0;
    }
#pragma unroll
    for (int i = 0; i < PT; ++i)
        if (own[i]) {
            double2 v = a.psi[gix[i]];
            if (held[i]) v = make_double2(0.0, 0.0);
            if constexpr (KREG) pr[i] = v; else psi_s[tid + i * NT] = v;
        }
    __syncthreads();

    unsigned int n_pub = 0;     // stage vectors published so far (the sequence number of the packets)
    int cur = 0;                // which copy of the tile holds the stage vector being read
    // Form g_{s+1} = psi + sum_{j < s} (h a_{sj}) k_j at the owned points into the OTHER copy of the tile, send the edge
    // points to the neighbours as they are formed, receive theirs into the halo columns, switch the copies.
    auto form = [&](auto S) {
        constexpr int s = decltype(S)::value;
        ++n_pub;
        const int par = (int)(n_pub & 1u);
        double2 *tn = tile + (cur ^ 1) * TS;
        unsigned long long *mine = a.halo + (size_t)(par * G + cta) * 2 * per * 4;
#pragma unroll
        for (int i = 0; i < PT; ++i) {
            if (!own[i]) continue;
            const int p = tid + i * NT;
            double2 acc;
            if constexpr (KREG) acc = pr[i]; else acc = psi_s[p];
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                if (j < s) {
                    const double aj = coef[s * 7 + j];
                    double2 kj;
                    if constexpr (KREG) kj = kr[KREG ? j : 0][i]; else kj = k_s[(size_t)j * Pcap + p];
                    if (aj != 0.0) acc = caxpy_r(aj, kj, acc);
                }
            }
            tn[tix[i]] = acc;
            if (sl[i] >= 0) { ll_send(mine + (size_t)sl[i] * 4, acc.x, n_pub); ll_send(mine + (size_t)sl[i] * 4 + 2, acc.y, n_pub); }
            if (sr[i] >= 0) { ll_send(mine + (size_t)(per + sr[i]) * 4, acc.x, n_pub); ll_send(mine + (size_t)(per + sr[i]) * 4 + 2, acc.y, n_pub); }
        }
    };
    // The neighbours' edge columns -> the halo columns of the copy being formed.  The first packets of a thread are
    // requested BEFORE the interior points are worked on and looked at afterwards: the trip through L2 hides behind them.
    unsigned long long hw0 = 0, hw1 = 0, hw2 = 0, hw3 = 0;
    auto halo_src = [&](const int idx, int &dst) -> const unsigned long long * {
        const int par = (int)(n_pub & 1u);
        const int side = idx / per, rem = idx - side * per, row = rem / HW, hh = rem - row * HW;
        const int nb = side == 0 ? cta - 1 : cta + 1;
        if (nb < 0 || nb >= G) return nullptr;                 // the wall: the halo stays zero
        dst = (row + 1) * pitch + (side == 0 ? hh : HW + wc + hh);
        // the left neighbour's RIGHT edge / the right neighbour's LEFT edge
        return a.halo + ((size_t)(par * G + nb) * 2 * per + (size_t)(1 - side) * per + rem) * 4;
    };
    auto halo_request = [&]() {
        int dst;
        if (tid < 2 * per) {
            const unsigned long long *src = halo_src(tid, dst);
            if (src) { ll_peek(src, hw0, hw1); ll_peek(src + 2, hw2, hw3); }
        }
    };
    auto halo_receive = [&]() {
        double2 *tn = tile + (cur ^ 1) * TS;
        for (int idx = tid; idx < 2 * per; idx += NT) {
            int dst;
            const unsigned long long *src = halo_src(idx, dst);
            if (!src) continue;
            double2 v;
            if (idx == tid) { v.x = ll_finish(src, n_pub, hw0, hw1); v.y = ll_finish(src + 2, n_pub, hw2, hw3); }
            else { v.x = ll_recv(src, n_pub); v.y = ll_recv(src + 2, n_pub); }
            tn[dst] = v;
        }
    };
    // k_s = -i H(t + c_s h) g_s at the owned points, g_s = the vector in the current copy of the tile
    auto apply = [&](auto S, const double2 *tc, const bool edge_points) {
        constexpr int s = decltype(S)::value;
#pragma unroll
        for (int i = 0; i < PT; ++i) {
            if (!own[i] || edge[i] != edge_points) continue;
            const double2 *cpt = tc + tix[i];
            const double2 f = cpt[0], fm1 = cpt[-1], fp1 = cpt[1];
            double2 fm2 = fm1, fp2 = fp1;
            if (FD == 5) { fm2 = cpt[-2]; fp2 = cpt[2]; }
            const double2 lo = cpt[-pitch], up = cpt[pitch];
            const double afield = etab[s * B + bb[i]];
            double2 h = h_point<FD>(g, dd[i], VG ? 0.0 : afield * rj[i], cm[i], cp[i], f, fm1, fp1, fm2, fp2, lo, up);
            if (VG) {
                const int l = (tix[i] / pitch - 1) - bb[i] * L;
                vg_couple<FD>(g, cpt, pitch, l, 1.0 / rj[i], cm[i], cp[i], afield, lo, up, h);
            }
            if (held[i]) h = make_double2(0.0, 0.0);
            if constexpr (KREG) kr[KREG ? s : 0][i] = make_double2(h.y, -h.x);
            else k_s[(size_t)s * Pcap + tid + i * NT] = make_double2(h.y, -h.x);
        }
    };
    // one stage: form g_{s+1} (edge points first, sent at once), then k_{s+1} = -i H g_{s+1}: interior points while the
    // neighbours' packets travel, edge points once they are in
    auto stage = [&](auto S) {
        form(S);
        halo_request();
        __syncthreads();
        const double2 *tn = tile + (cur ^ 1) * TS;
        apply(S, tn, false);
        halo_receive();
        __syncthreads();
        apply(S, tn, true);
        cur ^= 1;
    };

    bool have_k1 = false;
    constexpr bool fixed = FIXED;
    const int ns = FIXED ? a.n_stage : 7;
    long long step = 0;
    if (fixed) {
        const double hh = a.ctl->dt;
        if (tid < 49) coef[tid] = hh * a.a[tid / 7][tid % 7];
        if (tid < ns * B) etab[tid] = __ldg(a.e_tab + tid);
        __syncthreads();
    }
    while (fixed ? step < a.n_fixed : (!c.done && !c.stop)) {
        double e_next = 0.0;    // fixed: the field value this thread carries over to the next step
        const bool carries = fixed && tid < ns * B && step + 1 < a.n_fixed;
        if (carries) e_next = __ldg(a.e_tab + (size_t)(step + 1) * ns * B + tid);
        if (!fixed) {
        // ---- start of an attempted step: clip the step to t_end (or take the replayed one), field values of the stages
        if (tid == 0) {
            double h = c.h;
            if (c.replay) { h = a.replay[c.n_attempt]; c.last = 0; }
            else if (__dadd_rn(c.t, h) >= c.t_end) { h = c.t_end - c.t; c.last = 1; }
            else c.last = 0;
            c.h = h;
        }
        __syncthreads();
        const double hh = c.h, t = c.t;
        for (int i = tid; i < 7 * B; i += NT) {
            const int st = i / B, b = i - st * B;
            const double cst = (st == 0) ? 0.0 : (st == 1) ? 1.0 / 5 : (st == 2) ? 3.0 / 10 : (st == 3) ? 4.0 / 5 : (st == 4) ? 8.0 / 9 : 1.0;
            etab[i] = pulse_field(a.pulse[b], __dadd_rn(t, __dmul_rn(cst, hh)), g.gauge);
        }
        if (tid < 49) coef[tid] = hh * a.a[tid / 7][tid % 7];
        else if (tid < 56) coef[tid] = hh * a.d_err[tid - 49];
        __syncthreads();
        }
        if (!have_k1) {         // the first attempted step: k_1 = -i H(t) psi (afterwards FSAL supplies it)
            stage(RkpI<0>{});
            have_k1 = true;
        }
        // ---- stages 2..7: g_{s+1} = psi + h sum_j a_{s+1,j} k_j, then k_{s+1}; the last one is psi_new and k_7 -------------
        stage(RkpI<1>{});
        if (ns > 2) stage(RkpI<2>{});
        if (ns > 3) stage(RkpI<3>{});
        if (ns > 4) stage(RkpI<4>{});
        if (ns > 5) stage(RkpI<5>{});
        if (ns > 6) stage(RkpI<6>{});
        if (!fixed) {
        // ---- embedded error estimate: Delta = h sum_j (b_j - bhat_j) k_j against psi_new ---------------------------
        {
            const double2 *tc = tile + cur * TS;
#pragma unroll
            for (int i = 0; i < PT; ++i) {
                if (!own[i]) continue;
                const int p = tid + i * NT;
                double2 d = make_double2(0.0, 0.0);
#pragma unroll
                for (int j = 0; j < 7; ++j) {
                    const double dj = coef[49 + j];
                    double2 kj;
                    if constexpr (KREG) kj = kr[KREG ? j : 0][i]; else kj = k_s[(size_t)j * Pcap + p];
                    if (dj != 0.0) d = caxpy_r(dj, kj, d);
                }
                const double2 f = tc[tix[i]];
                ev[nix[i]] = make_double2(d.x * d.x + d.y * d.y, f.x * f.x + f.y * f.y);
            }
        }
        __syncthreads();
        // per member: its owned points are contiguous in ev; CH chunks per member, one warp per chunk, fixed order
        const int CH = (NW >= B) ? NW / B : 1, Pm = L * wc;
        for (int q = warp; q < B * CH; q += NW) {
            const int b = q / CH, ic = q - b * CH;
            const int lo = b * Pm + (int)((long long)Pm * ic / CH), hi = b * Pm + (int)((long long)Pm * (ic + 1) / CH);
            double s0 = 0.0, s1 = 0.0;
            for (int p = lo + lane; p < hi; p += 32) { const double2 v = ev[p]; s0 += v.x; s1 += v.y; }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, off);
                s1 += __shfl_xor_sync(0xffffffffu, s1, off);
            }
            if (lane == 0) { csum[2 * q] = s0; csum[2 * q + 1] = s1; }
        }
        __syncthreads();
        // every CTA publishes its member sums and gathers those of all CTAs
        const unsigned int n_att = (unsigned int)(c.n_attempt + 1);
        const int par2 = (int)(n_att & 1u);
        if (tid < B) {
            double s0 = 0.0, s1 = 0.0;
            for (int ic = 0; ic < CH; ++ic) { s0 += csum[2 * (tid * CH + ic)]; s1 += csum[2 * (tid * CH + ic) + 1]; }
            unsigned long long *dst = a.part + ((size_t)(par2 * G + cta) * B + tid) * 4;
            ll_send(dst, s0, n_att);
            ll_send(dst + 2, s1, n_att);
        }
        for (int i = tid; i < G * B * 2; i += NT) gath[i] = ll_recv(a.part + ((size_t)par2 * G * B * 2 + i) * 2, n_att);
        __syncthreads();
        for (int b = warp; b < B; b += NW) {
            double s0 = 0.0, s1 = 0.0;
            for (int i = lane; i < G; i += 32) { s0 += gath[(i * B + b) * 2]; s1 += gath[(i * B + b) * 2 + 1]; }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, off);
                s1 += __shfl_xor_sync(0xffffffffu, s1, off);
            }
            if (lane == 0) { msum[2 * b] = s0; msum[2 * b + 1] = s1; }
        }
        __syncthreads();
        // ---- controller (reading R-C4), identical in every CTA -------------------------------------------------------------
        if (tid == 0) {
            double emax = 0.0;
            for (int b = 0; b < B; ++b) {
                const double e = sqrt(msum[2 * b]) / sqrt(msum[2 * b + 1]);
                if (!(e <= emax)) emax = e;
            }
            const double err = emax / c.rtol;
            const long long slot = c.n_accept;
            const double h = c.h;
            const bool accept = c.replay || (err <= 1.0);
            if (accept) {
                if (cta == 0 && slot < c.max_log) { a.dt_log[slot] = h; a.err_log[slot] = err; }
                c.n_accept = slot + 1;
                c.t = c.last ? c.t_end : __dadd_rn(c.t, h);
            } else {
                c.n_reject += 1;
            }
            c.n_attempt += 1;
            c.accept = accept ? 1 : 0;
            if (c.replay) {
                if (c.n_attempt >= c.n_replay) c.done = 1;
            } else {
                double fac = 0.9 * pow(err, -0.2);
                if (!(fac >= 0.2)) fac = 0.2;
                if (fac > 5.0) fac = 5.0;
                if (accept) {
                    if (c.after_reject && fac > 1.0) fac = 1.0;
                    c.after_reject = 0;
                    if (!(c.t < c.t_end)) c.done = 1;
                } else {
                    if (fac > 1.0) fac = 1.0;
                    c.after_reject = 1;
                }
                double hn = __dmul_rn(h, fac);
                if (c.dt_max > 0.0 && hn > c.dt_max) hn = c.dt_max;
                c.h = hn;
                if (!c.done && !(hn > 0.0)) c.stop = 1;     // no positive step left: the host reports TDSE_ERR_NONFINITE
            }
        }
        }
        __syncthreads();        // (fixed: every thread is done with the field values of this step)
        if (fixed || c.accept) {    // psi <- psi_new (the vector in the tile), k_1 <- the closing k (FSAL: same time t_{n+1})
            const double2 *tc = tile + cur * TS;
#pragma unroll
            for (int i = 0; i < PT; ++i) {
                if (!own[i]) continue;
                const int p = tid + i * NT;
                if constexpr (KREG) {
                    pr[i] = tc[tix[i]];
                    double2 kl = kr[KREG ? 6 : 0][i];
                    if (ns == 6) kl = kr[KREG ? 5 : 0][i];
                    if (ns == 5) kl = kr[KREG ? 4 : 0][i];
                    if (ns == 4) kl = kr[KREG ? 3 : 0][i];
                    if (ns == 3) kl = kr[KREG ? 2 : 0][i];
                    if (ns == 2) kl = kr[KREG ? 1 : 0][i];
                    kr[0][i] = kl;
                } else {
                    psi_s[p] = tc[tix[i]];
                    k_s[p] = k_s[(size_t)(ns - 1) * Pcap + p];
                }
            }
        }
        if (carries) etab[tid] = e_next;
        ++step;
        __syncthreads();
    }

#pragma unroll
    for (int i = 0; i < PT; ++i)
        if (own[i]) {
            if constexpr (KREG) a.psi[gix[i]] = pr[i]; else a.psi[gix[i]] = psi_s[tid + i * NT];
        }
    if (cta == 0 && tid == 0 && !fixed) {
        Ctl &s = *a.ctl;
        s.t = c.t; s.h = c.h; s.done = c.done; s.last = c.last; s.after_reject = c.after_reject;
        s.n_accept = c.n_accept; s.n_reject = c.n_reject; s.n_attempt = c.n_attempt;
    }
}

}  // namespace tdse
