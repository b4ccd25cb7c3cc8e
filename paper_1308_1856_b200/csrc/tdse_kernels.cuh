// tdse_kernels.cuh -- the sm_100a kernels of the one-pass path: H.psi on shared-memory (l, r) tiles with the
// propagator arithmetic fused into the epilogue, element-wise/reduction kernels, observables, the one-warp
// tridiagonal exponential and the control kernels.  Product path; shares nothing with oracle/.
#pragma once
#include "tdse_device.cuh"

namespace tdse {

// ------------------------------------------------------------------------------------------------------
// Tile geometry: TL partial waves x TW radial points of complex128 per CTA, staged in shared memory with
// a radial halo of HW points on both sides and the l-1 / l+1 rows (NS: "(l, r) tiles ... staged with their
// radial halo and l+-1 neighbours").  256 threads; each thread owns one column and marches RPT rows, keeping
// the l-1, l, l+1 values in registers.
// ------------------------------------------------------------------------------------------------------
template <int FD>
struct Tile {
    static constexpr int HW = (FD == 3) ? 1 : 2;
#ifndef TDSE_TILE_TL
#define TDSE_TILE_TL 8
#endif
    static constexpr int TW = 128, TL = TDSE_TILE_TL, NT = 256;
    static constexpr int RPT = TL / (NT / TW);          // rows per thread
    static constexpr int PITCH = TW + 2 * HW;           // double2 elements per shared row
    static constexpr int ROWS = TL + 2;
    static constexpr int ELEMS = ROWS * PITCH;
};

// One pass: out/epilogue <- H(E_b) in, for every member b.  grid = (ceil(n_r/TW), ceil(n_l/TL), batch).
// Epi supplies: NRED, SCALED; begin(); skip_all(); member_active(b); input(); in_scale(b); efield(b);
// point(b,l,j,idx,f,h,red); finish_member(b,s); finish_all().
// VG: velocity gauge (the l+-1 rows enter through d/dr -+ l/r instead of r; a template flag so that the
// length-gauge instantiations keep their register budget).
template <int FD, class Epi, bool VG = false>
__global__ void __launch_bounds__(256, Epi::MINB) tile_kernel(GridDev g, Epi epi_in, RedCtx rc) {
    using T = Tile<FD>;
    __shared__ double2 tile[T::ELEMS];
    __shared__ double red_s[(Epi::NRED > 0 ? Epi::NRED : 1) * (T::NT / 32)];
    __shared__ int last_flag;
    Epi epi = epi_in;
    epi.begin();
    if (epi.skip_all()) return;

    const int tid = threadIdx.x;
    const int b = blockIdx.z, l0 = blockIdx.y * T::TL, j0 = blockIdx.x * T::TW;
    double red[Epi::NRED > 0 ? Epi::NRED : 1];
#pragma unroll
    for (int r = 0; r < (Epi::NRED > 0 ? Epi::NRED : 1); ++r) red[r] = 0.0;

    if (epi.member_active(b)) {
        epi.prepare(b);
        const double2 *base = epi.input() + (size_t)b * g.n_l * g.n_r;
        const double sc = Epi::SCALED ? epi.in_scale(b) : 1.0;
        const bool cut_tile = g.j0 != nullptr && j0 - T::HW < g.j0_max;         // the tile touches held points
        // optional second source: the tile holds in + c2in * in2 (a stage vector formed while loading)
        const double2 *base2 = Epi::TWO_IN ? epi.input2() + (size_t)b * g.n_l * g.n_r : nullptr;
        const double c2in = Epi::TWO_IN ? epi.in2_coef() : 0.0;
        // stage the tile (zero outside the index box: Dirichlet walls, f_{-1} = f_L = 0)
#pragma unroll
        for (int it = 0; it < (T::ELEMS + T::NT - 1) / T::NT; ++it) {
            const int i = tid + it * T::NT;
            if (i < T::ELEMS) {
                const int rr = i / T::PITCH, cc = i - rr * T::PITCH;
                const int l = l0 - 1 + rr, j = j0 - T::HW + cc;
                double2 v = make_double2(0.0, 0.0);
                if (l >= 0 && l < g.n_l && j >= 0 && j < g.n_r) {
                    if (Epi::CUSTOM_LOAD) {
                        v = epi.load(((size_t)b * g.n_l + l) * g.n_r + j);      // a vector formed from several arrays
                    } else {
                        v = __ldg(base + (size_t)l * g.n_r + j);
                        if (Epi::TWO_IN) v = caxpy_r(c2in, __ldg(base2 + (size_t)l * g.n_r + j), v);
                    }
                }
                if (Epi::SCALED) { v.x *= sc; v.y *= sc; }
                if (cut_tile && held_pt(g, l, j)) v = make_double2(0.0, 0.0);      // P H P: held points read as zero
                tile[i] = v;
            }
        }
        __syncthreads();

        const int tx = tid % T::TW, ty = tid / T::TW;
        const int j = j0 + tx;
        if (j < g.n_r) {
            const double vj = __ldg(g.vj + j), cen = __ldg(g.cen + j);
            const double afield = epi.efield(b), rinv = 1.0 / (g.dr * (double)(j + 1));
            const double er = afield * (g.dr * (double)(j + 1));
            const int r0 = ty * T::RPT;
            const double2 *col = tile + (r0 + 1) * T::PITCH + T::HW + tx;
            double2 lo = col[-T::PITCH], f = col[0];
#pragma unroll
            for (int rr = 0; rr < T::RPT; ++rr) {
                const int l = l0 + r0 + rr;
                if (l >= g.n_l) break;
                const double2 *c = col + rr * T::PITCH;
                const double2 up = c[T::PITCH];
                const double2 fm1 = c[-1], fp1 = c[1];
                double2 fm2 = fm1, fp2 = fp1;
                if (FD == 5) { fm2 = c[-2]; fp2 = c[2]; }
                const double d = fma((double)(l * (l + 1)), cen, vj);
                const double cm = (l > 0) ? __ldg(g.cl + l - 1) : 0.0;
                const double cp = __ldg(g.cl + l);
                double2 h = h_point<FD>(g, d, VG ? 0.0 : er, cm, cp, f, fm1, fp1, fm2, fp2, lo, up);
                if (VG) vg_couple<FD>(g, c, T::PITCH, l, rinv, cm, cp, afield, lo, up, h);
                if (cut_tile && held_pt(g, l, j)) h = make_double2(0.0, 0.0);    // ... and come out as zero
                const size_t idx = ((size_t)b * g.n_l + l) * g.n_r + j;
                epi.point(b, l, j, idx, f, h, red);
                lo = f; f = up;
            }
        }
    }
    if (Epi::NRED > 0) {
        const int cta = (b * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
        grid_reduce_finish<T::NT, (Epi::NRED > 0 ? Epi::NRED : 1)>(red, rc, cta, gridDim.x * gridDim.y * gridDim.z,
                                                                  g.batch, epi, red_s, &last_flag);
    }
}

// Defaults shared by the epilogues.
struct EpiBase {
    static constexpr int NRED = 0;
    static constexpr bool SCALED = false;
    static constexpr bool TWO_IN = false;
    static constexpr bool CUSTOM_LOAD = false;
    static constexpr int MINB = 3;              // CTAs per SM the register budget is set for
    __device__ __forceinline__ void prepare(int) {}
    __device__ __forceinline__ double2 load(size_t) const { return make_double2(0.0, 0.0); }

    __device__ __forceinline__ const double2 *input2() const { return nullptr; }
    __device__ __forceinline__ double in2_coef() const { return 0.0; }
    __device__ __forceinline__ void begin() {}
    __device__ __forceinline__ bool skip_all() const { return false; }
    __device__ __forceinline__ bool member_active(int) const { return true; }
    __device__ __forceinline__ double in_scale(int) const { return 1.0; }
    __device__ __forceinline__ void finish_member(int, const double *) {}
    __device__ __forceinline__ void finish_all() {}
};

// out = H in  (tdse_apply_H)
struct EpiApply : EpiBase {
    const double2 *in; const double *ef; double2 *out;
    __device__ __forceinline__ const double2 *input() const { return in; }
    __device__ __forceinline__ double efield(int b) const { return __ldg(ef + b); }
    __device__ __forceinline__ void point(int, int, int, size_t idx, double2, double2 h, double *) { out[idx] = h; }
};

// One Taylor order (Eq. 37, "only one kernel"): term_k = (-i dt/k) H term_{k-1}; acc += term_k.
struct EpiTaylor : EpiBase {
    const double2 *in; const double *ef; const double *dtp; int k, first, write_term;
    int imag;               // 1: imaginary time (-i -> 1), term_k = (-dt/k) H term_{k-1}
    double2 *term_out; const double2 *acc_in; double2 *acc_out;
    double s;
    __device__ __forceinline__ void begin() { s = *dtp / (double)k; }
    __device__ __forceinline__ const double2 *input() const { return in; }
    __device__ __forceinline__ double efield(int b) const { return __ldg(ef + b); }
    __device__ __forceinline__ void point(int, int, int, size_t idx, double2 f, double2 h, double *) {
        const double2 t = imag ? make_double2(-s * h.x, -s * h.y)
                               : make_double2(s * h.y, -s * h.x);      // (-i s)(x + i y) = s y - i s x
        if (write_term) term_out[idx] = t;
        const double2 a = first ? f : acc_in[idx];
        acc_out[idx] = cadd(a, t);
    }
};

// One explicit Runge-Kutta stage (Eq. 38, stage loop P:469-478) with the next stage vector formed in the
// epilogue: k_i = -i H(t_n + c_i h) g_i;  g_{i+1} = psi + sum_{j<=i} (h a_{i+1,j}) k_j  (or psi_new with the b row).
// Buffers are addressed through roles so that the adaptive driver can swap psi/psi_new and k1/k7 on the device.
template <bool EMBED, bool TWO = false>
struct EpiRK : EpiBase {
    static constexpr int NRED = EMBED ? 2 : 0;
    static constexpr bool TWO_IN = TWO;     // tile = bufs[in_role] + (h * in2_a) * bufs[in2_role]
    int in2_role; double in2_a;
    Ctl *ctl; double2 *const *bufs; const double *ef; const double *hptr;
    int stage;              // i (0-based)
    int in_role;            // role of the tile source
    int k_role[7];          // roles of k_0..k_6
    int store_k;            // write k_i
    int out_role;           // role receiving g_{i+1} / psi_new, -1: none
    int psi_role;
    double a_next[7];       // a_{i+1,j} (or b_j), j = 0..i; 0 entries are skipped like in the paper's loop
    double d_err[7];        // b_j - bhat_j  (embedded pair difference)
    int check_done;
    double *dt_log, *err_log;
    int passive;            // EMBED: no controller, only the passive error sum of P:827-833 (fixed-step methods)
    double *sigma_acc; double inv_m;     // sigma_acc[b] += sqrt(|Delta_b|^2 / M), inv_m = 1/M
    // resolved at begin()
    const double2 *in_p; const double2 *in2_p; double2 *out_p; const double2 *psi_p; double2 *k_p[7]; double hh; double emax;

    __device__ __forceinline__ void begin() {
        in_p = bufs[ctl->perm[in_role]];
        in2_p = TWO ? bufs[ctl->perm[in2_role]] : nullptr;
        out_p = out_role >= 0 ? bufs[ctl->perm[out_role]] : nullptr;
        psi_p = bufs[ctl->perm[psi_role]];
#pragma unroll
        for (int j = 0; j < 7; ++j) k_p[j] = (k_role[j] >= 0) ? bufs[ctl->perm[k_role[j]]] : nullptr;
        hh = *hptr;
        emax = 0.0;
    }
    __device__ __forceinline__ bool skip_all() const { return check_done && ctl->done; }
    __device__ __forceinline__ const double2 *input() const { return in_p; }
    __device__ __forceinline__ const double2 *input2() const { return in2_p; }
    __device__ __forceinline__ double in2_coef() const { return hh * in2_a; }
    __device__ __forceinline__ double efield(int b) const { return __ldg(ef + b); }
    __device__ __forceinline__ void point(int, int, int, size_t idx, double2 f, double2 h, double *red) {
        const double2 k = make_double2(h.y, -h.x);              // -i H g
        if (store_k) k_p[stage][idx] = k;
        if (out_role >= 0) {
            double2 acc = (stage == 0) ? f : psi_p[idx];
#pragma unroll
            for (int j = 0; j < 7; ++j) {
                if (j < stage && a_next[j] != 0.0) acc = caxpy_r(hh * a_next[j], k_p[j][idx], acc);
            }
            if (a_next[stage] != 0.0) acc = caxpy_r(hh * a_next[stage], k, acc);
            out_p[idx] = acc;
        }
        if (EMBED) {
            double2 d = make_double2(0.0, 0.0);
#pragma unroll
            for (int j = 0; j < 7; ++j) {
                if (j < stage && d_err[j] != 0.0) d = caxpy_r(hh * d_err[j], k_p[j][idx], d);
            }
            if (d_err[stage] != 0.0) d = caxpy_r(hh * d_err[stage], k, d);
            red[0] += d.x * d.x + d.y * d.y;
            red[1] += f.x * f.x + f.y * f.y;                    // the tile source of the last stage is psi_new
        }
    }
    // controller (R-C4): runs once per attempted step in the last CTA
    __device__ __forceinline__ void finish_member(int b, const double *s) {
        if (EMBED && passive) { sigma_acc[b] += sqrt(s[0] * inv_m); return; }
        if (EMBED) { const double e = sqrt(s[0]) / sqrt(s[1]); if (!(e <= emax)) emax = e; }
    }
    __device__ __forceinline__ void finish_all() {
        if (!EMBED || passive) return;
        Ctl &c = *ctl;
        const double err = emax / c.rtol;
        const long long slot = c.n_accept;
        const double h = c.h;
        bool accept = c.replay || (err <= 1.0);
        if (accept) {
            if (slot < c.max_log) { dt_log[slot] = h; err_log[slot] = err; }
            c.n_accept = slot + 1;
            // psi <- psi_new (held by the last stage's tile source), k1 <- k7 (FSAL: same time t_{n+1})
            int tmp = c.perm[psi_role]; c.perm[psi_role] = c.perm[in_role]; c.perm[in_role] = tmp;
            tmp = c.perm[k_role[0]]; c.perm[k_role[0]] = c.perm[k_role[6]]; c.perm[k_role[6]] = tmp;
            c.t = c.last ? c.t_end : __dadd_rn(c.t, h);
        } else {
            c.n_reject += 1;
        }
        c.n_attempt += 1;
        if (c.replay) {
            if (c.n_attempt >= c.n_replay) c.done = 1;
            return;
        }
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
    }
};

// One Lanczos vector per PASS (App. B in reading R-G16; the paper uses 3 kernels per vector).
// Stored vectors are v_0 = psi and v_p = w_{p-1} (the orthogonalised, UNnormalised residual, norm beta_{p-1});
// q_p = s_p v_p with s_0 = 1/||psi||, s_p = 1/beta_{p-1}.  Pass p forms, while loading its tile,
//     v_p = s_{p-1} g_{p-1} - alpha_{p-1} q_{p-1} - beta_{p-2} q_{p-2}          (g_{p-1} = H v_{p-1}, so s g = H q)
// applies H (g_p = H v_p, linear, so the normalisation can wait), writes v_p and g_p, and reduces BOTH
// <v_p|g_p> and ||v_p||^2 in the same pass; the last CTA turns them into beta_{p-1} = ||v_p||, s_p, the
// breakdown flag and alpha_p = s_p^2 Re<v_p|g_p> = Re<q_p|H q_p>.  80 B/point/vector in one kernel instead of
// 112 B in two; the norm of psi is pass 0's second reduction.
struct EpiLanczosF : EpiBase {
    static constexpr int NRED = 2;
    static constexpr bool CUSTOM_LOAD = true;
#ifndef TDSE_LZ_MINB
#define TDSE_LZ_MINB 5
#endif
    static constexpr int MINB = TDSE_LZ_MINB;   // latency-bound on HBM: measured 2295 / 1923 / 1776 us per CFG4 step at 3 / 4 / 5
    const double2 *psi, *g_in, *v1, *v2;       // psi (p = 0); g_{p-1}, v_{p-1}, v_{p-2}
    double2 *v_out, *g_out;
    const double *ef; double *alpha, *beta, *sc, *nrm; int *m_used; int p, K; double tol;
    double s1, a1, b2s2, sc_prev;               // per-member scalars of the load (set by prepare)
    __device__ __forceinline__ bool member_active(int b) const { return p == 0 || m_used[b] > p; }
    __device__ __forceinline__ const double2 *input() const { return psi; }
    __device__ __forceinline__ double efield(int b) const { return __ldg(ef + b); }
    __device__ __forceinline__ void prepare(int b) {
        s1 = a1 = b2s2 = 0.0;
        if (p >= 1) { s1 = sc[b * K + p - 1]; a1 = alpha[b * K + p - 1]; }
        sc_prev = 0.0;
        if (p >= 2) { b2s2 = beta[b * K + p - 2]; sc_prev = sc[b * K + p - 2]; }
    }
    __device__ __forceinline__ const double2 *src(int i) const {
        return (i == 0) ? (p == 0 ? psi : g_in) : (i == 1 ? v1 : v2);
    }
    // raw values of (g_{p-1} | psi), v_{p-1}, v_{p-2} at one point -> v_p
    __device__ __forceinline__ double2 combine(double2 g, double2 x1, double2 x2) const {
        if (p == 0) return g;
        double2 w = make_double2(g.x * s1, g.y * s1);                            // H q_{p-1}
        w = caxpy_r(-a1, make_double2(x1.x * s1, x1.y * s1), w);                 // - alpha_{p-1} q_{p-1}
        if (p >= 2) w = caxpy_r(-b2s2, make_double2(x2.x * sc_prev, x2.y * sc_prev), w);   // - beta_{p-2} q_{p-2}
        return w;
    }
    __device__ __forceinline__ double2 load(size_t idx) const {
        const double2 z = make_double2(0.0, 0.0);
        return combine(__ldg((p == 0 ? psi : g_in) + idx), p >= 1 ? __ldg(v1 + idx) : z, p >= 2 ? __ldg(v2 + idx) : z);
    }
    __device__ __forceinline__ void point(int, int, int, size_t idx, double2 f, double2 h, double *red) {
        v_out[idx] = f;
        if (g_out) g_out[idx] = h;
        red[0] += f.x * h.x + f.y * h.y;
        red[1] += f.x * f.x + f.y * f.y;
    }
    __device__ __forceinline__ void finish_member(int b, const double *s) {
        if (p > 0 && m_used[b] <= p) return;
        const double n = sqrt(s[1]);
        const double sp = 1.0 / n;
        if (p == 0) { nrm[b] = n; m_used[b] = K; }
        else {
            beta[b * K + p - 1] = n;
            if (n < tol) { m_used[b] = p; return; }   // breakdown (R-G17): vectors 0 .. p-1 span the space
        }
        sc[b * K + p] = sp;
        alpha[b * K + p] = (s[0] * sp) * sp;
    }
};


// ------------------------------------------------------------------------------------------------------
// Element-wise kernels with optional fused reduction.  grid = (chunks, 1, batch); a CTA handles EW_CHUNK
// consecutive points of one member.
// ------------------------------------------------------------------------------------------------------
constexpr int EW_NT = 256, EW_PER = 8, EW_CHUNK = EW_NT * EW_PER;

template <class Op>
__global__ void __launch_bounds__(EW_NT) ew_kernel(long long n_per_member, int n_members, Op op_in, RedCtx rc) {
    __shared__ double red_s[(Op::NRED > 0 ? Op::NRED : 1) * (EW_NT / 32)];
    __shared__ int last_flag;
    Op op = op_in;
    op.begin();
    const int b = blockIdx.z;
    double red[Op::NRED > 0 ? Op::NRED : 1];
#pragma unroll
    for (int r = 0; r < (Op::NRED > 0 ? Op::NRED : 1); ++r) red[r] = 0.0;
    if (op.member_active(b)) {
        const long long base = (long long)blockIdx.x * EW_CHUNK;
#pragma unroll
        for (int u = 0; u < EW_PER; ++u) {
            const long long i = base + threadIdx.x + u * EW_NT;
            if (i < n_per_member) op.point(b, (size_t)b * n_per_member + i, red);
        }
    }
    if (Op::NRED > 0) {
        const int cta = b * gridDim.x + blockIdx.x;
        grid_reduce_finish<EW_NT, (Op::NRED > 0 ? Op::NRED : 1)>(red, rc, cta, gridDim.x * gridDim.z, n_members, op,
                                                              red_s, &last_flag);
    }
}

struct OpBase {
    static constexpr int NRED = 0;
    __device__ __forceinline__ void begin() {}
    __device__ __forceinline__ bool member_active(int) const { return true; }
    __device__ __forceinline__ void finish_member(int, const double *) {}
    __device__ __forceinline__ void finish_all() {}
};

// F(t+dt) = ||F|| sum_{p<m} c_p q_p  (Taylor2)
struct OpCombine : OpBase {
    double2 *psi; const double2 *q; size_t q_stride; const double2 *coef; const double *nrm, *sc; const int *m_used; int K;
    __device__ __forceinline__ void point(int b, size_t idx, double *) {
        const int m = m_used[b];
        const double n = nrm[b];
        double2 acc = make_double2(0.0, 0.0);
        for (int p0 = 0; p0 < m; p0 += 8) {                 // 8 basis vectors' loads in flight per point
            double2 x[8];
#pragma unroll
            for (int i = 0; i < 8; ++i)
                x[i] = (p0 + i < m) ? __ldcs(q + (size_t)(p0 + i) * q_stride + idx) : make_double2(0.0, 0.0);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (p0 + i >= m) break;
                const double2 c = coef[b * K + p0 + i];
                const double sp = sc[b * K + p0 + i];               // q_p = s_p v_p
                const double ar = n * c.x, ai = n * c.y;
                const double vx = x[i].x * sp, vy = x[i].y * sp;
                acc.x += ar * vx - ai * vy;
                acc.y += ar * vy + ai * vx;
            }
        }
        psi[idx] = acc;
    }
};

// Imaginary-time step, part 2 (Eq. 24 in reading R-G25): n2 = dr sum |psi|^2;
// E = -ln(n2) / (2 dt) logged for the step; inv = 1/sqrt(n2) for the re-normalisation that follows.
struct OpImagNorm : OpBase {
    static constexpr int NRED = 1;
    const double2 *psi; const Ctl *ctl; int step_off, batch; double dr; double *elog, *inv;
    __device__ __forceinline__ void point(int, size_t idx, double *red) {
        const double2 v = psi[idx];
        red[0] += v.x * v.x + v.y * v.y;
    }
    __device__ __forceinline__ void finish_member(int b, const double *s) {
        const double n2 = dr * s[0];
        elog[(ctl->step_base + step_off) * batch + b] = -log(n2) / (2.0 * ctl->dt);
        inv[b] = 1.0 / sqrt(n2);
    }
};

struct OpScaleMember : OpBase {
    double2 *psi; const double *inv;
    __device__ __forceinline__ void point(int b, size_t idx, double *) {
        const double s = inv[b];
        double2 v = psi[idx];
        v.x *= s; v.y *= s;
        psi[idx] = v;
    }
};

// Absorbing boundary as a split step (Eq. 18, reading R-G26): psi_{l,j} *= mask_j after a propagator step.
struct OpMask : OpBase {
    double2 *psi; const double *mask; int n_r;
    __device__ __forceinline__ void point(int, size_t idx, double *) {
        const double m = __ldg(mask + (int)(idx % (size_t)n_r));
        double2 v = psi[idx];
        v.x *= m; v.y *= m;
        psi[idx] = v;
    }
};

// p_b = dr sum_l sum_{r_j <= r_b} |f_{l,j}|^2  (Eq. 26, reading R-G27)
struct OpBoundPop : OpBase {
    static constexpr int NRED = 1;
    const double2 *psi; int n_r, j_max; double dr; double *out;     // j_max: number of radial points with r_j <= r_b
    __device__ __forceinline__ void point(int, size_t idx, double *red) {
        if ((int)(idx % (size_t)n_r) < j_max) {
            const double2 v = psi[idx];
            red[0] += v.x * v.x + v.y * v.y;
        }
    }
    __device__ __forceinline__ void finish_member(int b, const double *s) { out[b] = dr * s[0]; }
};

// psi <- P psi: zero the points the centrifugal cut-off holds (tdse_set_cutoff, tdse_set_state)
struct OpProject : OpBase {
    double2 *psi; const int *j0; int n_r, n_l;
    __device__ __forceinline__ void point(int, size_t idx, double *) {
        const int j = (int)(idx % (size_t)n_r), l = (int)((idx / (size_t)n_r) % (size_t)n_l);
        if (j < __ldg(j0 + l)) psi[idx] = make_double2(0.0, 0.0);
    }
};

struct OpCopy : OpBase {
    double2 *dst; const double2 *src;
    __device__ __forceinline__ void point(int, size_t idx, double *) { dst[idx] = src[idx]; }
};

// ------------------------------------------------------------------------------------------------------
// c = exp(-i T dt) e_1 on the K x K real tridiagonal T by a sub-stepped Taylor series (Taylor1, P:511:
// "only one work group" -> one warp, lane i owns coefficient i; R-G18 for the sub-step count).
// grid = batch, block = 32.
// ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) small_exp_kernel(const double *alpha, const double *beta, const int *m_used,
                                                       const double *dtp, int K, int order, double2 *coef,
                                                       int *n_sub_out) {
    const int b = blockIdx.x, i = threadIdx.x;
    const int m = m_used[b];
    const double dt = *dtp;
    const bool on = i < m;
    const double a = on ? alpha[b * K + i] : 0.0;
    const double bl = (on && i > 0) ? beta[b * K + i - 1] : 0.0;        // beta_{i-1}
    const double br = (on && i < m - 1) ? beta[b * K + i] : 0.0;        // beta_i
    double gr = on ? (fabs(a) + bl + br) : 0.0;                          // Gershgorin radius of row i
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) gr = fmax(gr, __shfl_xor_sync(0xffffffffu, gr, off));
    int s = (int)ceil(dt * gr / 3.0);
    if (s < 1) s = 1;
    const double h = dt / (double)s;
    double2 c = make_double2(i == 0 ? 1.0 : 0.0, 0.0);
    for (int rep = 0; rep < s; ++rep) {
        double2 t = c;
        for (int k = 1; k <= order; ++k) {
            const double tlx = __shfl_up_sync(0xffffffffu, t.x, 1), tly = __shfl_up_sync(0xffffffffu, t.y, 1);
            const double trx = __shfl_down_sync(0xffffffffu, t.x, 1), try_ = __shfl_down_sync(0xffffffffu, t.y, 1);
            double ux = a * t.x, uy = a * t.y;
            if (i > 0) { ux += bl * tlx; uy += bl * tly; }
            if (i < m - 1) { ux += br * trx; uy += br * try_; }
            const double f = h / (double)k;
            t = on ? make_double2(f * uy, -f * ux) : make_double2(0.0, 0.0);
            c.x += t.x; c.y += t.y;
        }
    }
    if (i < K) coef[b * K + i] = on ? c : make_double2(0.0, 0.0);
    if (i == 0) n_sub_out[b] = s;
}

// ------------------------------------------------------------------------------------------------------
// Field tables and control kernels (time loop, row a7).
// ------------------------------------------------------------------------------------------------------
// mode 0: Taylor/Lanczos (one value per step, at t_n + dt/2 or t_n);  mode 1: RK4 (4 stage times).
// e_tab[(step*n_stage + stage)*B + b]
__global__ void field_table_kernel(const Ctl *ctl, const tdse_pulse *pulse, int B, int n_steps, int mode,
                                   double *e_tab, int gauge) {
    const int n_stage = (mode == 1) ? 4 : 1;
    const int total = n_steps * n_stage * B;
    const double t0 = ctl->t0, dt = ctl->dt;
    const long long base = ctl->step_base;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int b = i % B, st = (i / B) % n_stage, s = i / (B * n_stage);
        const double n = (double)(base + s);
        double t;
        if (mode == 1) {
            const double c = (st == 0) ? 0.0 : (st == 3 ? 1.0 : 0.5);
            t = __dadd_rn(time_at(t0, n, dt), __dmul_rn(c, dt));
        } else {
            t = ctl->field_sample == 1 ? time_at(t0, n, dt) : time_at(t0, n + 0.5, dt);
        }
        e_tab[i] = pulse_field(pulse[b], t, gauge);      // E(t), or A(t) in the velocity gauge
    }
}

// field values at the stage times t_n + c_i dt of any tableau: e_tab[(step*n_stage + stage)*B + b]
struct StageTimes { double c[7]; };
__global__ void field_table_rk_kernel(const Ctl *ctl, const tdse_pulse *pulse, int B, int n_steps, int n_stage,
                                      StageTimes cs, double *e_tab, int gauge) {
    const int total = n_steps * n_stage * B;
    const double t0 = ctl->t0, dt = ctl->dt;
    const long long base = ctl->step_base;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int b = i % B, st = (i / B) % n_stage, s = i / (B * n_stage);
        const double t = __dadd_rn(time_at(t0, (double)(base + s), dt), __dmul_rn(cs.c[st], dt));
        e_tab[i] = pulse_field(pulse[b], t, gauge);
    }
}

// Velocity gauge, pulses given by their field (kind 0): the field tables come from the running quadrature of P:186-188 /
// P:480.  a_run[b] holds A(t_n) of the first step of the block and is advanced past its last step; one thread per
// member walks the steps in order (the sum is sequential by definition).  Members whose pulse has a closed-form A(t)
// get exactly the values of field_table_kernel / field_table_rk_kernel.  e_tab[(step*n_stage + stage)*B + b].
// mid_rule: 1 for Taylor / Lanczos (n_stage = 1, sample at t_n + dt/2 or, field_sample = 1, at t_n), 0 for stage times cs.
__global__ void field_table_quad_kernel(const Ctl *ctl, const tdse_pulse *pulse, int B, int n_steps, int n_stage,
                                        StageTimes cs, int mid_rule, double *e_tab, double *a_run) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const tdse_pulse p = pulse[b];
    const bool quad = pulse_needs_quadrature(p, 1);
    const double t0 = ctl->t0, dt = ctl->dt;
    const long long base = ctl->step_base;
    double a = a_run[b];
    for (int s = 0; s < n_steps; ++s) {
        const double n = (double)(base + s);
        const double tn = time_at(t0, n, dt);
        for (int st = 0; st < n_stage; ++st) {
            double v;
            if (mid_rule) {
                const bool at_start = ctl->field_sample == 1;
                if (quad) v = at_start ? a : a - gl5_field(p, tn, tn + 0.5 * dt);
                else v = pulse_A(p, at_start ? tn : time_at(t0, n + 0.5, dt));
            } else {
                const double c = cs.c[st];
                if (quad) v = (c == 0.0) ? a : a - gl5_field(p, tn, tn + c * dt);
                else v = pulse_A(p, __dadd_rn(tn, __dmul_rn(c, dt)));
            }
            e_tab[((size_t)s * n_stage + st) * B + b] = v;
        }
        if (quad) a -= gl5_field(p, tn, tn + dt);
    }
    a_run[b] = a;
}

// A(t0) of the members that need the quadrature (reading R-V4): minus the 5-point rule summed over the panels
// [m dt, (m+1) dt] from 0 and the last partial panel up to t0.  grid = batch, block = 256.
__global__ void __launch_bounds__(256) vecpot_init_kernel(const Ctl *ctl, const tdse_pulse *pulse, double *a_run) {
    __shared__ double red_s[8];
    const int b = blockIdx.x;
    const tdse_pulse p = pulse[b];
    const double t0 = ctl->t0, dt = ctl->dt;
    double acc[1] = {0.0};
    const bool quad = pulse_needs_quadrature(p, 1) && t0 > 0.0;
    long long m = 0;
    if (quad) {
        m = (long long)floor(t0 / dt);
        for (long long i = threadIdx.x; i < m; i += 256) acc[0] -= gl5_field(p, (double)i * dt, (double)(i + 1) * dt);
    }
    block_reduce<256, 1>(acc, red_s);
    if (threadIdx.x == 0) {
        double a = acc[0];
        if (quad && t0 > (double)m * dt) a -= gl5_field(p, (double)m * dt, t0);
        a_run[b] = quad ? a : 0.0;
    }
}

__global__ void ctl_init_kernel(Ctl *c, CtlInit v) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        c->t0 = v.t0; c->dt = v.dt; c->step_base = 0; c->obs_every = v.obs_every; c->field_sample = v.field_sample;
        c->t = v.t; c->h = v.h; c->t_end = v.t_end; c->rtol = v.rtol; c->dt_max = v.dt_max;
        c->done = 0; c->last = 0; c->after_reject = 0; c->replay = v.replay;
        c->n_accept = 0; c->n_reject = 0; c->n_attempt = 0; c->n_replay = v.n_replay; c->max_log = v.max_log;
        for (int i = 0; i < kRkRoles; ++i) c->perm[i] = i;
    }
}

__global__ void ctl_advance_kernel(Ctl *c, int n) {
    if (threadIdx.x == 0 && blockIdx.x == 0) c->step_base += n;
}

// Loop condition of the device-driven adaptive run (a CUDA-graph WHILE node around a block of attempted steps): go on
// while the controller has not finished and its step is still a positive finite number.
__global__ void rk45_cond_kernel(const Ctl *c, cudaGraphConditionalHandle handle) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const bool stop = c->done || !(c->h > 0.0) || c->n_attempt > (1LL << 40);
        cudaGraphSetConditional(handle, stop ? 0u : 1u);
    }
}

// Start of an attempted Dormand-Prince step: clip the step to t_end (or take the replayed one) and tabulate
// E_b(t + c_i h) for the 7 stages.  e_tab[stage*B + b].  One block.
__global__ void rk45_begin_kernel(Ctl *c, const tdse_pulse *pulse, int B, const double *replay, double *e_tab,
                                  int gauge) {
    if (c->done) return;
    __shared__ double sh_h;
    if (threadIdx.x == 0) {
        double h = c->h;
        if (c->replay) {
            h = replay[c->n_attempt];
            c->last = 0;
        } else if (__dadd_rn(c->t, h) >= c->t_end) {
            h = c->t_end - c->t; c->last = 1;
        } else {
            c->last = 0;
        }
        c->h = h;
        sh_h = h;
    }
    __syncthreads();
    const double h = sh_h, t = c->t;
    const double cs[7] = {0.0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1.0, 1.0};
    for (int i = threadIdx.x; i < 7 * B; i += blockDim.x) {
        const int st = i / B, b = i - st * B;
        e_tab[i] = pulse_field(pulse[b], __dadd_rn(t, __dmul_rn(cs[st], h)), gauge);
    }
}

// ------------------------------------------------------------------------------------------------------
// Observables (row a6): norm, dipole and acceleration sums, bound-state overlaps and the row assembly in one launch.
// A thread takes one radial column of a chunk of kObsRows partial waves (plus the first row of the next chunk for
// the l, l+1 products) with all its loads issued at once -- a serial march over all l was latency-bound (64
// dependent iterations on CFG3).  grid = (ceil(n_r/256), batch, ceil(n_l/kObsRows) + n_states).
// ------------------------------------------------------------------------------------------------------
constexpr int kObsRows = 8;

// ONE launch per logged row for the sums: CTAs (chunk_r, b, z) reduce the norm / dipole / acceleration sums of a chunk;
// the last CTA of a member to finish (ticket counter) adds the partials in a fixed order and writes
// {norm, <z>, <z''>} of the row (Eq. 34, Eq. 36).  The bound-state populations of the row are written by
// pop_kernel below.  partials[b][chunks_r*chunks_l][3], counters[b] (zero between launches).
// t_direct: if use_direct, the time for -E(t); else t_{n+1} = t0 + (n+1) dt of the step being logged.
__global__ void __launch_bounds__(256) obs_kernel(GridDev g, const double2 *psi, int n_states, const tdse_pulse *pulse,
                                                  const Ctl *ctl, int step_off, int predicated, int use_direct,
                                                  double t_direct, double *partials, unsigned int *counters,
                                                  double *rows, int rows_per) {
    __shared__ double red_s[3 * 8];
    __shared__ int last_flag;
    long long row = 0;
    double t = t_direct;
    if (!use_direct) {
        const long long n = ctl->step_base + step_off + 1;
        if (predicated && (ctl->obs_every <= 0 || (n % ctl->obs_every) != 0)) return;
        row = n / ctl->obs_every - 1;
        t = time_at(ctl->t0, (double)n, ctl->dt);
    }
    const int chunks_r = gridDim.x, chunks_l = gridDim.z;     // chunks_l = l segments of rows_per rows
    const int b = blockIdx.y, j = blockIdx.x * 256 + threadIdx.x;
    double red[3] = {0.0, 0.0, 0.0};
    {
        const int l_lo = blockIdx.z * rows_per, l_hi = min(g.n_l, l_lo + rows_per);
        if (j < g.n_r) {
            double nn = 0.0, sz = 0.0;
            for (int l0 = l_lo; l0 < l_hi; l0 += kObsRows) {
                const double2 *p = psi + ((size_t)b * g.n_l + l0) * g.n_r + j;
                double2 v[kObsRows + 1];
#pragma unroll
                for (int r = 0; r <= kObsRows; ++r)
                    v[r] = (l0 + r < g.n_l) ? p[(size_t)r * g.n_r] : make_double2(0.0, 0.0);
#pragma unroll
                for (int r = 0; r < kObsRows; ++r) {
                    if (l0 + r >= l_hi) break;
                    nn += v[r].x * v[r].x + v[r].y * v[r].y;
                    if (l0 + r + 1 < g.n_l) sz = fma(__ldg(g.cl + l0 + r), v[r].x * v[r + 1].x + v[r].y * v[r + 1].y, sz);
                }
            }
            const double r = g.dr * (double)(j + 1);
            red[0] = nn; red[1] = r * sz; red[2] = sz / (r * r);
        }
        block_reduce<256, 3>(red, red_s);
        if (threadIdx.x == 0) {
            double *o = partials + (((size_t)b * chunks_r + blockIdx.x) * chunks_l + blockIdx.z) * 3;
            o[0] = red[0]; o[1] = red[1]; o[2] = red[2];
        }
    }
    // ---- last CTA of this member assembles the sums of the row ---------------------------------------------------
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int ticket = atomicAdd(counters + b, 1u);
        last_flag = (ticket == (unsigned int)(gridDim.x * gridDim.z - 1));
    }
    __syncthreads();
    if (!last_flag) return;
    __threadfence();
    const int W = 3 + n_states, chunks = chunks_r * chunks_l;
    double sum[3] = {0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < chunks; i += 256) {
        const double *p = partials + ((size_t)b * chunks + i) * 3;
        sum[0] += __ldcg(p); sum[1] += __ldcg(p + 1); sum[2] += __ldcg(p + 2);
    }
    block_reduce<256, 3>(sum, red_s);
    double *o = rows + ((size_t)row * g.batch + b) * W;
    if (threadIdx.x == 0) {
        o[0] = g.dr * sum[0];
        o[1] = 2.0 * g.dr * sum[1];
        o[2] = -pulse_E(pulse[b], t) - 2.0 * g.z * g.dr * sum[2];
        counters[b] = 0u;
    }
}

// Bound-state populations of a row (Eq. 25 with the modulus squared, R-G12): p_s = |dr sum_j phi_s[j] f_{l_s,j}|^2.
// grid = (n_l, batch): the CTA of (l, b) walks the states with l_s = l (state_list[l_off[l] .. l_off[l+1])), four at a
// time, so that the row f_l of a member is read from L1/L2 once per four states and a whole overlap is reduced inside one
// CTA in a fixed order -- the ~170 bound states of the CFG5 yield (R-G23) cost one launch.
__global__ void __launch_bounds__(256) pop_kernel(GridDev g, const double2 *psi, const double *phi, const int *l_off,
                                                  const int *state_list, int n_states, const Ctl *ctl, int step_off,
                                                  int predicated, int use_direct, double *rows) {
    __shared__ double red_s[8 * 8];
    long long row = 0;
    if (!use_direct) {
        const long long n = ctl->step_base + step_off + 1;
        if (predicated && (ctl->obs_every <= 0 || (n % ctl->obs_every) != 0)) return;
        row = n / ctl->obs_every - 1;
    }
    const int l = blockIdx.x, b = blockIdx.y;
    const int s_lo = l_off[l], s_hi = l_off[l + 1];
    if (s_lo == s_hi) return;
    const double2 *f = psi + ((size_t)b * g.n_l + l) * g.n_r;
    double *o = rows + ((size_t)row * g.batch + b) * (3 + n_states) + 3;
    for (int s0 = s_lo; s0 < s_hi; s0 += 4) {
        int sid[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) sid[i] = state_list[min(s0 + i, s_hi - 1)];
        double a[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        for (int j = threadIdx.x; j < g.n_r; j += 256) {
            const double2 v = f[j];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const double w = __ldg(phi + (size_t)sid[i] * g.n_r + j);
                a[2 * i] = fma(w, v.x, a[2 * i]); a[2 * i + 1] = fma(w, v.y, a[2 * i + 1]);
            }
        }
        block_reduce<256, 8>(a, red_s);
        if (threadIdx.x == 0) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (s0 + i < s_hi) {
                    const double ar = g.dr * a[2 * i], ai = g.dr * a[2 * i + 1];
                    o[sid[i]] = ar * ar + ai * ai;
                }
            }
        }
    }
}

// Ionisation yield from the bound-state populations of a row (CFG5, R-G23): 1 - sum_s p_s.  grid = batch, block = 32.
__global__ void __launch_bounds__(32) yield_kernel(const double *rows, int n_states, double *out) {
    const double *o = rows + (size_t)blockIdx.x * (3 + n_states) + 3;
    double s = 0.0;
    for (int i = threadIdx.x; i < n_states; i += 32) s += o[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
    if (threadIdx.x == 0) out[blockIdx.x] = 1.0 - s;
}

// The same for small grids: ONE CTA per member loops over all chunks and states, so that no cross-CTA hand-over
// (fence, ticket, second pass over partials) sits on the critical path of a launch-latency-bound step.
// grid = batch, block = 256.
__global__ void __launch_bounds__(256) obs_small_kernel(GridDev g, const double2 *psi, const double *phi,
                                                        const int *l_of_state, int n_states, const tdse_pulse *pulse,
                                                        const Ctl *ctl, int step_off, int predicated, int use_direct,
                                                        double t_direct, double *rows) {
    __shared__ double red_s[3 * 8];
    long long row = 0;
    double t = t_direct;
    if (!use_direct) {
        const long long n = ctl->step_base + step_off + 1;
        if (predicated && (ctl->obs_every <= 0 || (n % ctl->obs_every) != 0)) return;
        row = n / ctl->obs_every - 1;
        t = time_at(ctl->t0, (double)n, ctl->dt);
    }
    const int b = blockIdx.x, W = 3 + n_states;
    double *o = rows + ((size_t)row * g.batch + b) * W;
    double red[3] = {0.0, 0.0, 0.0};
    for (int j = threadIdx.x; j < g.n_r; j += 256) {
        const double2 *p = psi + (size_t)b * g.n_l * g.n_r + j;
        double nn = 0.0, sz = 0.0;
        for (int l0 = 0; l0 < g.n_l; l0 += kObsRows) {
            double2 v[kObsRows + 1];
#pragma unroll
            for (int r = 0; r <= kObsRows; ++r)
                v[r] = (l0 + r < g.n_l) ? p[(size_t)(l0 + r) * g.n_r] : make_double2(0.0, 0.0);
#pragma unroll
            for (int r = 0; r < kObsRows; ++r) {
                nn += v[r].x * v[r].x + v[r].y * v[r].y;
                if (l0 + r + 1 < g.n_l) sz = fma(__ldg(g.cl + l0 + r), v[r].x * v[r + 1].x + v[r].y * v[r + 1].y, sz);
            }
        }
        const double r = g.dr * (double)(j + 1);
        red[0] += nn; red[1] = fma(r, sz, red[1]); red[2] += sz / (r * r);
    }
    block_reduce<256, 3>(red, red_s);
    if (threadIdx.x == 0) {
        o[0] = g.dr * red[0];
        o[1] = 2.0 * g.dr * red[1];
        o[2] = -pulse_E(pulse[b], t) - 2.0 * g.z * g.dr * red[2];
    }
    for (int s = 0; s < n_states; ++s) {
        double a[3] = {0.0, 0.0, 0.0};
        const double2 *f = psi + ((size_t)b * g.n_l + l_of_state[s]) * g.n_r;
        for (int j = threadIdx.x; j < g.n_r; j += 256) {
            const double w = __ldg(phi + (size_t)s * g.n_r + j);
            const double2 v = f[j];
            a[0] = fma(w, v.x, a[0]); a[1] = fma(w, v.y, a[1]);
        }
        block_reduce<256, 3>(a, red_s);
        if (threadIdx.x == 0) {
            const double ar = g.dr * a[0], ai = g.dr * a[1];
            o[3 + s] = ar * ar + ai * ai;
        }
    }
}

}  // namespace tdse
