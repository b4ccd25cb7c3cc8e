// tdse_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See tdse_oracle.h.
//
// Plain CPU oracle for the CLTDSE hot path (arXiv:1308.1856; P:<n> = line n of
// /root/reference/PAPER.md).  Every function follows the cited passage step by
// step in the paper's order; nothing is blocked, fused or reordered.  Complex
// numbers are (re, im) pairs of doubles.  Build: oracle/build.py
// (g++ -O2 -ffp-contract=off -fopenmp, no fast-math).
#include "tdse_oracle.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

// the time-dependent factor of the coupling: E(t) in the length gauge, A(t) in the velocity gauge
static double coupling_field(const oracle_grid *g, const oracle_pulse *p, double t) {
    return g->gauge == 1 ? oracle_pulse_A(p, t) : oracle_pulse_E(p, t);
}

// ---- vector potential of a pulse given by its FIELD (kind 0) -- P:186-188: "we numerically calculate the potential
// field A(t), for each time step, as A(t_{n+1}) = A(t_n) - int_{t_n}^{t_n+h} E dtau, where the integral is performed using
// a standard 5-point Gaussian quadrature" (c dropped), and inside a step A(t_n + c_i h) = A(t_n) -
// int_{t_n}^{t_n + c_i h} E dtau.  Reading R-V4: a call that starts at t0 > 0 starts from
// A(t0) = - sum of the same 5-point rule over the panels [m dt, (m+1) dt] from 0 and the last partial panel up to t0.
static double gl5(const oracle_pulse *p, double ta, double tb) {
    // nodes and weights of the 5-point Gauss-Legendre rule on [-1, 1] (Abramowitz & Stegun 25.4.30, table 25.4)
    static const double x[5] = {-0.9061798459386640, -0.5384693101056831, 0.0, 0.5384693101056831, 0.9061798459386640};
    static const double w[5] = {0.2369268850561891, 0.4786286704993665, 0.5688888888888889, 0.4786286704993665,
                                0.2369268850561891};
    const double half = 0.5 * (tb - ta), mid = 0.5 * (tb + ta);
    double s = 0.0;
    for (int i = 0; i < 5; ++i) s += w[i] * oracle_pulse_E(p, mid + half * x[i]);
    return half * s;
}
static bool needs_quadrature(const oracle_grid *g, const oracle_pulse *p) {
    return g->gauge == 1 && p->omega != 0.0 && p->kind == 0;
}
struct VecPot {                     // A(t_n) of every member that needs the running quadrature
    std::vector<double> a;
    void init(const oracle_grid *g, const oracle_pulse *pulse, double t0, double dt) {
        a.assign(g->batch, 0.0);
        for (int b = 0; b < g->batch; ++b) {
            if (!needs_quadrature(g, &pulse[b]) || !(t0 > 0.0)) continue;
            const long m = (long)std::floor(t0 / dt);
            double acc = 0.0;
            for (long i = 0; i < m; ++i) acc -= gl5(&pulse[b], i * dt, (i + 1) * dt);
            if (t0 > m * dt) acc -= gl5(&pulse[b], m * dt, t0);
            a[b] = acc;
        }
    }
    // the time-dependent factor of the coupling at t_n + tau
    // (t_abs: the same instant as the propagator computes it, used by the pulses that have a closed form)
    double at(const oracle_grid *g, const oracle_pulse *pulse, int b, double tn, double tau, double t_abs) const {
        if (!needs_quadrature(g, &pulse[b])) return coupling_field(g, &pulse[b], t_abs);
        return tau == 0.0 ? a[b] : a[b] - gl5(&pulse[b], tn, tn + tau);
    }
    void advance(const oracle_grid *g, const oracle_pulse *pulse, double tn, double h) {
        for (int b = 0; b < g->batch; ++b)
            if (needs_quadrature(g, &pulse[b])) a[b] -= gl5(&pulse[b], tn, tn + h);
    }
};

namespace {

int g_threads = 1;

inline long n_points(const oracle_grid *g) { return (long)g->n_l * g->n_r; }
inline double r_of(const oracle_grid *g, int j) { return j * g->dr + g->r_offset; }  // j = 1..N_r

bool grid_ok(const oracle_grid *g) {
    return g && g->n_r >= 1 && g->n_l >= 1 && g->dr > 0.0 && g->batch >= 1 &&
           (g->fd_order == 3 || g->fd_order == 5);
}

// k_{l,l+1}(m = 0) = sqrt(l_>^2 / (4 l_>^2 - 1)), l_> = l + 1  (Eq. 9)  = (l+1)/sqrt((2l+1)(2l+3))
inline double coupling(int l) { return (l + 1) / std::sqrt((2.0 * l + 1.0) * (2.0 * l + 3.0)); }

// V_l(r) = l(l+1)/(2 r^2) - Z/r  (Eq. 7)
inline double v_eff(int l, double r, double z) { return l * (l + 1.0) / (2.0 * r * r) - z / r; }

// centrifugal inner cut-off (extension beyond the paper): point (l, j) is held at zero iff
// l(l+1)/(2 r_j^2) > Lambda, decided as l(l+1) > (2 Lambda) r_j^2 in this operation order
inline bool held(const oracle_grid *g, int l, int j) {
    if (!(g->cutoff_lambda > 0.0)) return false;
    const double r = r_of(g, j);
    return (double)(l * (l + 1)) > (2.0 * g->cutoff_lambda) * (r * r);
}

void project_member(const oracle_grid *g, double *f) {
    for (int l = 0; l < g->n_l; ++l)
        for (int j = 1; j <= g->n_r; ++j)
            if (held(g, l, j)) { f[2L * l * g->n_r + 2 * (j - 1)] = 0.0; f[2L * l * g->n_r + 2 * (j - 1) + 1] = 0.0; }
}
void project_all(const oracle_grid *g, double *psi) {
    if (!(g->cutoff_lambda > 0.0)) return;
    for (int b = 0; b < g->batch; ++b) project_member(g, psi + 2 * n_points(g) * b);
}

// one member: out = H(E) f.  f, out: [L][N_r] complex.  With a cut-off: out = P H P f (held points read as zero and
// come out as zero: the principal sub-matrix of H on the points that are not held).
void apply_H_member(const oracle_grid *g, const double *f, double e, double *out) {
    const int N = g->n_r, L = g->n_l;
    const double dr = g->dr, z = g->z_nuc;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int l = 0; l < L; ++l) {
        const double *fl = f + 2L * l * N;
        const double *flm = (l > 0) ? f + 2L * (l - 1) * N : nullptr;      // f_{l-1}; f_{-1} = 0
        const double *flp = (l < L - 1) ? f + 2L * (l + 1) * N : nullptr;  // f_{l+1}; f_{L}  = 0
        const double cm = (l > 0) ? coupling(l - 1) : 0.0;                  // kappa_{l}
        const double cp = coupling(l);                                      // kappa_{l+1}
        for (int j = 1; j <= N; ++j) {
            const double r = r_of(g, j);
            for (int c = 0; c < 2; ++c) {  // real and imaginary part: H is real
                auto F = [&](int jj) -> double {  // zero outside the box and at held points
                    return (jj >= 1 && jj <= N && !held(g, l, jj)) ? fl[2 * (jj - 1) + c] : 0.0;
                };
                double d2;
                if (g->fd_order == 3)
                    d2 = (F(j + 1) - 2.0 * F(j) + F(j - 1)) / (dr * dr);
                else  // P:122 Eq. 15
                    d2 = (-F(j + 2) + 16.0 * F(j + 1) - 30.0 * F(j) + 16.0 * F(j - 1) - F(j - 2)) /
                         (12.0 * dr * dr);
                const double kin = -0.5 * d2;
                const double pot = v_eff(l, r, z) * F(j);
                const double fm = (flm && !held(g, l - 1, j)) ? flm[2 * (j - 1) + c] : 0.0;
                const double fp = (flp && !held(g, l + 1, j)) ? flp[2 * (j - 1) + c] : 0.0;
                const double cpl = (g->gauge == 1) ? 0.0 : e * r * (cm * fm + cp * fp);  // P:104 Eq. 11, length gauge
                out[2L * l * N + 2 * (j - 1) + c] = kin + pot + cpl;
            }
            if (g->gauge == 1) {
                // P:106 Eq. 12 (e = A(t); the factor 1/c is dropped) in reading R-V2:
                //   -i A [ (d/dr - l/r) kappa_l f_{l-1} + (d/dr + (l+1)/r) kappa_{l+1} f_{l+1} ].
                // The printed equation has the two 1/r terms with the opposite signs; d/dz applied to
                // (f_l / r) Y_l0 gives the signs used here, and only they make the two gauges agree (pin P13).
                // d/dr by the central formula of the stencil (Eq. 14, reading R-V1), zero outside the box
                double s[2];
                for (int c = 0; c < 2; ++c) {
                    auto G = [&](const double *row, int lr, int jj) -> double {
                        return (row && jj >= 1 && jj <= N && !held(g, lr, jj)) ? row[2 * (jj - 1) + c] : 0.0;
                    };
                    auto D1 = [&](const double *row, int lr) -> double {
                        if (g->fd_order == 3) return (G(row, lr, j + 1) - G(row, lr, j - 1)) / (2.0 * dr);
                        return (-G(row, lr, j + 2) + 8.0 * G(row, lr, j + 1) - 8.0 * G(row, lr, j - 1) + G(row, lr, j - 2)) / (12.0 * dr);
                    };
                    s[c] = cm * (D1(flm, l - 1) - (l / r) * G(flm, l - 1, j)) + cp * (D1(flp, l + 1) + ((l + 1) / r) * G(flp, l + 1, j));
                }
                // -i (s0 + i s1) = s1 - i s0
                out[2L * l * N + 2 * (j - 1)] += e * s[1];
                out[2L * l * N + 2 * (j - 1) + 1] += -e * s[0];
            }
            if (held(g, l, j)) { out[2L * l * N + 2 * (j - 1)] = 0.0; out[2L * l * N + 2 * (j - 1) + 1] = 0.0; }
        }
    }
}

// y[i] += (ar + i ai) * x[i] over n complex elements
void caxpy(long n, double ar, double ai, const double *x, double *y) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (long i = 0; i < n; ++i) {
        const double xr = x[2 * i], xi = x[2 * i + 1];
        y[2 * i] += ar * xr - ai * xi;
        y[2 * i + 1] += ar * xi + ai * xr;
    }
}
// plain sums in index order (no dr factor)
void cdot(long n, const double *a, const double *b, double *re, double *im) {  // sum conj(a) b
    double sr = 0.0, si = 0.0;
    for (long i = 0; i < n; ++i) {
        sr += a[2 * i] * b[2 * i] + a[2 * i + 1] * b[2 * i + 1];
        si += a[2 * i] * b[2 * i + 1] - a[2 * i + 1] * b[2 * i];
    }
    *re = sr; *im = si;
}
double sumsq(long n, const double *a) {
    double s = 0.0;
    for (long i = 0; i < n; ++i) s += a[2 * i] * a[2 * i] + a[2 * i + 1] * a[2 * i + 1];
    return s;
}

void observables_member(const oracle_grid *g, const double *f, double e_now, int n_states,
                        const int *l_of_state, const double *phi, double *row) {
    const int N = g->n_r, L = g->n_l;
    const double dr = g->dr;
    // norm = dr sum |f|^2 (rectangle rule: the inner product under which H is Hermitian)
    row[0] = dr * sumsq((long)L * N, f);
    // <z> = 2 sum_l kappa_{l+1,0} Re int r f_l^* f_{l+1}      (Eq. 34)
    // <z''> = -E(t) - 2 Z sum_l kappa_{l+1,0} Re int r^-2 f_l^* f_{l+1}   (Eq. 36)
    double zsum = 0.0, asum = 0.0;
    for (int l = 0; l + 1 < L; ++l) {
        const double *a = f + 2L * l * N, *b = f + 2L * (l + 1) * N;
        double sz = 0.0, sa = 0.0;
        for (int j = 1; j <= N; ++j) {
            const double r = r_of(g, j);
            const double re = a[2 * (j - 1)] * b[2 * (j - 1)] + a[2 * (j - 1) + 1] * b[2 * (j - 1) + 1];
            sz += r * re;
            sa += re / (r * r);
        }
        zsum += coupling(l) * sz;
        asum += coupling(l) * sa;
    }
    row[1] = 2.0 * dr * zsum;
    row[2] = -e_now - 2.0 * g->z_nuc * dr * asum;
    // pop_s = | dr sum_j phi_s[j] f_{l_s, j} |^2        (Eq. 25 with modulus squared)
    for (int s = 0; s < n_states; ++s) {
        const double *p = phi + (long)s * N;
        const double *a = f + 2L * l_of_state[s] * N;
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < N; ++j) { sr += p[j] * a[2 * j]; si += p[j] * a[2 * j + 1]; }
        sr *= dr; si *= dr;
        row[3 + s] = sr * sr + si * si;
    }
}

void log_obs(const oracle_grid *g, const oracle_pulse *pulse, const double *psi, double t,
             const oracle_obs *obs, long block) {
    const int w = 3 + obs->n_states;
    for (int b = 0; b < g->batch; ++b)
        observables_member(g, psi + 2L * b * n_points(g), oracle_pulse_E(&pulse[b], t), obs->n_states,
                           obs->l_of_state, obs->phi, obs->obs_out + ((long)block * g->batch + b) * w);
}

// ---- Runge-Kutta tableaux -------------------------------------------------
struct Tableau { int s; const double *c; const double *a; const double *b; const double *bh; };
// classic RK4 ("ClassicRK4")
const double rk4_c[4] = {0.0, 0.5, 0.5, 1.0};
const double rk4_a[16] = {0, 0, 0, 0, 0.5, 0, 0, 0, 0, 0.5, 0, 0, 0, 0, 1.0, 0};
const double rk4_b[4] = {1.0 / 6, 1.0 / 3, 1.0 / 3, 1.0 / 6};
// Dormand-Prince 5(4), 7 stages, FSAL (named P:796; coefficients: Dormand & Prince 1980)
const double dp_c[7] = {0.0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1.0, 1.0};
const double dp_a[49] = {
    0, 0, 0, 0, 0, 0, 0,
    1.0 / 5, 0, 0, 0, 0, 0, 0,
    3.0 / 40, 9.0 / 40, 0, 0, 0, 0, 0,
    44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0, 0,
    19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0, 0,
    9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0, 0,
    35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0};
const double dp_b[7] = {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0};
const double dp_bh[7] = {5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40};

// The other methods named at P:796 / P:813 (coefficients from the literature; the order conditions of every row
// are verified in exact rationals in tests/test_oracle_pins.py).  b = the higher-order weights, which are the ones
// propagated (reading R-C4 / R-G28); bh = the lower-order companion.
const double eu_c[1] = {0.0}, eu_a[1] = {0.0}, eu_b[1] = {1.0};
// Runge-Kutta-Fehlberg 4(5)
const double rkf_c[6] = {0.0, 1.0 / 4, 3.0 / 8, 12.0 / 13, 1.0, 1.0 / 2};
const double rkf_a[36] = {
    0, 0, 0, 0, 0, 0,
    1.0 / 4, 0, 0, 0, 0, 0,
    3.0 / 32, 9.0 / 32, 0, 0, 0, 0,
    1932.0 / 2197, -7200.0 / 2197, 7296.0 / 2197, 0, 0, 0,
    439.0 / 216, -8.0, 3680.0 / 513, -845.0 / 4104, 0, 0,
    -8.0 / 27, 2.0, -3544.0 / 2565, 1859.0 / 4104, -11.0 / 40, 0};
const double rkf_b[6] = {16.0 / 135, 0, 6656.0 / 12825, 28561.0 / 56430, -9.0 / 50, 2.0 / 55};
const double rkf_bh[6] = {25.0 / 216, 0, 1408.0 / 2565, 2197.0 / 4104, -1.0 / 5, 0};
// Cash-Karp 5(4)
const double ck_c[6] = {0.0, 1.0 / 5, 3.0 / 10, 3.0 / 5, 1.0, 7.0 / 8};
const double ck_a[36] = {
    0, 0, 0, 0, 0, 0,
    1.0 / 5, 0, 0, 0, 0, 0,
    3.0 / 40, 9.0 / 40, 0, 0, 0, 0,
    3.0 / 10, -9.0 / 10, 6.0 / 5, 0, 0, 0,
    -11.0 / 54, 5.0 / 2, -70.0 / 27, 35.0 / 27, 0, 0,
    1631.0 / 55296, 175.0 / 512, 575.0 / 13824, 44275.0 / 110592, 253.0 / 4096, 0};
const double ck_b[6] = {37.0 / 378, 0, 250.0 / 621, 125.0 / 594, 0, 512.0 / 1771};
const double ck_bh[6] = {2825.0 / 27648, 0, 18575.0 / 48384, 13525.0 / 55296, 277.0 / 14336, 1.0 / 4};
// Kutta-Merson 4(3)
const double me_c[5] = {0.0, 1.0 / 3, 1.0 / 3, 1.0 / 2, 1.0};
const double me_a[25] = {
    0, 0, 0, 0, 0,
    1.0 / 3, 0, 0, 0, 0,
    1.0 / 6, 1.0 / 6, 0, 0, 0,
    1.0 / 8, 0, 3.0 / 8, 0, 0,
    1.0 / 2, 0, -3.0 / 2, 2.0, 0};
const double me_b[5] = {1.0 / 6, 0, 0, 2.0 / 3, 1.0 / 6};
const double me_bh[5] = {1.0 / 10, 0, 3.0 / 10, 2.0 / 5, 1.0 / 5};

// 0 ClassicRK4, 1 DormandPrince, 2 Euler, 3 RKF, 4 CashKarp, 5 Merson (the names of P:796)
Tableau tableau_of(int id) {
    switch (id) {
        case 1: return {7, dp_c, dp_a, dp_b, dp_bh};
        case 2: return {1, eu_c, eu_a, eu_b, nullptr};
        case 3: return {6, rkf_c, rkf_a, rkf_b, rkf_bh};
        case 4: return {6, ck_c, ck_a, ck_b, ck_bh};
        case 5: return {5, me_c, me_a, me_b, me_bh};
        default: return {4, rk4_c, rk4_a, rk4_b, nullptr};
    }
}

// One RK step of size h from t for all members.  k: s arrays of B*L*N complex.
// k1_valid: k[0] already holds f(t, psi) (FSAL).  On return psi_new holds the b-solution,
// *err = max_b ||Delta_b|| / ||psi_new,b||  (0 without an embedded pair).  psi is not modified.
void rk_step(const oracle_grid *g, const oracle_pulse *pulse, const Tableau &tb, const double *psi,
             double t, double h, std::vector<std::vector<double>> &k, bool k1_valid,
             std::vector<double> &gbuf, std::vector<double> &hbuf, double *psi_new, double *err,
             const VecPot &vp) {
    const long M = n_points(g);
    const int B = g->batch;
    for (int i = (k1_valid ? 1 : 0); i < tb.s; ++i) {
        // g <- f_n + h sum_{j<i} a_ij k_j
        std::memcpy(gbuf.data(), psi, sizeof(double) * 2 * M * B);
        for (int j = 0; j < i; ++j) {
            const double aij = tb.a[i * tb.s + j];
            if (aij != 0.0) caxpy(M * B, h * aij, 0.0, k[j].data(), gbuf.data());
        }
        // k_i <- f(t_n + c_i h, g) = -i H(t_n + c_i h) g      (Eq. 17)
        for (int b = 0; b < B; ++b) {
            const double e = vp.at(g, pulse, b, t, tb.c[i] * h, t + tb.c[i] * h);   // (P:480 for a pulse given by its field)
            apply_H_member(g, gbuf.data() + 2 * M * b, e, hbuf.data() + 2 * M * b);
        }
        double *ki = k[i].data();
        for (long n = 0; n < M * B; ++n) {  // multiply by -i: (x + iy) -> (y - ix)
            ki[2 * n] = hbuf[2 * n + 1];
            ki[2 * n + 1] = -hbuf[2 * n];
        }
    }
    // f_{n+1} <- f_n + h sum b_i k_i
    std::memcpy(psi_new, psi, sizeof(double) * 2 * M * B);
    for (int i = 0; i < tb.s; ++i)
        if (tb.b[i] != 0.0) caxpy(M * B, h * tb.b[i], 0.0, k[i].data(), psi_new);
    *err = 0.0;
    if (tb.bh) {
        // Delta = F^(2) - F^(1) = h sum (b_i - bh_i) k_i
        std::fill(gbuf.begin(), gbuf.end(), 0.0);
        for (int i = 0; i < tb.s; ++i) {
            const double d = tb.b[i] - tb.bh[i];
            if (d != 0.0) caxpy(M * B, h * d, 0.0, k[i].data(), gbuf.data());
        }
        for (int b = 0; b < B; ++b) {
            const double e = std::sqrt(sumsq(M, gbuf.data() + 2 * M * b)) /
                             std::sqrt(sumsq(M, psi_new + 2 * M * b));
            if (e > *err) *err = e;
        }
    }
}

// ---- symmetric band matrix h_l (half bandwidth w = 1 or 2) -------------------
struct Band { int n, w; std::vector<double> d, e1, e2; };  // diagonal, first, second off-diagonal

Band band_of(const oracle_grid *g, int l) {
    Band m; m.n = g->n_r; m.w = (g->fd_order == 3) ? 1 : 2;
    const double dr2 = g->dr * g->dr;
    m.d.resize(m.n); m.e1.assign(m.n, 0.0); m.e2.assign(m.n, 0.0);
    for (int j = 1; j <= m.n; ++j) {
        const double v = v_eff(l, r_of(g, j), g->z_nuc);
        if (m.w == 1) { m.d[j - 1] = 1.0 / dr2 + v; m.e1[j - 1] = -0.5 / dr2; }
        else { m.d[j - 1] = 30.0 / (24.0 * dr2) + v; m.e1[j - 1] = -16.0 / (24.0 * dr2); m.e2[j - 1] = 1.0 / (24.0 * dr2); }
    }
    return m;
}
inline double band_at(const Band &m, int i, int j) {  // symmetric access
    if (i > j) std::swap(i, j);
    const int k = j - i;
    if (k == 0) return m.d[i];
    if (k == 1) return m.e1[i];
    if (k == 2 && m.w == 2) return m.e2[i];
    return 0.0;
}
// number of eigenvalues < sigma: negative pivots of the LDL^T of (A - sigma I) (Sylvester inertia)
int count_below(const Band &m, double sigma) {
    const int n = m.n, w = m.w;
    std::vector<double> D(n);
    std::vector<double> Lm((size_t)n * (w + 1), 0.0);  // Lm[i*(w+1) + (i-k)] = L_ik for k = i-w..i-1
    int cnt = 0;
    for (int i = 0; i < n; ++i) {
        for (int k = std::max(0, i - w); k < i; ++k) {  // L_ik
            double s = band_at(m, i, k);
            for (int p = std::max(0, i - w); p < k; ++p)
                if (k - p <= w) s -= Lm[(size_t)i * (w + 1) + (i - p)] * Lm[(size_t)k * (w + 1) + (k - p)] * D[p];
            Lm[(size_t)i * (w + 1) + (i - k)] = s / D[k];
        }
        double di = m.d[i] - sigma;
        for (int p = std::max(0, i - w); p < i; ++p) {
            const double lip = Lm[(size_t)i * (w + 1) + (i - p)];
            di -= lip * lip * D[p];
        }
        if (std::fabs(di) < 1e-300) di = -1e-300;
        D[i] = di;
        if (di < 0.0) ++cnt;
    }
    return cnt;
}
// solve (A - sigma I) x = b, banded Gaussian elimination with partial pivoting; b overwritten by x
void band_solve(const Band &m, double sigma, std::vector<double> &b) {
    const int n = m.n, w = m.w, W = 3 * w + 1;
    // row r holds columns r-w .. r+2w at offset (c - (r - w))
    std::vector<double> A((size_t)n * W, 0.0);
    auto at = [&](int r, int c) -> double & { return A[(size_t)r * W + (c - (r - w))]; };
    for (int r = 0; r < n; ++r)
        for (int c = std::max(0, r - w); c <= std::min(n - 1, r + w); ++c)
            at(r, c) = band_at(m, r, c) - (r == c ? sigma : 0.0);
    for (int i = 0; i < n; ++i) {
        int p = i; double best = std::fabs(at(i, i));
        for (int r = i + 1; r <= std::min(n - 1, i + w); ++r)
            if (std::fabs(at(r, i)) > best) { best = std::fabs(at(r, i)); p = r; }
        const int cmax = std::min(n - 1, i + 2 * w);
        if (p != i) {
            for (int c = i; c <= cmax; ++c) std::swap(at(i, c), at(p, c));
            std::swap(b[i], b[p]);
        }
        if (std::fabs(at(i, i)) < 1e-300) at(i, i) = 1e-300;
        for (int r = i + 1; r <= std::min(n - 1, i + w); ++r) {
            const double f = at(r, i) / at(i, i);
            if (f == 0.0) continue;
            for (int c = i; c <= cmax; ++c) at(r, c) -= f * at(i, c);
            b[r] -= f * b[i];
        }
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = b[i];
        for (int c = i + 1; c <= std::min(n - 1, i + 2 * w); ++c) s -= at(i, c) * b[c];
        b[i] = s / at(i, i);
    }
}

// c = exp(-i T dt) e_1 by sub-stepped Taylor of order P on the m x m real tridiagonal T (P:511 Taylor1)
int small_exponential(int m, const double *alpha, const double *beta, int order, double dt,
                      double *coef /* [m] complex */) {
    // Gershgorin radius g = max_i(|alpha_i| + beta_{i-1} + beta_i); s = max(1, ceil(dt g / 3))
    double gr = 0.0;
    for (int i = 0; i < m; ++i) {
        double v = std::fabs(alpha[i]);
        if (i > 0) v += beta[i - 1];
        if (i < m - 1) v += beta[i];
        if (v > gr) gr = v;
    }
    int s = (int)std::ceil(dt * gr / 3.0);
    if (s < 1) s = 1;
    const double h = dt / s;
    std::vector<double> c(2 * m, 0.0), t(2 * m), u(2 * m);
    c[0] = 1.0;
    for (int rep = 0; rep < s; ++rep) {
        t = c;
        for (int k = 1; k <= order; ++k) {
            for (int i = 0; i < m; ++i)  // u = T t
                for (int q = 0; q < 2; ++q) {
                    double v = alpha[i] * t[2 * i + q];
                    if (i > 0) v += beta[i - 1] * t[2 * (i - 1) + q];
                    if (i < m - 1) v += beta[i] * t[2 * (i + 1) + q];
                    u[2 * i + q] = v;
                }
            const double f = h / k;  // t <- (-i h/k) u
            for (int i = 0; i < m; ++i) { t[2 * i] = f * u[2 * i + 1]; t[2 * i + 1] = -f * u[2 * i]; }
            for (int i = 0; i < 2 * m; ++i) c[i] += t[i];
        }
    }
    std::memcpy(coef, c.data(), sizeof(double) * 2 * m);
    return s;
}

// One Lanczos step for one member at frozen field e (reading R-C5).  q: K vectors of M complex.
int lanczos_member(const oracle_grid *g, double *psi, double e, int K, int order, double dt,
                   double beta_tol, std::vector<double> &q, std::vector<double> &w,
                   double *alpha, double *beta, double *coef, int *n_sub) {
    const long M = n_points(g);
    const double nrm = std::sqrt(sumsq(M, psi));  // ||F|| (plain 2-norm; dr factors cancel)
    // Q_1 <- F / ||F||
    for (long i = 0; i < 2 * M; ++i) q[i] = psi[i] / nrm;
    int m = K;
    for (int p = 0; p < K; ++p) {
        double *qp = q.data() + 2 * M * p;
        apply_H_member(g, qp, e, w.data());              // w = H q_p        (LanczosLoop1)
        double ar, ai;
        cdot(M, qp, w.data(), &ar, &ai);                  // alpha_p = Re<q_p|w>
        alpha[p] = ar;
        caxpy(M, -alpha[p], 0.0, qp, w.data());           // w -= alpha_p q_p  (LanczosLoop2)
        if (p > 0) caxpy(M, -beta[p - 1], 0.0, qp - 2 * M, w.data());  // w -= beta_{p-1} q_{p-1}
        beta[p] = std::sqrt(sumsq(M, w.data()));          // beta_p = ||w||   (NormKrylov)
        if (p == K - 1) break;                            // last beta not needed
        if (beta[p] < beta_tol) { m = p + 1; break; }     // "if beta = 0 then quit"
        double *qn = qp + 2 * M;
        for (long i = 0; i < 2 * M; ++i) qn[i] = w[i] / beta[p];
    }
    *n_sub = small_exponential(m, alpha, beta, order, dt, coef);
    // F(t+dt) = ||F|| sum_p c_p q_p      (Taylor2)
    std::fill(psi, psi + 2 * M, 0.0);
    for (int p = 0; p < m; ++p) caxpy(M, nrm * coef[2 * p], nrm * coef[2 * p + 1], q.data() + 2 * M * p, psi);
    return m;
}

}  // namespace

extern "C" {

void oracle_set_threads(int n) { g_threads = n < 1 ? 1 : n; }
int oracle_get_threads(void) { return g_threads; }

double oracle_pulse_E(const oracle_pulse *p, double t) {
    if (p->omega == 0.0) return p->e0;  // test aid: static field (frozen-H pins), not a paper pulse
    const double T = 2.0 * M_PI * p->n_cycles / p->omega;
    if (t < 0.0 || t > T) return 0.0;
    const double Om = p->omega / (2.0 * p->n_cycles);
    if (p->kind == 1) {
        // E = -dA/dt of A = -(e0/omega) sin^2(Om t) sin(omega t + cep): the expression printed at P:188 with the
        // normalisation 1/omega_0 restored (reading R-V3)
        const double s = std::sin(Om * t), c = std::cos(Om * t), ph = p->omega * t + p->cep;
        return (p->e0 / p->omega) * s * (2.0 * Om * c * std::sin(ph) + p->omega * s * std::cos(ph));
    }
    const double s = std::sin(Om * t);
    return p->e0 * s * s * std::cos(p->omega * t + p->cep);
}

double oracle_pulse_A(const oracle_pulse *p, double t) {
    if (p->omega == 0.0) return p->e0;  // test aid: static vector potential
    if (p->kind != 1) return std::nan("");
    const double T = 2.0 * M_PI * p->n_cycles / p->omega;
    if (t < 0.0 || t > T) return 0.0;
    const double s = std::sin(p->omega * t / (2.0 * p->n_cycles));
    return -(p->e0 / p->omega) * s * s * std::sin(p->omega * t + p->cep);
}

double oracle_gl5_field_integral(const oracle_pulse *p, double ta, double tb) { return gl5(p, ta, tb); }

int oracle_vecpot_running(const oracle_pulse *p, double t0, double dt, long nsteps, double *a_out) {
    if (!p || !(dt > 0.0) || nsteps < 0 || !a_out) return -1;
    // the running scheme of P:188 on the field E(t) of this pulse, whatever its kind (for a kind-1 pulse the result can
    // be compared with its analytic A(t): the paper's Fig. 8)
    const long m = (t0 > 0.0) ? (long)std::floor(t0 / dt) : 0;
    double acc = 0.0;
    for (long i = 0; i < m; ++i) acc -= gl5(p, i * dt, (i + 1) * dt);
    if (t0 > m * dt) acc -= gl5(p, m * dt, t0);
    a_out[0] = acc;
    for (long n = 0; n < nsteps; ++n) { acc -= gl5(p, t0 + n * dt, t0 + (n + 1) * dt); a_out[n + 1] = acc; }
    return 0;
}

void oracle_coupling(int n_l, double *c) { for (int l = 0; l < n_l; ++l) c[l] = coupling(l); }

int oracle_apply_H(const oracle_grid *g, const double *psi, const double *e_field, double *out) {
    if (!grid_ok(g) || !psi || !e_field || !out) return -1;
    const long M = n_points(g);
    for (int b = 0; b < g->batch; ++b) apply_H_member(g, psi + 2 * M * b, e_field[b], out + 2 * M * b);
    return 0;
}

int oracle_is_held(const oracle_grid *g, int l, int j) { return (grid_ok(g) && held(g, l, j)) ? 1 : 0; }

int oracle_project(const oracle_grid *g, double *psi) {
    if (!grid_ok(g) || !psi) return -1;
    project_all(g, psi);
    return 0;
}

int oracle_dense_H(const oracle_grid *g, double e_field, double *h) {
    if (!grid_ok(g) || !h) return -1;
    const int N = g->n_r, L = g->n_l;
    const long n = (long)N * L;
    const double dr2 = g->dr * g->dr;
    // P:134/Fig. 1: diagonal blocks h_l are multi-diagonal, off-diagonal blocks (l, l+-1)
    // are diagonal in the length gauge.  Loop over every pair of indices and ask which rule applies.
    for (int l = 0; l < L; ++l)
        for (int j = 1; j <= N; ++j)
            for (int lp = 0; lp < L; ++lp)
                for (int jp = 1; jp <= N; ++jp) {
                    double v = 0.0;
                    const int dj = std::abs(j - jp);
                    if (l == lp) {
                        if (g->fd_order == 3) {
                            if (dj == 0) v = 1.0 / dr2;            // -1/2 * (-2)/dr^2
                            else if (dj == 1) v = -0.5 / dr2;      // -1/2 * 1/dr^2
                        } else {
                            if (dj == 0) v = 15.0 / (12.0 * dr2);  // -1/2 * (-30)/(12 dr^2)
                            else if (dj == 1) v = -8.0 / (12.0 * dr2);
                            else if (dj == 2) v = 0.5 / (12.0 * dr2);
                        }
                        if (dj == 0) {
                            const double r = r_of(g, j);
                            v += 0.5 * l * (l + 1) / (r * r) - g->z_nuc / r;
                        }
                    } else if (std::abs(l - lp) == 1 && dj == 0) {
                        const int lg = std::max(l, lp);  // l_> of P:94 Eq. 9
                        v = e_field * r_of(g, j) * std::sqrt((double)lg * lg / (4.0 * lg * lg - 1.0));
                    }
                    if (held(g, l, j) || held(g, lp, jp)) v = 0.0;      // cut-off: rows and columns of held points vanish
                    h[((long)l * N + (j - 1)) * n + ((long)lp * N + (jp - 1))] = v;
                }
    return 0;
}

int oracle_bound_states(const oracle_grid *g, int l, int n_want, int only_negative,
                        double *energies, double *phi) {
    if (!grid_ok(g) || l < 0 || n_want < 0 || !energies || !phi) return -1;
    const Band m = band_of(g, l);
    const int n = m.n;
    // Gershgorin bounds
    double lo = 1e300, hi = -1e300;
    for (int i = 0; i < n; ++i) {
        double rad = 0.0;
        for (int k = 1; k <= m.w; ++k) {
            if (i - k >= 0) rad += std::fabs(band_at(m, i, i - k));
            if (i + k < n) rad += std::fabs(band_at(m, i, i + k));
        }
        lo = std::min(lo, m.d[i] - rad); hi = std::max(hi, m.d[i] + rad);
    }
    int found = 0;
    std::vector<double> x(n), prev;
    for (int k = 0; k < n_want && k < n; ++k) {
        // bisection for the (k+1)-th smallest eigenvalue
        double a = lo, b = hi;
        if (only_negative) { if (count_below(m, 0.0) <= k) break; b = 0.0; }
        for (int it = 0; it < 200; ++it) {
            const double mid = 0.5 * (a + b);
            if (mid == a || mid == b) break;
            if (count_below(m, mid) > k) b = mid; else a = mid;
        }
        double lam = 0.5 * (a + b);
        // inverse iteration from a deterministic start vector
        for (int i = 0; i < n; ++i) x[i] = 1.0 + 0.37 * std::sin(1.0 + 0.91 * i);
        for (int it = 0; it < 4; ++it) {
            band_solve(m, lam + 1e-13 * std::max(1.0, std::fabs(lam)), x);
            double s = 0.0;
            for (int i = 0; i < n; ++i) s += x[i] * x[i];
            s = 1.0 / std::sqrt(s);
            for (int i = 0; i < n; ++i) x[i] *= s;
        }
        // Rayleigh quotient (x has unit 2-norm)
        double rq = 0.0;
        for (int i = 0; i < n; ++i) {
            double hx = 0.0;
            for (int c = std::max(0, i - m.w); c <= std::min(n - 1, i + m.w); ++c) hx += band_at(m, i, c) * x[c];
            rq += x[i] * hx;
        }
        // normalise dr sum phi^2 = 1, sign phi(r_1) > 0  (reading R-C7)
        const double sc = (x[0] < 0.0 ? -1.0 : 1.0) / std::sqrt(g->dr);
        for (int i = 0; i < n; ++i) phi[(long)k * n + i] = sc * x[i];
        energies[k] = rq;
        ++found;
    }
    return found;
}

int oracle_observables(const oracle_grid *g, const double *psi, const double *e_now,
                       int n_states, const int *l_of_state, const double *phi, double *out) {
    if (!grid_ok(g) || !psi || !e_now || !out || n_states < 0) return -1;
    for (int s = 0; s < n_states; ++s) if (l_of_state[s] < 0 || l_of_state[s] >= g->n_l) return -1;
    for (int b = 0; b < g->batch; ++b)
        observables_member(g, psi + 2L * b * n_points(g), e_now[b], n_states, l_of_state, phi,
                           out + (long)b * (3 + n_states));
    return 0;
}

int oracle_step_taylor(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                       int order, double t0, double dt, long nsteps, int field_sample,
                       const oracle_obs *obs) {
    if (!grid_ok(g) || !pulse || !psi || order < 1 || nsteps < 0) return -1;
    project_all(g, psi);       // centrifugal cut-off (if any): the held points are zero from here on
    const long M = n_points(g);
    std::vector<double> term(2 * M), hterm(2 * M);
    long block = 0;
    VecPot vp;
    vp.init(g, pulse, t0, dt);
    for (long n = 0; n < nsteps; ++n) {
        const double ts = field_sample == 1 ? t0 + n * dt : t0 + (n + 0.5) * dt;  // reading R-G7
        for (int b = 0; b < g->batch; ++b) {
            double *f = psi + 2 * M * b;
            const double e = vp.at(g, pulse, b, t0 + n * dt, field_sample == 1 ? 0.0 : 0.5 * dt, ts);
            // F^(0) = F_n; F^(k) = (-i dt/k) H F^(k-1); F_{n+1} = sum_k F^(k)   (Eq. 37)
            std::memcpy(term.data(), f, sizeof(double) * 2 * M);
            for (int k = 1; k <= order; ++k) {
                apply_H_member(g, term.data(), e, hterm.data());
                const double s = dt / k;
                for (long i = 0; i < M; ++i) {  // (-i s)(x + iy) = s y - i s x
                    term[2 * i] = s * hterm[2 * i + 1];
                    term[2 * i + 1] = -s * hterm[2 * i];
                }
                for (long i = 0; i < 2 * M; ++i) f[i] += term[i];
            }
        }
        vp.advance(g, pulse, t0 + n * dt, dt);       // A(t_{n+1}) = A(t_n) - int E
        if (obs && obs->obs_every > 0 && (n + 1) % obs->obs_every == 0)
            log_obs(g, pulse, psi, t0 + (n + 1) * dt, obs, block++);
    }
    return 0;
}

// Imaginary-time ("diffusion") propagation: the field-free equation with -i -> 1, i.e.
// F^(k) = (-dt/k) H F^(k-1), F(t+dt) = sum_k F^(k) (the Taylor recursion of P:456 Eq. 37 with the replacement),
// followed by re-normalisation after every step.  Energy estimate P:212 Eq. 24; the norm taken is that of
// the whole wavefunction and, since <psi|psi> = exp(-2 E dt) for a normalised eigenstate evolved by exp(-H dt),
// E = -ln<psi(t+dt)|psi(t+dt)> / (2 dt)  (reading R-G25: the factor 2 is absent from the printed equation; the
// closed-form ground-state energy of the 3-point scheme pins it).
int oracle_step_imag(const oracle_grid *g, double *psi, int order, double dt, long nsteps, double *energy_out) {
    if (!grid_ok(g) || !psi || order < 1 || nsteps < 0 || !(dt > 0.0)) return -1;
    project_all(g, psi);       // centrifugal cut-off (if any): the held points are zero from here on
    const long M = n_points(g);
    std::vector<double> term(2 * M), hterm(2 * M);
    for (long n = 0; n < nsteps; ++n) {
        for (int b = 0; b < g->batch; ++b) {
            double *f = psi + 2 * M * b;
            std::memcpy(term.data(), f, sizeof(double) * 2 * M);
            for (int k = 1; k <= order; ++k) {
                apply_H_member(g, term.data(), 0.0, hterm.data());
                const double s = dt / k;
                for (long i = 0; i < 2 * M; ++i) term[i] = -s * hterm[i];
                for (long i = 0; i < 2 * M; ++i) f[i] += term[i];
            }
            double n2 = 0.0;
            for (long i = 0; i < 2 * M; ++i) n2 += f[i] * f[i];
            n2 *= g->dr;                                   // rectangle rule (reading R-G13)
            if (energy_out) energy_out[n * g->batch + b] = -std::log(n2) / (2.0 * dt);
            const double inv = 1.0 / std::sqrt(n2);
            for (long i = 0; i < 2 * M; ++i) f[i] *= inv;
        }
    }
    return 0;
}

int oracle_step_rk_fixed(const oracle_grid *g, const oracle_pulse *pulse, double *psi, int tableau,
                         double t0, double dt, long nsteps, double *err_out, const oracle_obs *obs) {
    if (!grid_ok(g) || !pulse || !psi || nsteps < 0 || tableau < 0 || tableau > 5) return -1;
    project_all(g, psi);       // centrifugal cut-off (if any): the held points are zero from here on
    const Tableau tb = tableau_of(tableau);
    const long MB = n_points(g) * g->batch;
    std::vector<std::vector<double>> k(tb.s, std::vector<double>(2 * MB));
    std::vector<double> gbuf(2 * MB), hbuf(2 * MB), next(2 * MB);
    long block = 0;
    VecPot vp;
    vp.init(g, pulse, t0, dt);
    for (long n = 0; n < nsteps; ++n) {
        double err;
        rk_step(g, pulse, tb, psi, t0 + n * dt, dt, k, false, gbuf, hbuf, next.data(), &err, vp);
        vp.advance(g, pulse, t0 + n * dt, dt);
        std::memcpy(psi, next.data(), sizeof(double) * 2 * MB);
        if (err_out) err_out[n] = err;
        if (obs && obs->obs_every > 0 && (n + 1) % obs->obs_every == 0)
            log_obs(g, pulse, psi, t0 + (n + 1) * dt, obs, block++);
    }
    return 0;
}

int oracle_step_rk4(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                    double t0, double dt, long nsteps, const oracle_obs *obs) {
    return oracle_step_rk_fixed(g, pulse, psi, 0, t0, dt, nsteps, nullptr, obs);
}

// Fixed-step propagation with any of the tableaux and the PASSIVE error sum of P:827-833: per member
// sigma_n = sqrt(|Delta|^2 / M), Delta = F^(2) - F^(1) = h sum (b_i - bh_i) k_i over the M complex elements of the
// member's vector (reading R-G19), sigma = sum_n sigma_n.  sigma_out[b] (may be NULL) receives sigma; 0 without a pair.
int oracle_step_rk_sigma(const oracle_grid *g, const oracle_pulse *pulse, double *psi, int tableau,
                         double t0, double dt, long nsteps, double *sigma_out, const oracle_obs *obs) {
    if (!grid_ok(g) || !pulse || !psi || nsteps < 0 || tableau < 0 || tableau > 5) return -1;
    project_all(g, psi);       // centrifugal cut-off (if any): the held points are zero from here on
    const Tableau tb = tableau_of(tableau);
    const long M = n_points(g), MB = M * g->batch;
    std::vector<std::vector<double>> k(tb.s, std::vector<double>(2 * MB));
    std::vector<double> gbuf(2 * MB), hbuf(2 * MB), next(2 * MB);
    if (sigma_out) for (int b = 0; b < g->batch; ++b) sigma_out[b] = 0.0;
    long block = 0;
    VecPot vp;
    vp.init(g, pulse, t0, dt);
    for (long n = 0; n < nsteps; ++n) {
        double err;
        rk_step(g, pulse, tb, psi, t0 + n * dt, dt, k, false, gbuf, hbuf, next.data(), &err, vp);   // gbuf <- Delta
        vp.advance(g, pulse, t0 + n * dt, dt);
        std::memcpy(psi, next.data(), sizeof(double) * 2 * MB);
        if (sigma_out && tb.bh)
            for (int b = 0; b < g->batch; ++b) sigma_out[b] += std::sqrt(sumsq(M, gbuf.data() + 2 * M * b) / (double)M);
        if (obs && obs->obs_every > 0 && (n + 1) % obs->obs_every == 0)
            log_obs(g, pulse, psi, t0 + (n + 1) * dt, obs, block++);
    }
    return 0;
}

int oracle_step_rk45(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                     double t0, double t_end, double dt_init, double rtol, double dt_max,
                     const double *dt_replay, long n_replay,
                     long *n_accept, long *n_reject, double *dt_log, double *err_log, long max_log) {
    if (!grid_ok(g) || !pulse || !psi || rtol <= 0.0) return -1;
    project_all(g, psi);       // centrifugal cut-off (if any): the held points are zero from here on
    const Tableau tb = tableau_of(1);
    const long MB = n_points(g) * g->batch;
    std::vector<std::vector<double>> k(tb.s, std::vector<double>(2 * MB));
    std::vector<double> gbuf(2 * MB), hbuf(2 * MB), next(2 * MB);
    long na = 0, nr = 0;
    double t = t0;
    bool fsal = false;
    VecPot vp;
    vp.init(g, pulse, t0, dt_replay ? (n_replay > 0 ? dt_replay[0] : 1.0) : dt_init);
    if (dt_replay) {
        for (long n = 0; n < n_replay; ++n) {
            double err;
            const double h = dt_replay[n];
            rk_step(g, pulse, tb, psi, t, h, k, fsal, gbuf, hbuf, next.data(), &err, vp);
            std::memcpy(psi, next.data(), sizeof(double) * 2 * MB);
            k[0].swap(k[6]); fsal = true;  // k_7 of this step is k_1 of the next (same time t_{n+1})
            if (na < max_log) { if (dt_log) dt_log[na] = h; if (err_log) err_log[na] = err / rtol; }
            vp.advance(g, pulse, t, h);
            ++na; t += h;
        }
    } else {
        if (!(dt_init > 0.0) || !(t_end > t0)) return -1;
        double h = dt_init;
        if (dt_max > 0.0 && h > dt_max) h = dt_max;
        bool after_reject = false;
        while (t < t_end) {
            bool last = false;
            if (t + h >= t_end) { h = t_end - t; last = true; }  // land on t_end exactly
            double e;
            rk_step(g, pulse, tb, psi, t, h, k, fsal, gbuf, hbuf, next.data(), &e, vp);
            const double err = e / rtol;
            double fac = 0.9 * std::pow(err, -0.2);
            if (!(fac >= 0.2)) fac = 0.2;   // also catches NaN
            if (fac > 5.0) fac = 5.0;
            if (err <= 1.0) {
                std::memcpy(psi, next.data(), sizeof(double) * 2 * MB);
                k[0].swap(k[6]); fsal = true;
                if (na < max_log) { if (dt_log) dt_log[na] = h; if (err_log) err_log[na] = err; }
                ++na;
                vp.advance(g, pulse, t, h);
                t = last ? t_end : t + h;
                if (after_reject && fac > 1.0) fac = 1.0;
                after_reject = false;
            } else {
                ++nr;
                if (fac > 1.0) fac = 1.0;
                after_reject = true;
                fsal = true;  // k[0] holds f(t, psi) for the unchanged (t, psi): reuse it
            }
            h *= fac;
            if (dt_max > 0.0 && h > dt_max) h = dt_max;
        }
    }
    if (n_accept) *n_accept = na;
    if (n_reject) *n_reject = nr;
    return 0;
}

int oracle_step_lanczos(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                        int krylov_dim, int taylor_order, double t0, double dt, long nsteps,
                        int field_sample, double beta_tol, const oracle_obs *obs) {
    if (!grid_ok(g) || !pulse || !psi || krylov_dim < 1 || taylor_order < 1 || nsteps < 0) return -1;
    project_all(g, psi);       // centrifugal cut-off (if any): the held points are zero from here on
    const long M = n_points(g);
    std::vector<double> q(2 * M * krylov_dim), w(2 * M);
    std::vector<double> alpha(krylov_dim), beta(krylov_dim), coef(2 * krylov_dim);
    long block = 0;
    VecPot vp;
    vp.init(g, pulse, t0, dt);
    for (long n = 0; n < nsteps; ++n) {
        const double ts = field_sample == 1 ? t0 + n * dt : t0 + (n + 0.5) * dt;
        for (int b = 0; b < g->batch; ++b) {
            int n_sub;
            lanczos_member(g, psi + 2 * M * b, vp.at(g, pulse, b, t0 + n * dt, field_sample == 1 ? 0.0 : 0.5 * dt, ts),
                           krylov_dim, taylor_order,
                           dt, beta_tol, q, w, alpha.data(), beta.data(), coef.data(), &n_sub);
        }
        vp.advance(g, pulse, t0 + n * dt, dt);
        if (obs && obs->obs_every > 0 && (n + 1) % obs->obs_every == 0)
            log_obs(g, pulse, psi, t0 + (n + 1) * dt, obs, block++);
    }
    return 0;
}

int oracle_lanczos_internals(const oracle_grid *g, const double *psi, double e_field,
                             int krylov_dim, int taylor_order, double dt, double beta_tol,
                             double *q, double *alpha, double *beta, double *coef, int *n_sub) {
    if (!grid_ok(g) || !psi || krylov_dim < 1) return -1;
    const long M = n_points(g);
    std::vector<double> qv(2 * M * krylov_dim, 0.0), w(2 * M), f(psi, psi + 2 * M);
    std::fill(alpha, alpha + krylov_dim, 0.0);
    std::fill(beta, beta + krylov_dim, 0.0);
    std::fill(coef, coef + 2 * krylov_dim, 0.0);
    const int m = lanczos_member(g, f.data(), e_field, krylov_dim, taylor_order, dt, beta_tol, qv, w,
                                 alpha, beta, coef, n_sub);
    std::memcpy(q, qv.data(), sizeof(double) * 2 * M * krylov_dim);
    return m;
}

}  // extern "C"
