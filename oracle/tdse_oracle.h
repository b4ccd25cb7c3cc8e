/*
 * tdse_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, host memory) of the
 * hot path of Ó Broin & Nikolopoulos, "A GPGPU based program to solve the TDSE
 * in intense laser fields through the finite difference approach"
 * (arXiv:1308.1856; text at /root/reference/PAPER.md, cited below as P:<line>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code, header,
 * table or helper with the CUDA path under paper_1308_1856_b200/csrc/, and
 * neither imports the other.
 *
 * Conventions (readings of the paper are listed in DESIGN.md, "Readings"):
 *   - state f[b][l][j-1], b = 0..B-1 members, l = 0..L-1 partial waves (m = 0),
 *     j = 1..N_r radial points r_j = j*dr (+ r_offset), complex128 stored as
 *     interleaved (re, im) doubles; f = 0 outside the index box.
 *   - all sums run in index order, j inner, l outer; no blocking, no fusion.
 *   - complex arithmetic is written out on (re, im) pairs.
 *   - compiled with -O2 -ffp-contract=off, no fast-math.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): every function below is pinned
 * by something other than itself; the list is in DESIGN.md "Oracle pins".
 * The only unpinned quantity is the paper's Example-1 population 0.27144
 * (P:644): "parity unpinned" -- its inputs are not recoverable from the text.
 */
#ifndef TDSE_ORACLE_H
#define TDSE_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int    n_r;       /* radial points N_r                                   */
    double dr;        /* spacing; r_j = j*dr + r_offset, j = 1..N_r          */
    int    n_l;       /* number of partial waves L (l = 0..L-1)     */
    int    fd_order;  /* 3 or 5 point second derivative (Eq. 15)       */
    double z_nuc;     /* V(r) = -z_nuc / r                            */
    int    batch;     /* B independent members                               */
    double r_offset;  /* the paper's grid `Offset`; 0 normally   */
    int    gauge;     /* 0 length gauge (Eq. 11), 1 velocity gauge (Eq. 12) */
    double cutoff_lambda; /* centrifugal inner cut-off Lambda (an EXTENSION beyond the paper, motivated
                         by P:454 "not always stable"): 0 = none; > 0: f_l(r_j) is held at zero wherever
                         l(l+1)/(2 r_j^2) > Lambda, i.e. H is replaced by its principal sub-matrix on the remaining
                         points (still real symmetric), which bounds the centrifugal part of rho(H) by Lambda */
} oracle_grid;

typedef struct {      /* kind 0: E(t) = e0 sin^2(omega t/(2 n_c)) cos(omega t + cep) */
    double e0, omega, n_cycles, cep;   /* on 0 <= t <= 2 pi n_c/omega, else 0 (Eq. 19);
                                          omega == 0: static field E(t) = e0 (test aid)              */
    int kind;         /* 1: the Hann shape is on the vector potential (reading R-V3):
                         A(t) = -(e0/omega) sin^2(omega t/(2 n_c)) sin(omega t + cep), E(t) = -dA/dt  */
} oracle_pulse;

/* --- pieces of H ------------------------------------------------------- */
double oracle_pulse_E(const oracle_pulse *p, double t);
/* A(t) with E = -dA/dt (Eq. 20 with the factor c dropped as in P:182); defined for kind 1 pulses and for the
 * static test aid (omega == 0: A = e0); NaN for kind 0, whose A(t) exists only as the running quadrature below. */
double oracle_pulse_A(const oracle_pulse *p, double t);
/* Vector potential of a pulse given by its FIELD (kind 0) in the velocity gauge: the running 5-point Gauss-Legendre
 * quadrature of P:186-188, A(t_{n+1}) = A(t_n) - int_{t_n}^{t_n+h} E dtau (c dropped), and inside a step
 * A(t_n + c_i h) = A(t_n) - int_{t_n}^{t_n + c_i h} E dtau.  A call that starts at t0 > 0 starts from the same
 * rule summed over the panels [m dt, (m+1) dt] from 0 and the last partial panel (reading R-V4).  Every propagator uses
 * this scheme when grid.gauge = 1 and pulse.kind = 0.
 *   oracle_gl5_field_integral: int_{ta}^{tb} E(tau) dtau by ONE 5-point rule.
 *   oracle_vecpot_running: a_out[0..nsteps] = A(t0), A(t0 + dt), ... by the running scheme on E(t) of `p` (any kind). */
double oracle_gl5_field_integral(const oracle_pulse *p, double ta, double tb);
int    oracle_vecpot_running(const oracle_pulse *p, double t0, double dt, long nsteps, double *a_out);
/* c[l] = (l+1)/sqrt((2l+1)(2l+3)), l = 0..n_l-1: k_{l,l+1}(m=0) of P:94 Eq. 9 */
void   oracle_coupling(int n_l, double *c);

/* out = H(E) psi, matrix-free (Eq. 11 with P:89 Eq. 7, Eq. 9, Eq. 15).
 * psi, out: [B][L][N_r] complex128; e_field: [B]. returns 0 or <0 on bad args.
 * With a centrifugal cut-off this is P H P: held points read as zero and come out as zero. */
int oracle_apply_H(const oracle_grid *g, const double *psi, const double *e_field, double *out);

/* Centrifugal cut-off: 1 if point (l, j), j = 1..N_r, is HELD at zero, i.e. cutoff_lambda > 0 and
 * l(l+1) > 2 Lambda r_j^2 (evaluated as (double)(l(l+1)) > (2.0*Lambda)*(r_j*r_j) with r_j = j*dr + r_offset). */
int oracle_is_held(const oracle_grid *g, int l, int j);
/* psi <- P psi: zero the held points of every member (the propagators do this on entry when a cut-off is set). */
int oracle_project(const oracle_grid *g, double *psi);

/* Dense real-symmetric H for ONE member (g->batch ignored), built entry by entry
 * from the block structure of P:134/P:142 (Fig. 1): h[(l*N_r + j-1)*n + (l'*N_r + j'-1)].
 * Written independently of oracle_apply_H so that the two check each other. */
int oracle_dense_H(const oracle_grid *g, double e_field, double *h);

/* --- bound states of the discrete h_l ("ground state corresponding to the
 * discretised numerical system"): lowest n_want eigenpairs of the symmetric band
 * matrix h_l by inertia-count bisection + inverse iteration. phi: [n_want][N_r],
 * normalised dr*sum phi^2 = 1, phi(r_1) > 0. If only_negative != 0 stop at E >= 0.
 * Returns number found (>= 0) or <0 on error. */
int oracle_bound_states(const oracle_grid *g, int l, int n_want, int only_negative,
                        double *energies, double *phi);

/* --- observables (Eq. 25, Eq. 34, Eq. 36) -------
 * row = { norm, <z>, <z''>, pop[0..n_states-1] } per member; out: [B][3+n_states].
 * e_now[b] = E(t) of member b used in <z''>. phi: [n_states][N_r] real. */
int oracle_observables(const oracle_grid *g, const double *psi, const double *e_now,
                       int n_states, const int *l_of_state, const double *phi, double *out);

/* --- propagators --------------------------------------------------------
 * All advance psi in place over nsteps steps of size dt from t0; member b sees
 * pulse[b]. field_sample: 0 = H frozen at t_n + dt/2 (default), 1 = at t_n
 * (Taylor and Lanczos only; RK uses its stage times).  If obs_every > 0 an
 * observable row block [B][3+n_states] is appended to obs_out after every
 * obs_every-th step, evaluated at t_{n+1} (obs_out must hold nsteps/obs_every blocks). */
typedef struct {
    int n_states; const int *l_of_state; const double *phi;  /* may be 0/NULL */
    int obs_every; double *obs_out;
} oracle_obs;

/* Imaginary-time propagation: term_k = (-dt/k) H term_{k-1} with E = 0, psi += term_k, then
 * psi /= ||psi||; energy_out[n*batch + b] = -ln<psi|psi> / (2 dt) before the re-normalisation (Eq. 24 in
 * reading R-G25).  psi must be normalised on entry for the first estimate to be meaningful. */
int oracle_step_imag(const oracle_grid *g, double *psi, int order, double dt, long nsteps, double *energy_out);

/* P:456 Eq. 37 (index corrected): term_k = (-i dt/k) H term_{k-1}, psi += term_k */
int oracle_step_taylor(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                       int order, double t0, double dt, long nsteps, int field_sample,
                       const oracle_obs *obs);

/* P:462 Eq. 38 with the classic RK4 tableau */
int oracle_step_rk4(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                    double t0, double dt, long nsteps, const oracle_obs *obs);

/* Any explicit tableau through the same stage loop: tableau id
 * 0 = ClassicRK4, 1 = DormandPrince 5(4), 2 = Euler, 3 = RKF 4(5), 4 = CashKarp 5(4), 5 = Merson 4(3) (the methods
 * named at P:796 / P:813), each advancing with its higher-order weights.
 * err_out (may be NULL) receives, per step, max_b ||Delta_b||_2 / ||psi_new,b||_2
 * (embedded-pair difference; 0 for RK4). */
int oracle_step_rk_fixed(const oracle_grid *g, const oracle_pulse *pulse, double *psi, int tableau,
                         double t0, double dt, long nsteps, double *err_out, const oracle_obs *obs);

/* The same with the passive error sum of P:827-833: sigma_out[b] = sum_n sqrt(|Delta_n,b|^2 / M), M = complex
 * elements per member (R-G19); may be NULL; 0 for the methods without an embedded pair. */
int oracle_step_rk_sigma(const oracle_grid *g, const oracle_pulse *pulse, double *psi, int tableau,
                         double t0, double dt, long nsteps, double *sigma_out, const oracle_obs *obs);

/* Adaptive Dormand-Prince 5(4) (paper: controller "not implemented"; ours, DESIGN.md R-C4):
 * err = max_b ||Delta_b|| / (rtol ||psi_new,b||); accept iff err <= 1;
 * dt_next = dt*clamp(0.9 err^-1/5, 0.2, 5) (<= 1 after a reject), capped at dt_max (<=0: none);
 * last step clipped to land on t_end; FSAL.  If dt_replay != NULL the n_replay given steps
 * are taken unconditionally (each still reports its err in err_log).
 * dt_log/err_log (may be NULL) receive accepted steps, at most max_log. */
int oracle_step_rk45(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                     double t0, double t_end, double dt_init, double rtol, double dt_max,
                     const double *dt_replay, long n_replay,
                     long *n_accept, long *n_reject, double *dt_log, double *err_log, long max_log);

/* Lanczos-Krylov step (App. B; reading R-C5 in DESIGN.md) */
int oracle_step_lanczos(const oracle_grid *g, const oracle_pulse *pulse, double *psi,
                        int krylov_dim, int taylor_order, double t0, double dt, long nsteps,
                        int field_sample, double beta_tol, const oracle_obs *obs);

/* Internals of one Lanczos step for ONE member at a fixed field (pin P9):
 * q: [krylov_dim][L][N_r] complex basis, alpha[K], beta[K] (beta[p] = ||w|| after step p),
 * coef: [K] complex Krylov coefficients c = exp(-i T dt) e_1, returns m = dimension used. */
int oracle_lanczos_internals(const oracle_grid *g, const double *psi, double e_field,
                             int krylov_dim, int taylor_order, double dt, double beta_tol,
                             double *q, double *alpha, double *beta, double *coef, int *n_sub);

void oracle_set_threads(int n);   /* OpenMP threads for the row loops (elementwise work only) */
int  oracle_get_threads(void);

#ifdef __cplusplus
}
#endif
#endif
