/*
 * tdse.h -- C ABI of the B200-native TDSE hot path (libtdse_b200.so).
 *
 * Method: O Broin & Nikolopoulos, "A GPGPU based program to solve the TDSE in intense laser
 * fields through the finite difference approach" (arXiv:1308.1856).  P:<n> below is line n of the
 * paper text; readings of garbled or silent passages are R-* in DESIGN.md.
 *
 * What the library does: applies the matrix-free finite-difference Hamiltonian
 *     (H f)_{l,j} = -1/2 D2 f_l |_j + [ l(l+1)/(2 r_j^2) - Z/r_j ] f_{l,j}
 *                   + E(t) r_j [ c_{l-1} f_{l-1,j} + c_l f_{l+1,j} ]                 (Eq. 11, Eq. 7)
 * with D2 the 3-point or the 5-point (Eq. 15) second difference, c_l = (l+1)/sqrt((2l+1)(2l+3))
 * (Eq. 9 at m = 0), r_j = j*dr, j = 1..n_r, f = 0 outside the index box, and advances
 * i dF/dt = H(t) F (Eq. 17) with the paper's propagators.  Every step runs in CUDA kernels for
 * sm_100a; there is no CPU fallback: without a CUDA device every compute entry point returns
 * TDSE_ERR_CUDA.
 *
 * Data layout.  A state is psi[b][l][j-1]: b = 0..batch-1 independent members, l = 0..n_l-1
 * partial waves (block-contiguous in r), complex128 stored as interleaved (re, im) doubles,
 * 16-byte aligned.  "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors);
 * "host" pointers are ordinary host memory owned by the caller, only touched during the call.
 *
 * Streams.  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Work is
 * enqueued asynchronously on it unless the call returns data to the host, in which case the call
 * synchronises that stream before returning.
 *
 * Errors.  Every function returns 0 (TDSE_OK) or a negative code; no exceptions cross the ABI, nothing
 * aborts, and the handle stays valid after an error.
 */
#ifndef TDSE_B200_H
#define TDSE_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define TDSE_OK               0
#define TDSE_ERR_ARG         (-1)   /* null pointer, non-positive size, order < 1, ...           */
#define TDSE_ERR_ALLOC       (-2)   /* host or device allocation failed                           */
#define TDSE_ERR_CUDA        (-3)   /* CUDA runtime error (no device, launch failure)             */
#define TDSE_ERR_NONFINITE   (-4)   /* a logged norm is NaN/Inf (unstable step size)       */
#define TDSE_ERR_UNSUPPORTED (-5)   /* gauge not 0/1, fd_order not 3/5, krylov_dim > 32           */
#define TDSE_ERR_TOO_LARGE   (-6)   /* beyond the fixed scratch of tdse_observables_noalloc       */

typedef struct tdse_handle tdse_handle;   /* opaque; owns the state, all scratch, tables and CUDA graphs */

typedef struct {
    int    n_r;       /* radial points N_r; r_j = j*dr, j = 1..n_r (reading R-G1)          */
    double dr;        /* radial spacing                                                           */
    int    n_l;       /* number of partial-wave blocks L, l = 0..n_l-1 (`NumBlocks`)       */
    int    fd_order;  /* 3 or 5 point second derivative (Eq. 15)                            */
    int    gauge;     /* 0 = length gauge (Eq. 11), 1 = velocity gauge (Eq. 12 in reading R-V2,
                         first derivative of P:119 Eq. 14); else TDSE_ERR_UNSUPPORTED */
    double z_nuc;     /* V(r) = -z_nuc/r                                                   */
    int    batch;     /* B >= 1 independent members sharing the grid                      */
} tdse_grid;

typedef struct {      /* E(t) = e0 sin^2(omega t/(2 n_cycles)) cos(omega t + cep) on 0 <= t <= 2 pi n_cycles/omega, */
    double e0, omega, n_cycles, cep;   /* else 0 (Eq. 19; R-G8).  omega == 0: static field e0 */
    int kind;         /* 0: as above.  1: the Hann shape is on the vector potential (R-V3):
                         A(t) = -(e0/omega) sin^2(omega t/(2 n_cycles)) sin(omega t + cep), E(t) = -dA/dt.
                         In the velocity gauge (tdse_grid.gauge = 1) a kind-0 pulse gets its A(t) from the running
                         5-point Gauss quadrature of the field, A(t_{n+1}) = A(t_n) - int E, with
                         A(t_n + c_i h) = A(t_n) - int_{t_n}^{t_n + c_i h} E inside a step; a call starting at
                         t0 > 0 starts from the same rule summed over panels of width dt from 0 (reading R-V4).  The
                         static test aid omega = 0 has the constant A = e0. */
} tdse_pulse;

/* Create / destroy.  tdse_create builds the device tables (diagonal of h_l, c_l) and allocates the state
 * (zero-initialised).  Survives repeated create/destroy cycles (the paper's program was not tested for
 * that). */
int  tdse_create (const tdse_grid *grid, tdse_handle **out);
void tdse_destroy(tdse_handle *h);

/* Options (all default to the value in brackets):
 *   "field_sample"     [0] 0: H frozen at t_n + dt/2 in Taylor/Lanczos steps, 1: at t_n (R-G7)
 *   "use_graph"        [1] capture blocks of steps in a CUDA graph
 *   "graph_steps"      [16] steps per captured graph (four times as many on the small grids whose launches take
 *                          several steps, option "persist")
 *   "apply_tma"        [1] tdse_apply_H: tiles fetched by TMA tensor copies (zero fill outside the index box by the
 *                          hardware) when n_r % 8 == 0 and the grid is many rounds of
 *                          resident CTAs; 2: whenever the layout allows it; 0: the (l, r) tile kernel
 *   "lanczos_tma"      [1] Lanczos pass: the (up to three) source arrays of a tile are fetched by TMA when
 *                          n_r % 8 == 0; 0: register-staged tile kernel
 *   "rk4_block"        [1] tdse_step_rk4: 1 all four stages in one pass over HBM (register-patch kernel in RK mode)
 *                          when the grid is at least one 128-column tile wide; 0 one kernel per stage
 *   "taylor_block"     [1] 0: one kernel per Taylor order; 1: temporally blocked step, all orders in one
 *                          pass over HBM (persistent register-patch kernel; n_l <= 128, else falls back to 0)
 *   "taylor_rp_variant" [-1] instantiation of the register-patch kernel (-1: heuristic; 0..4: 16 points per thread,
 *                          5..7: 8 points per thread, multi-step launches only)
 *   "taylor_rp_tma"    [-1] register-patch kernel: fetch tiles by TMA tensor copies (-1: heuristic, 0: never,
 *                          1: whenever n_r % 8 == 0 and the grid is wider than a tile)
 *   "persist"          [8] tdse_step_taylor on SMALL grids (at most one wave of CTAs; no cut-off; logged rows, if any,
 *                          fusable: at most 4 bound states): temporal blocking across steps -- the halo of a tile covers
 *                          up to this many steps, so one launch takes that many steps with psi in registers (halved
 *                          until the interior of a tile is at least half of it); 0 / 1: one launch per step
 *   "obs_fused"        [1] logged observable rows are reduced inside the register-patch step kernel (from the registers
 *                          that hold psi(t + dt); no extra pass over psi) when it runs on full tiles, at most 4 bound
 *                          states are set and the grid is at most 16 CTAs (beyond that the separate pass measured
 *                          faster); 2: wherever the kernel can; 0: always the separate observable kernels
 *   "lanczos_beta_tol" [1e-12] breakdown threshold on beta ("if beta = 0 then quit", R-G17)
 *   "rk45_dt_max"      [0 = none] cap on the adaptive step
 *   "rk4_persist"      [1] tdse_step_rk4 with obs_every = 0 and no absorber runs in the same persistent kernel as
 *                          "rk45_persist" below when the grid fits on chip (classic RK4 as an FSAL scheme of five stage
 *                          vectors, field values from a table, one launch per 2048 steps); 0: stage kernels
 *   "rk45_persist"     [1] tdse_step_rk45 runs as ONE persistent cooperative kernel when the grid fits the shared memory
 *                          of the device (batch * n_l * ceil(n_r / #SMs) <= 2048 points per CTA, batch <= 32): psi and
 *                          k_1..k_7 stay on chip (registers or shared memory) from t0 to t_end, neighbouring CTAs hand
 *                          their edge columns over as self-validating packets through L2, every CTA runs the controller
 *                          (the paper's kernel boundaries are its only global synchronisation); 0, a larger grid
 *                          or a device that cannot hold the grid at once: one kernel per stage, see below
 *   "rk45_loop"        [1] (stage by stage) tdse_step_rk45 runs as ONE graph launch: a CUDA-graph WHILE node repeats a block of attempted
 *                          steps until the device controller is done (no host poll); 0: the host enqueues blocks and
 *                          polls the `done` flag between them
 *   "rk45_check_every" [8] attempted steps per block of that loop (or between host checks) */
int  tdse_set_option(tdse_handle *h, const char *key, double value);

/* Absorbing boundary (Eq. 18): W(r) = (i/dt) ln{1 - cos^p[(pi/2)(1 - r/r_b)]} enters as a split step, i.e.
 * after every step of tdse_step_taylor / rk4 / lanczos the state is multiplied by exp(-i W(r_j) dt) =
 * 1 - cos^p[(pi/2)(1 - r_j/r_b)] (0 for r_j >= r_b) -- the factor Eq. 18 is built to give, independent of dt (reading
 * R-G26).  r_b <= 0 removes the absorber.  tdse_step_rk45 returns TDSE_ERR_UNSUPPORTED while one is set; the
 * imaginary-time propagation ignores it.  Synchronises the device. */
int  tdse_set_absorber(tdse_handle *h, double r_b, int p);

/* Centrifugal inner cut-off -- an EXTENSION beyond the paper, motivated by its remark that the
 * explicit propagators are "not always stable": with lambda > 0 every point (l, j) with l(l+1)/(2 r_j^2) > lambda
 * is HELD at zero and H is replaced by its principal sub-matrix on the remaining points (still real symmetric), so the
 * centrifugal part of the spectral radius is at most lambda and the stable step grows from about 1/(L^2/(2 dr^2)) to
 * about 1/(kappa/dr^2 + lambda).  The rule is evaluated as (double)(l(l+1)) > (2.0*lambda)*(r_j*r_j), r_j = j*dr.
 * Applies to tdse_apply_H (P H P: held inputs read as zero, held outputs are zero) and to every propagator; the
 * current state and every later tdse_set_state are projected.  lambda = 0 removes it.  Synchronises the device. */
int  tdse_set_cutoff(tdse_handle *h, double lambda);

/* One pulse per member, host array [batch]. */
int  tdse_set_pulse(tdse_handle *h, const tdse_pulse *per_member_host);

/* Real bound-state vectors for the population observable p_s = |dr sum_j phi_s[j] f_{l_s,j}|^2
 * (Eq. 25 with the modulus squared, R-G12).  l_of_state: host [n_states]; phi: host [n_states][n_r]. */
int  tdse_set_bound_states(tdse_handle *h, int n_states, const int *l_of_state, const double *phi);

/* Copy the whole state [batch][n_l][n_r] complex128 in / out.  is_device = 0: host pointer (the call
 * synchronises `stream`), 1: device pointer (asynchronous on `stream`), 2: PINNED host pointer, asynchronous on
 * `stream` (the caller keeps the buffer alive and synchronises the stream itself: lets the transfers of one handle
 * overlap the steps of another, e.g. a batch split over several handles and streams). */
int  tdse_set_state(tdse_handle *h, const void *psi, int is_device, void *stream);
int  tdse_get_state(tdse_handle *h, void *psi, int is_device, void *stream);

/* out = H(E) psi for caller-owned device arrays (must not alias); e_field_host: host [batch], the field
 * value each member sees (Eq. 11).  Asynchronous on `stream`. */
int  tdse_apply_H(tdse_handle *h, const void *psi_dev, void *out_dev, const double *e_field_host, void *stream);

/* Propagators.  All advance the handle's state in place over nsteps steps of size dt starting at t0;
 * member b sees pulse b.  If obs_every > 0 an observable row block is logged after every obs_every-th
 * step (evaluated at t_{n+1}); the log restarts at row 0 on every call.  Asynchronous on `stream`.
 *   taylor : F_{n+1} = sum_{k=0..order} F^(k), F^(k) = (-i dt/k) H F^(k-1)         (Eq. 37, R-G6)
 *   rk4    : classic Runge-Kutta through the stage loop of P:462 Eq. 38 / P:469-478
 *   lanczos: Krylov basis by the three-term recurrence, c = exp(-i T dt) e_1 by a (sub-stepped) Taylor
 *            series of order taylor_order on the tridiagonal T, F_{n+1} = ||F|| sum_p c_p q_p
 *            (App. B, R-C5); krylov_dim <= 32. */
int  tdse_step_taylor (tdse_handle *h, int order, double t0, double dt, long nsteps, int obs_every, void *stream);
int  tdse_step_rk4    (tdse_handle *h, double t0, double dt, long nsteps, int obs_every, void *stream);
int  tdse_step_lanczos(tdse_handle *h, int krylov_dim, int taylor_order, double t0, double dt, long nsteps,
                       int obs_every, void *stream);

/* Fixed-step propagation with any of the Runge-Kutta methods the paper lists: method 0 ClassicRK4,
 * 1 DormandPrince 5(4), 2 Euler, 3 RKF 4(5), 4 CashKarp 5(4), 5 Merson 4(3), through the stage loop of P:469-478; the
 * pairs advance with their higher-order weights and accumulate the PASSIVE error sum of P:827-833,
 * sigma_b = sum_n sqrt(|F2 - F1|^2_{n,b} / M) with M = n_l n_r (reading R-G19), read back by tdse_rk_sigma
 * (host [batch]; 0 for Euler and ClassicRK4; synchronises `stream`). */
int  tdse_step_rk(tdse_handle *h, int method, double t0, double dt, long nsteps, int obs_every, void *stream);
int  tdse_rk_sigma(tdse_handle *h, double *sigma_host, void *stream);

/* Imaginary-time ("diffusion") propagation for ground states: no field, -i -> 1, i.e.
 * F^(k) = (-dt/k) H F^(k-1), F_{n+1} = sum_{k<=order} F^(k), then F_{n+1} /= ||F_{n+1}|| (whole wavefunction of the
 * member, rectangle rule) after every step.  The energy estimate of the step, E = -ln<F_{n+1}|F_{n+1}> / (2 dt)
 * taken before the re-normalisation (Eq. 24 in reading R-G25), is logged on the device; the state must be
 * normalised on entry for the first estimate to be meaningful.  Asynchronous on `stream`. */
int  tdse_step_imag(tdse_handle *h, int order, double dt, long nsteps, void *stream);
/* Energy estimates of the last tdse_step_imag call: energy_host [rows][batch], at most max_rows rows.
 * Synchronises `stream`. */
int  tdse_energy_log(tdse_handle *h, double *energy_host, long max_rows, void *stream);

/* Embedded Dormand-Prince 5(4) (named P:796; error estimate P:813-833; the adaptive controller is ours,
 * R-C4, the paper's is "not implemented"): err = max_b ||Delta_b||_2 / (rtol ||psi_new,b||_2), accept iff
 * err <= 1, dt_next = dt clamp(0.9 err^(-1/5), 0.2, 5) (<= 1 right after a reject), last step clipped to t_end,
 * FSAL.  If dt_replay != NULL (host [n_replay]) exactly those steps are taken, all accepted.  TDSE_ERR_UNSUPPORTED
 * in the velocity gauge with kind-0 pulses (the running quadrature of A(t) serves the fixed-step propagators).
 * Synchronises `stream`; n_accept / n_reject may be NULL. */
int  tdse_step_rk45(tdse_handle *h, double t0, double t_end, double dt_init, double rtol,
                    const double *dt_replay, long n_replay, long *n_accept, long *n_reject, void *stream);

/* Observable row of member b: { norm, <z>, <z''>, pop[0..n_states-1] }:
 *   norm = dr sum |f|^2;  <z> = 2 dr sum_l c_l sum_j r_j Re(conj f_{l,j} f_{l+1,j})          (Eq. 34)
 *   <z''> = -E(t) - 2 Z dr sum_l c_l sum_j r_j^-2 Re(conj f_{l,j} f_{l+1,j})                  (Eq. 36)
 * tdse_observables: current state, field taken at time t; out_host: [batch][3 + n_states]; synchronises. */
int  tdse_observables(tdse_handle *h, double t, double *out_host, void *stream);
/* Bound population by spatial integration, out_host [batch]: p_b = sum_l int_0^{r_b} |f_l|^2 dr (Eq. 26,
 * rectangle rule over r_j <= r_b, reading R-G27); the spatial ionisation yield is p_i = 1 - p_b (Eq. 27-28),
 * plus the norm lost to an absorber.  Synchronises `stream`. */
int  tdse_bound_population(tdse_handle *h, double r_b, double *out_host, void *stream);
/* Rows logged by the last step call: out_host [rows][batch][3+n_states]; at most max_rows row blocks are
 * copied, *rows = number logged.  Synchronises the device.  TDSE_ERR_NONFINITE if a logged norm is not finite. */
int  tdse_obs_log(tdse_handle *h, double *out_host, long max_rows, long *rows);
/* Accepted step sizes (and their err values; err_host may be NULL) of the last tdse_step_rk45 call. */
int  tdse_dt_log(tdse_handle *h, double *dt_host, double *err_host, long max, long *n);
/* Krylov data of the LAST Lanczos step: alpha, beta host [batch][krylov_dim]; coef host [batch][krylov_dim]
 * complex (re, im); m_used, n_sub host [batch] (dimension used after breakdown, Taylor sub-steps). Any may be NULL. */
int  tdse_lanczos_info(tdse_handle *h, double *alpha, double *beta, double *coef, int *m_used, int *n_sub);

/* Ionisation yield of the current state from the bound-state populations (CFG5 of BASELINE.json: "final ionisation
 * yield 1 - sum of bound populations per member"; Eq. 25 generalised to every supplied bound state, reading
 * R-G23): out_host [batch] = 1 - sum_s p_s over the states of tdse_set_bound_states.  Synchronises `stream`. */
int  tdse_ionisation_yield(tdse_handle *h, double *out_host, void *stream);

/* Number of CUDA kernels this handle has launched so far (graph nodes counted per graph launch). */
long tdse_launch_count(tdse_handle *h);
/* Number of CUDA graphs this handle has captured and instantiated so far (a step call does that on first use of a
 * (propagator, order, block length, ...) combination; a timed region should see this number unchanged). */
long tdse_graph_instantiations(tdse_handle *h);
/* Kernel used by the last tdse_step_taylor call (after tdse_step_rk4: 3 / 4 if the four stages ran fused, else 0):
 * 0 one kernel per order, 3 persistent register-patch kernel with direct global loads, 4 the same with TMA tile
 * fetches (3, 4: all orders in one pass). */
int  tdse_taylor_was_blocked(tdse_handle *h);
/* Plan of the register-patch kernel the last tdse_step_taylor / tdse_step_rk4 / tdse_step_imag call ran with (any
 * pointer may be NULL): *variant = instantiation (index into the table of csrc/tdse_taylor_rp_plan.h; -1 if the call did
 * not use that kernel), *steps_per_launch = steps one launch takes (1, or up to option "persist" on small grids),
 * *ctas = CTAs of a launch.  Returns TDSE_OK. */
int  tdse_taylor_plan(tdse_handle *h, int *variant, int *steps_per_launch, int *ctas);
/* 1 if the last tdse_step_rk45 / tdse_step_rk4 call ran in the persistent on-chip kernel (options "rk45_persist",
 * "rk4_persist"), 0 if it ran stage by stage. */
int  tdse_rk45_was_persistent(tdse_handle *h);

/* Observables WITHOUT ANY ALLOCATION (row a6; Eq. 34, Eq. 36): for callers that cannot call cudaMalloc
 * (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).  No handle: the caller passes the
 * inputs and the output, all DEVICE pointers:
 *   psi_dev    [batch][n_l][n_r] complex128 (re, im), the layout of tdse_set_state;
 *   e_now_dev  [batch] E_b(t) of the members at the time of psi (enters <z''> only), or NULL for a field-free state;
 *   out_dev    [batch][3] = {norm dr sum |f|^2, <z>, <z''> = -E_b(t) - 2 Z dr sum c_l Re(f_l* f_{l+1}) / r^2}.
 * The work is enqueued on `stream` and not synchronised.  The scratch of the two-stage reduction (per-CTA partial sums,
 * per-member counters) lives in ONE file-scope device array of 784 KiB that every GPU loading the library holds until
 * exit; it bounds the sizes: batch <= TDSE_NOALLOC_MAX_BATCH and ceil(n_r / 256) * batch * (l segments) <=
 * TDSE_NOALLOC_MAX_CTAS, else TDSE_ERR_TOO_LARGE (nothing is launched).  Calls no cudaMalloc / cudaFree and no
 * allocating library routine.  Every call on a device shares the array: calls that overlap on the GPU (different
 * streams or host threads) RACE on it; serialise them.  Ownership: nothing is retained. */
#define TDSE_NOALLOC_MAX_BATCH 4096
#define TDSE_NOALLOC_MAX_CTAS  32768
int  tdse_observables_noalloc(const void *psi_dev, int n_r, int n_l, int batch, double dr, double z_nuc,
                              const double *e_now_dev, double *out_dev, void *stream);

const char *tdse_strerror(int code);
const char *tdse_version(void);

#ifdef __cplusplus
}
#endif
#endif
