// tdse_api.cu -- host side of libtdse_b200: the C ABI of include/tdse.h, buffer ownership, the time loops
// (CUDA-graph captured blocks of steps) and the launch sequences of every propagator.
// Product path: there is no CPU fallback; without a CUDA device every compute entry point fails loudly.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <tuple>
#include <vector>

#include "tdse_kernels.cuh"
#include "tdse_taylor_rp_plan.h"
#include "tdse_tile_tma.cuh"
#include "tdse_rk45_persist.cuh"

using namespace tdse;

#define CU(call)                                                            \
    do {                                                                    \
        cudaError_t e_ = (call);                                            \
        if (e_ != cudaSuccess) {                                            \
            h->last_cuda = e_;                                              \
            return (e_ == cudaErrorMemoryAllocation) ? TDSE_ERR_ALLOC : TDSE_ERR_CUDA; \
        }                                                                   \
    } while (0)

#define RC(call)                     \
    do {                             \
        int rc_ = (call);            \
        if (rc_ != TDSE_OK) return rc_; \
    } while (0)

namespace tdse {
bool tma_available() { return tma_encode_fn() != nullptr; }
}  // namespace tdse

namespace {
enum Role { R_PSI = 0, R_G0 = 1, R_G1 = 2, R_K0 = 3 };

// Butcher tableaux (P:796-797 names them; coefficients: classic RK4 and Dormand & Prince 1980, R-C4)
const double RK4_A[4][4] = {{0, 0, 0, 0}, {0.5, 0, 0, 0}, {0, 0.5, 0, 0}, {0, 0, 1.0, 0}};
const double RK4_B[4] = {1.0 / 6, 1.0 / 3, 1.0 / 3, 1.0 / 6};
const double DP_A[7][7] = {
    {0, 0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0, 0},
    {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0}};
const double DP_B[7] = {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0};
const double DP_BH[7] = {5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40};

// All methods named at P:796 / P:813 for tdse_step_rk: b = the higher-order weights (propagated), bh = companion.
struct RkTab { int s, embedded; double c[7]; double a[7][7]; double b[7]; double bh[7]; };
const RkTab kRkTabs[6] = {
    // 0 ClassicRK4
    {4, 0, {0, 0.5, 0.5, 1.0}, {{0}, {0.5}, {0, 0.5}, {0, 0, 1.0}}, {1.0 / 6, 1.0 / 3, 1.0 / 3, 1.0 / 6}, {0}},
    // 1 DormandPrince 5(4)
    {7, 1, {0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1.0, 1.0},
     {{0}, {1.0 / 5}, {3.0 / 40, 9.0 / 40}, {44.0 / 45, -56.0 / 15, 32.0 / 9},
      {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729},
      {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656},
      {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}},
     {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0},
     {5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40}},
    // 2 Euler
    {1, 0, {0}, {{0}}, {1.0}, {0}},
    // 3 Runge-Kutta-Fehlberg 4(5)
    {6, 1, {0, 1.0 / 4, 3.0 / 8, 12.0 / 13, 1.0, 1.0 / 2},
     {{0}, {1.0 / 4}, {3.0 / 32, 9.0 / 32}, {1932.0 / 2197, -7200.0 / 2197, 7296.0 / 2197},
      {439.0 / 216, -8.0, 3680.0 / 513, -845.0 / 4104}, {-8.0 / 27, 2.0, -3544.0 / 2565, 1859.0 / 4104, -11.0 / 40}},
     {16.0 / 135, 0, 6656.0 / 12825, 28561.0 / 56430, -9.0 / 50, 2.0 / 55},
     {25.0 / 216, 0, 1408.0 / 2565, 2197.0 / 4104, -1.0 / 5, 0}},
    // 4 Cash-Karp 5(4)
    {6, 1, {0, 1.0 / 5, 3.0 / 10, 3.0 / 5, 1.0, 7.0 / 8},
     {{0}, {1.0 / 5}, {3.0 / 40, 9.0 / 40}, {3.0 / 10, -9.0 / 10, 6.0 / 5}, {-11.0 / 54, 5.0 / 2, -70.0 / 27, 35.0 / 27},
      {1631.0 / 55296, 175.0 / 512, 575.0 / 13824, 44275.0 / 110592, 253.0 / 4096}},
     {37.0 / 378, 0, 250.0 / 621, 125.0 / 594, 0, 512.0 / 1771},
     {2825.0 / 27648, 0, 18575.0 / 48384, 13525.0 / 55296, 277.0 / 14336, 1.0 / 4}},
    // 5 Kutta-Merson 4(3)
    {5, 1, {0, 1.0 / 3, 1.0 / 3, 1.0 / 2, 1.0}, {{0}, {1.0 / 3}, {1.0 / 6, 1.0 / 6}, {1.0 / 8, 0, 3.0 / 8}, {1.0 / 2, 0, -3.0 / 2, 2.0}},
     {1.0 / 6, 0, 0, 2.0 / 3, 1.0 / 6}, {1.0 / 10, 0, 3.0 / 10, 2.0 / 5, 1.0 / 5}},
};
}  // namespace

struct tdse_handle {
    tdse_grid grid{};
    GridDev gd{};
    size_t n_state = 0;                 // complex elements per state vector (B*L*N)
    cudaError_t last_cuda = cudaSuccess;
    // options
    int field_sample = 0, use_graph = 1, graph_steps = 16, taylor_block = 1, rk45_check_every = 8;
    double beta_tol = 1e-12, rk45_dt_max = 0.0;
    // device tables
    double *d_vj = nullptr, *d_cen = nullptr, *d_cl = nullptr;
    tdse_pulse *d_pulse = nullptr;
    // state vector pool; pool[psi_slot] is the state
    std::vector<double2 *> pool;
    int psi_slot = 0;
    double2 **d_bufs = nullptr;         // device copy of the role -> pointer table (RK)
    int role_slot[kRkRoles];
    // control, fields, reductions
    Ctl *d_ctl = nullptr;
    double *d_etab = nullptr; size_t etab_cap = 0;
    double *d_eapply = nullptr; std::vector<double> eapply_host; bool eapply_valid = false;
    double *d_partials = nullptr; size_t partials_cap = 0;
    unsigned int *d_counter = nullptr;
    // observables
    int n_states = 0; double *d_phi = nullptr; int *d_lstate = nullptr;
    double *d_obs_partials = nullptr; int *d_loff = nullptr, *d_slist = nullptr; unsigned int *d_obs_counters = nullptr;
    double *d_yield = nullptr;
    double *d_rp_part = nullptr; size_t rp_part_cap = 0; unsigned int *d_rp_counter = nullptr;   // fused observables
    int persist = 8;                        // option: up to this many steps per launch on small grids (0 / 1: one)
    int obs_fused = 1;                      // option: reduce the logged rows in the step kernel when it can
    double *d_rows = nullptr; size_t rows_cap = 0; long log_rows = 0; double *d_row_direct = nullptr;
    // rk45 logs
    double *d_dtlog = nullptr, *d_errlog = nullptr, *d_replay = nullptr; long log_cap = 0, replay_cap = 0;
    long last_accept = 0;
    // lanczos scalars
    int lz_K = 0; double *d_alpha = nullptr, *d_beta = nullptr, *d_nrm = nullptr, *d_inv = nullptr;
    double2 *d_coef = nullptr; int *d_m = nullptr, *d_nsub = nullptr; double2 *d_basis = nullptr;
    // graphs
    cudaStream_t cap_stream = nullptr;
    std::map<std::tuple<int, int, int, int, int, int>, cudaGraphExec_t> graphs;
    std::map<std::tuple<int, int, int, int, int, int>, long> graph_nodes;
    long launches = 0; long pending = 0; long graph_inst = 0; bool capturing = false;
    int rk45_persist = 1, rk4_persist = 1; int rk45_persist_last = 0;     // the whole adaptive run as one persistent kernel (small grids)
    void *d_rkp_ws = nullptr; size_t rkp_ws_cap = 0;
    cudaGraphExec_t rk45_loop = nullptr; long rk45_loop_nodes = 0; int rk45_loop_G = 0, rk45_use_loop = 1;   // device-driven adaptive run
    int taylor_blocked_last = 0;        // 0: one kernel per order, 3: all orders in one pass (persistent register-patch kernel)
    // blocked Taylor configuration
    RpPlan rpp{}; int n_sm = 148; int rp_variant = -1, rp_tma = -1;
    int rk4_block = 1, rk4_fused = 0;       // option: fuse the four RK4 stages; what the last tdse_step_rk4 used
    int imag = 0;                           // the running Taylor call is an imaginary-time propagation
    int apply_tma = 1;                      // tdse_apply_H: TMA-fetched tiles when n_r % 8 == 0
    int lanczos_tma = 1;                    // Lanczos pass: sources fetched by TMA when n_r % 8 == 0
    double *d_sigma = nullptr;              // passive RK error sums [batch] (tdse_step_rk)
    double *d_arun = nullptr; bool vg_quad = false;   // velocity gauge with kind-0 pulses: running A(t_n) per member
    int *d_j0 = nullptr; double cutoff = 0.0;     // centrifugal inner cut-off (tdse_set_cutoff)
    double *d_mask = nullptr; double *d_pb = nullptr;   // absorber mask [n_r] (or null), bound populations [batch]
    double *d_elog = nullptr, *d_imag_inv = nullptr; size_t elog_cap = 0; long elog_rows = 0;
};

namespace {

inline void count(tdse_handle *h) { ++h->pending; }

void free_graphs(tdse_handle *h) {
    if (h->rk45_loop) { cudaGraphExecDestroy(h->rk45_loop); h->rk45_loop = nullptr; }
    for (auto &kv : h->graphs) cudaGraphExecDestroy(kv.second);
    h->graphs.clear();
    h->graph_nodes.clear();
}

int ensure_pool(tdse_handle *h, int n) {
    while ((int)h->pool.size() < n) {
        double2 *p = nullptr;
        CU(cudaMalloc(&p, h->n_state * sizeof(double2)));
        CU(cudaMemset(p, 0, h->n_state * sizeof(double2)));
        h->pool.push_back(p);
    }
    return TDSE_OK;
}

template <class T>
int ensure_buf(tdse_handle *h, T **p, size_t *cap, size_t need) {
    if (*cap >= need && *p) return TDSE_OK;
    if (*p) { cudaDeviceSynchronize(); cudaFree(*p); *p = nullptr; free_graphs(h); }
    CU(cudaMalloc(p, need * sizeof(T)));
    CU(cudaMemset(*p, 0, need * sizeof(T)));
    *cap = need;
    return TDSE_OK;
}

dim3 tile_grid(const tdse_handle *h) {
    const int tw = Tile<3>::TW, tl = Tile<3>::TL;
    return dim3((h->grid.n_r + tw - 1) / tw, (h->grid.n_l + tl - 1) / tl, h->grid.batch);
}
int tile_ctas_per_member(const tdse_handle *h) { dim3 g = tile_grid(h); return (int)(g.x * g.y); }
long long pts_per_member(const tdse_handle *h) { return (long long)h->grid.n_l * h->grid.n_r; }
dim3 ew_grid(const tdse_handle *h) {
    return dim3((unsigned)((pts_per_member(h) + EW_CHUNK - 1) / EW_CHUNK), 1, h->grid.batch);
}

template <class Epi>
int launch_tile(tdse_handle *h, const Epi &epi, cudaStream_t s) {
    RedCtx rc{h->d_partials, h->d_counter, tile_ctas_per_member(h)};
    if (h->grid.gauge == 1) {
        if (h->grid.fd_order == 3) tile_kernel<3, Epi, true><<<tile_grid(h), 256, 0, s>>>(h->gd, epi, rc);
        else tile_kernel<5, Epi, true><<<tile_grid(h), 256, 0, s>>>(h->gd, epi, rc);
    } else if (h->grid.fd_order == 3) tile_kernel<3, Epi><<<tile_grid(h), 256, 0, s>>>(h->gd, epi, rc);
    else tile_kernel<5, Epi><<<tile_grid(h), 256, 0, s>>>(h->gd, epi, rc);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

template <class Op>
int launch_ew(tdse_handle *h, const Op &op, cudaStream_t s) {
    dim3 g = ew_grid(h);
    RedCtx rc{h->d_partials, h->d_counter, (int)g.x};
    ew_kernel<Op><<<g, EW_NT, 0, s>>>(pts_per_member(h), h->grid.batch, op, rc);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

int obs_chunks_r(const tdse_handle *h) { return (h->grid.n_r + 255) / 256; }
// l segments of the observable kernel: as few as keep about two CTAs per SM in flight
int obs_rows_per(const tdse_handle *h) {
    const int chunks = (h->grid.n_l + kObsRows - 1) / kObsRows;
    const long ctas_r = (long)obs_chunks_r(h) * h->grid.batch;
    int seg = (int)std::min<long>(chunks, std::max<long>(1, (2L * h->n_sm + ctas_r - 1) / ctas_r));
    const int per = (chunks + seg - 1) / seg;
    return per * kObsRows;
}
int obs_chunks_l(const tdse_handle *h) { return (h->grid.n_l + obs_rows_per(h) - 1) / obs_rows_per(h); }
int obs_chunks(const tdse_handle *h) { return obs_chunks_r(h) * obs_chunks_l(h); }

// Observable kernels for the state `psi`; logged row (predicated on the device step counter) or direct.
int enqueue_obs(tdse_handle *h, const double2 *psi, int step_off, int predicated, int use_direct, double t_direct,
                double *rows, cudaStream_t s) {
    const int B = h->grid.batch;
    if (obs_chunks_r(h) * ((h->grid.n_l + kObsRows - 1) / kObsRows) <= 8 && h->n_states <= 4) {   // small grid: one CTA per member
        obs_small_kernel<<<B, 256, 0, s>>>(h->gd, psi, h->d_phi, h->d_lstate, h->n_states, h->d_pulse, h->d_ctl, step_off,
                                           predicated, use_direct, t_direct, rows);
        count(h);
        CU(cudaGetLastError());
        return TDSE_OK;
    }
    obs_kernel<<<dim3(obs_chunks_r(h), B, obs_chunks_l(h)), 256, 0, s>>>(
        h->gd, psi, h->n_states, h->d_pulse, h->d_ctl, step_off, predicated, use_direct, t_direct, h->d_obs_partials,
        h->d_obs_counters, rows, obs_rows_per(h));
    count(h);
    if (h->n_states > 0) {
        pop_kernel<<<dim3(h->grid.n_l, B), 256, 0, s>>>(h->gd, psi, h->d_phi, h->d_loff, h->d_slist, h->n_states, h->d_ctl,
                                                         step_off, predicated, use_direct, rows);
        count(h);
    }
    CU(cudaGetLastError());
    return TDSE_OK;
}

int ensure_rows(tdse_handle *h, long nsteps, int obs_every) {
    const size_t W = 3 + h->n_states;
    size_t need = (size_t)h->grid.batch * W;
    if (obs_every > 0) need *= (size_t)std::max(1L, nsteps / obs_every);
    return ensure_buf(h, &h->d_rows, &h->rows_cap, need);
}

int init_ctl(tdse_handle *h, const CtlInit &v, cudaStream_t s) {
    ctl_init_kernel<<<1, 32, 0, s>>>(h->d_ctl, v);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

// ---- blocks of steps --------------------------------------------------------------------------------
// Each enqueue_* function enqueues `n` consecutive steps (reading t0, dt and the step counter from the device
// control block) and ends by advancing the counter; it is either captured into a graph or run eagerly.

// absorbing boundary after a step whose kernels did not apply it themselves
int enqueue_mask(tdse_handle *h, double2 *psi, cudaStream_t s) {
    if (!h->d_mask) return TDSE_OK;
    OpMask m{};
    m.psi = psi; m.mask = h->d_mask; m.n_r = h->grid.n_r;
    return launch_ew(h, m, s);
}

// imaginary time: E and 1/||psi|| of the step just taken, then psi *= 1/||psi||
int enqueue_imag_norm(tdse_handle *h, double2 *psi, int step_off, cudaStream_t s) {
    OpImagNorm on{};
    on.psi = psi; on.ctl = h->d_ctl; on.step_off = step_off; on.batch = h->grid.batch; on.dr = h->grid.dr;
    on.elog = h->d_elog; on.inv = h->d_imag_inv;
    RC(launch_ew(h, on, s));
    OpScaleMember sc{};
    sc.psi = psi; sc.inv = h->d_imag_inv;
    RC(launch_ew(h, sc, s));
    return TDSE_OK;
}

// the observable row of step `step_off` reduced inside the register-patch kernel (tdse_taylor_rp.cuh, OBS)
// Measured (profiles/r02_README.md): on grids of many CTAs the fused reduction costs more than it saves (one more
// barrier round per item, and a fence + ticket + last-CTA tail of 6-8 us per logged step against a 9 us pass of
// obs_kernel over an L2-resident CFG3 state), so obs_fused = 1 (auto) uses it for grids of at most 16 CTAs and
// obs_fused = 2 forces it wherever the kernel can do it.
bool obs_fused_wanted(const tdse_handle *h) {
    if (!h->obs_fused || h->d_j0 || !rp_obs_capable(h->rpp, h->grid, h->n_states)) return false;   // (no fused rows with a cut-off)
    return h->obs_fused == 2 || h->rpp.persist > 1 || (long)h->rpp.n_items * h->rpp.cl <= 16;
}
bool obs_fused_now(const tdse_handle *h, int obs) { return obs && h->d_rp_part && obs_fused_wanted(h); }
RpObs make_rp_obs(const tdse_handle *h, int step_off) {
    RpObs o{};
    o.ctl = h->d_ctl; o.pulse = h->d_pulse; o.phi = h->d_phi; o.l_of_state = h->d_lstate; o.n_states = h->n_states;
    o.step_off = step_off; o.partials = h->d_rp_part; o.counter = h->d_rp_counter; o.rows = h->d_rows;
    return o;
}
int ensure_rp_obs(tdse_handle *h, int obs_every) {
    if (obs_every <= 0 || !obs_fused_wanted(h)) return TDSE_OK;
    RC(ensure_buf(h, &h->d_rp_part, &h->rp_part_cap, rp_obs_partials(h->rpp)));
    if (!h->d_rp_counter) {
        CU(cudaMalloc(&h->d_rp_counter, sizeof(unsigned int)));
        CU(cudaMemset(h->d_rp_counter, 0, sizeof(unsigned int)));
    }
    return TDSE_OK;
}

// field tables of a block of n steps: e_tab[(step*n_stage + stage)*B + b].  mode 0: Taylor / Lanczos (one value per step),
// 1: classic RK4 stage times, 2: the stage times `cs` of any tableau.  Velocity gauge with pulses given by their field:
// the running quadrature (field_table_quad_kernel), else the closed-form kernels.
int enqueue_field_table(tdse_handle *h, int n, int mode, int n_stage, const StageTimes &cs, cudaStream_t s) {
    const int B = h->grid.batch;
    if (h->vg_quad) {
        StageTimes c = cs;
        if (mode == 1) { c.c[0] = 0.0; c.c[1] = 0.5; c.c[2] = 0.5; c.c[3] = 1.0; }
        field_table_quad_kernel<<<(B + 63) / 64, 64, 0, s>>>(h->d_ctl, h->d_pulse, B, n, mode == 0 ? 1 : n_stage, c, mode == 0 ? 1 : 0,
                                                             h->d_etab, h->d_arun);
    } else if (mode == 2) {
        field_table_rk_kernel<<<(n * n_stage * B + 255) / 256, 256, 0, s>>>(h->d_ctl, h->d_pulse, B, n, n_stage, cs, h->d_etab, h->gd.gauge);
    } else {
        field_table_kernel<<<(n * (mode == 1 ? 4 : 1) * B + 255) / 256, 256, 0, s>>>(h->d_ctl, h->d_pulse, B, n, mode, h->d_etab, h->gd.gauge);
    }
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

int enqueue_taylor_block(tdse_handle *h, int order, int n, int obs, cudaStream_t s) {
    const int B = h->grid.batch;
    if (h->imag) {
        CU(cudaMemsetAsync(h->d_etab, 0, sizeof(double) * (size_t)n * B, s));       // no field
    } else {
        RC(enqueue_field_table(h, n, 0, 1, StageTimes{}, s));
    }
    double2 *psi = h->pool[h->psi_slot];
    // scratch: three further pool slots
    int sl[3], c = 0;
    for (int i = 0; c < 3; ++i) if (i != h->psi_slot) sl[c++] = i;
    double2 *ta = h->pool[sl[0]], *tb = h->pool[sl[1]], *acc = h->pool[sl[2]];
    if (h->taylor_blocked_last && h->rpp.persist) {
        // temporal blocking across steps: launches of up to rpp.persist steps, psi in registers in between
        const bool fused = obs_fused_now(h, obs);
        if (obs && !fused) return TDSE_ERR_UNSUPPORTED;         // (step_taylor_impl plans persist only when the rows can be fused)
        double2 *src = psi, *dst = acc;
        for (int i = 0; i < n; i += h->rpp.persist) {
            const int k = std::min(h->rpp.persist, n - i);
            const RpObs ro = make_rp_obs(h, i);
            RC(launch_taylor_rp(h->gd, h->rpp, src, dst, h->d_etab + (size_t)i * B, &h->d_ctl->dt, order, s, fused ? &ro : nullptr, k));
            count(h);
            std::swap(src, dst);
        }
        if (src != psi) {                                       // odd number of launches: bring the state back
            OpCopy cp{}; cp.dst = psi; cp.src = acc;
            RC(launch_ew(h, cp, s));
        }
        ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, n);
        count(h);
        CU(cudaGetLastError());
        return TDSE_OK;
    }
    for (int i = 0; i < n; ++i) {
        const double *ef = h->d_etab + (size_t)i * B;
        if (h->taylor_blocked_last) {
            // ping-pong psi <-> acc: even steps read psi, odd steps read acc (n is even inside graphs)
            double2 *src = (i & 1) ? acc : psi, *dst = (i & 1) ? psi : acc;
            const bool fused = !h->imag && obs_fused_now(h, obs);
            const RpObs ro = make_rp_obs(h, i);
            RC(launch_taylor_rp(h->gd, h->rpp, src, dst, ef, &h->d_ctl->dt, order, s, fused ? &ro : nullptr));
            count(h);
            if (h->imag) RC(enqueue_imag_norm(h, dst, i, s));
            if (obs && !fused) RC(enqueue_obs(h, dst, i, 1, 0, 0.0, h->d_rows, s));
            continue;
        }
        for (int k = 1; k <= order; ++k) {
            EpiTaylor e{};
            e.in = (k == 1) ? psi : ((k & 1) ? tb : ta);       // term_{k-1}: k-1 odd -> ta, even -> tb
            e.ef = ef; e.dtp = &h->d_ctl->dt; e.k = k; e.first = (k == 1); e.write_term = (k < order); e.imag = h->imag;
            e.term_out = (k & 1) ? ta : tb;
            e.acc_in = acc;
            e.acc_out = (k == order && order > 1) ? psi : acc;  // the last order reads acc point-wise: write psi in place
            RC(launch_tile(h, e, s));
        }
        if (order == 1) {
            OpCopy cp{}; cp.dst = psi; cp.src = acc;
            RC(launch_ew(h, cp, s));
        }
        if (h->imag) RC(enqueue_imag_norm(h, psi, i, s));
        else RC(enqueue_mask(h, psi, s));
        if (obs) RC(enqueue_obs(h, psi, i, 1, 0, 0.0, h->d_rows, s));
    }
    if (h->taylor_blocked_last && (n & 1)) {   // odd eager remainder: bring the state back into the psi slot
        OpCopy cp{}; cp.dst = psi; cp.src = acc;
        RC(launch_ew(h, cp, s));
    }
    ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, n);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

void rk_roles(tdse_handle *h) {
    // role r lives in pool slot: PSI -> psi_slot, the others in increasing slot order
    int c = 0;
    for (int r = 0; r < kRkRoles; ++r) {
        if (r == R_PSI) { h->role_slot[r] = h->psi_slot; continue; }
        if (c == h->psi_slot) ++c;
        h->role_slot[r] = c++;
    }
}

int upload_bufs(tdse_handle *h, int n_roles, cudaStream_t s) {
    std::vector<double2 *> tab(kRkRoles, nullptr);
    for (int r = 0; r < n_roles; ++r) tab[r] = h->pool[h->role_slot[r]];
    CU(cudaMemcpyAsync(h->d_bufs, tab.data(), sizeof(double2 *) * kRkRoles, cudaMemcpyHostToDevice, s));
    CU(cudaStreamSynchronize(s));   // tab is a stack object
    return TDSE_OK;
}

template <class E>
void fill_rk_common(tdse_handle *h, E &e, int stage, const double *ef, const double *hptr) {
    e.ctl = h->d_ctl; e.bufs = h->d_bufs; e.ef = ef; e.hptr = hptr; e.stage = stage;
    e.psi_role = R_PSI;
    for (int j = 0; j < 7; ++j) { e.k_role[j] = -1; e.a_next[j] = 0.0; e.d_err[j] = 0.0; }
    e.check_done = 0; e.dt_log = h->d_dtlog; e.err_log = h->d_errlog;
    e.passive = 0; e.sigma_acc = nullptr; e.inv_m = 0.0;
}

int enqueue_rk4_block(tdse_handle *h, int n, int obs, cudaStream_t s) {
    const int B = h->grid.batch;
    RC(enqueue_field_table(h, n, 1, 4, StageTimes{}, s));
    double2 *psi = h->pool[h->psi_slot];
    if (h->rk4_fused) {
        // all four stages in one pass over HBM (taylor_rp_kernel in RK mode); ping-pong psi <-> scratch
        double2 *alt = h->pool[h->psi_slot == 0 ? 1 : 0];
        for (int i = 0; i < n; ++i) {
            double2 *src = (i & 1) ? alt : psi, *dst = (i & 1) ? psi : alt;
            const bool fused = obs_fused_now(h, obs);
            const RpObs ro = make_rp_obs(h, i);
            RC(launch_taylor_rp(h->gd, h->rpp, src, dst, h->d_etab + (size_t)i * 4 * B, &h->d_ctl->dt, 4, s, fused ? &ro : nullptr));
            count(h);
            if (obs && !fused) RC(enqueue_obs(h, dst, i, 1, 0, 0.0, h->d_rows, s));
        }
        if (n & 1) {   // odd eager remainder: bring the state back into the psi slot
            OpCopy cp{}; cp.dst = psi; cp.src = alt;
            RC(launch_ew(h, cp, s));
        }
        ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, n);
        count(h);
        CU(cudaGetLastError());
        return TDSE_OK;
    }
    for (int i = 0; i < n; ++i) {
        for (int st = 0; st < 4; ++st) {
            EpiRK<false> e{};
            fill_rk_common(h, e, st, h->d_etab + ((size_t)i * 4 + st) * B, &h->d_ctl->dt);
            e.in_role = (st == 0) ? R_PSI : ((st & 1) ? R_G1 : R_G0);      // stage st reads what stage st-1 wrote
            for (int j = 0; j < 3; ++j) e.k_role[j] = R_K0 + j;
            if (st < 3) {
                e.store_k = 1;
                e.out_role = ((st + 1) & 1) ? R_G1 : R_G0;
                for (int j = 0; j <= st; ++j) e.a_next[j] = RK4_A[st + 1][j];
            } else {
                e.store_k = 0;
                e.out_role = R_PSI;                                         // psi is read point-wise only: in place
                for (int j = 0; j < 4; ++j) e.a_next[j] = RK4_B[j];
            }
            RC(launch_tile(h, e, s));
        }
        RC(enqueue_mask(h, psi, s));
        if (obs) RC(enqueue_obs(h, psi, i, 1, 0, 0.0, h->d_rows, s));
    }
    ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, n);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

// Dormand-Prince stages [first_stage, 7) of `n` attempted steps; every kernel exits at once when ctl->done.
// Fixed-step propagation with any tableau of kRkTabs through the stage loop of P:469-478: stage st reads the stage
// vector its predecessor formed, stores k_st and forms g_{st+1} = psi + h sum_j a_{st+1,j} k_j in its epilogue; the
// last stage writes psi + h sum_j b_j k_j over psi (read point-wise only) and, for an embedded pair, reduces
// |Delta|^2 for the passive error sum.
int enqueue_rk_generic_block(tdse_handle *h, int method, int n, int obs, cudaStream_t s) {
    const int B = h->grid.batch;
    const RkTab &tb = kRkTabs[method];
    StageTimes cs{};
    for (int i = 0; i < 7; ++i) cs.c[i] = tb.c[i];
    RC(enqueue_field_table(h, n, 2, tb.s, cs, s));
    double2 *psi = h->pool[h->psi_slot];
    for (int i = 0; i < n; ++i) {
        for (int st = 0; st < tb.s; ++st) {
            const double *ef = h->d_etab + ((size_t)i * tb.s + st) * B;
            const bool last = (st == tb.s - 1);
            auto fill = [&](auto &e) {
                fill_rk_common(h, e, st, ef, &h->d_ctl->dt);
                e.in_role = (st == 0) ? R_PSI : ((st & 1) ? R_G1 : R_G0);
                for (int j = 0; j < 7; ++j) e.k_role[j] = R_K0 + j;
                if (!last) {
                    e.store_k = 1;
                    e.out_role = ((st + 1) & 1) ? R_G1 : R_G0;
                    for (int j = 0; j <= st; ++j) e.a_next[j] = tb.a[st + 1][j];
                } else {
                    e.store_k = 0;
                    // a one-stage method reads psi through the tile (halo): it must not be overwritten in place
                    e.out_role = (tb.s == 1) ? R_G0 : R_PSI;
                    for (int j = 0; j < tb.s; ++j) e.a_next[j] = tb.b[j];
                }
            };
            if (last && tb.embedded) {
                EpiRK<true> e{};
                fill(e);
                for (int j = 0; j < tb.s; ++j) e.d_err[j] = tb.b[j] - tb.bh[j];
                e.passive = 1; e.sigma_acc = h->d_sigma; e.inv_m = 1.0 / (double)pts_per_member(h);
                RC(launch_tile(h, e, s));
            } else {
                EpiRK<false> e{};
                fill(e);
                RC(launch_tile(h, e, s));
            }
        }
        if (tb.s == 1) {
            OpCopy cp{}; cp.dst = psi; cp.src = h->pool[h->role_slot[R_G0]];
            RC(launch_ew(h, cp, s));
        }
        RC(enqueue_mask(h, psi, s));
        if (obs) RC(enqueue_obs(h, psi, i, 1, 0, 0.0, h->d_rows, s));
    }
    ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, n);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

int enqueue_rk45_block(tdse_handle *h, int n, int first_stage, cudaStream_t s) {
    const int B = h->grid.batch;
    for (int i = 0; i < n; ++i) {
        rk45_begin_kernel<<<1, 256, 0, s>>>(h->d_ctl, h->d_pulse, B, h->d_replay, h->d_etab, h->gd.gauge);
        count(h);
        for (int st = (i == 0 ? first_stage : 1); st < 7; ++st) {
            const double *ef = h->d_etab + (size_t)st * B;
            if (st == 0) {
                // only the very first attempted step: k_1 = -i H(t) psi (afterwards FSAL supplies it); g_2 is
                // formed by stage 1 while loading its tile, because h changes between attempts
                EpiRK<false> e{};
                fill_rk_common(h, e, st, ef, &h->d_ctl->h);
                e.check_done = 1; e.in_role = R_PSI; e.k_role[0] = R_K0; e.store_k = 1; e.out_role = -1;
                RC(launch_tile(h, e, s));
            } else if (st == 1) {
                EpiRK<false, true> e{};
                fill_rk_common(h, e, st, ef, &h->d_ctl->h);
                e.check_done = 1;
                e.in_role = R_PSI; e.in2_role = R_K0; e.in2_a = DP_A[1][0];     // g_2 = psi + h a_21 k_1
                for (int j = 0; j < 7; ++j) e.k_role[j] = R_K0 + j;
                e.store_k = 1;
                e.out_role = R_G0;
                for (int j = 0; j <= st; ++j) e.a_next[j] = DP_A[st + 1][j];
                RC(launch_tile(h, e, s));
            } else if (st < 6) {
                EpiRK<false> e{};
                fill_rk_common(h, e, st, ef, &h->d_ctl->h);
                e.check_done = 1;
                e.in_role = (st == 0) ? R_PSI : ((st & 1) ? R_G1 : R_G0);
                for (int j = 0; j < 7; ++j) e.k_role[j] = R_K0 + j;
                e.store_k = 1;
                e.out_role = ((st + 1) & 1) ? R_G1 : R_G0;
                for (int j = 0; j <= st; ++j) e.a_next[j] = DP_A[st + 1][j];
                RC(launch_tile(h, e, s));
            } else {
                EpiRK<true> e{};
                fill_rk_common(h, e, st, ef, &h->d_ctl->h);
                e.check_done = 1;
                e.in_role = R_G0;                                           // stage 5 wrote psi_new = g_7 into G0
                for (int j = 0; j < 7; ++j) e.k_role[j] = R_K0 + j;
                e.store_k = 1;
                e.out_role = -1;
                for (int j = 0; j < 7; ++j) e.d_err[j] = DP_B[j] - DP_BH[j];
                RC(launch_tile(h, e, s));
            }
        }
    }
    CU(cudaGetLastError());
    return TDSE_OK;
}

// Lanczos step: per Krylov vector one tile kernel (matvec + alpha) and one element-wise kernel
// (orthogonalise + beta); then the one-warp exponential and the back-expansion.  The normalisation of q_{p+1}
// is folded into the next tile load.  w ping-pongs between two buffers because a tile source must not be
// written by the same kernel (halo race).
int enqueue_lanczos_block(tdse_handle *h, int K, int order, int n, int obs, cudaStream_t s) {
    const int B = h->grid.batch;
    RC(enqueue_field_table(h, n, 0, 1, StageTimes{}, s));
    double2 *psi = h->pool[h->psi_slot];
    double2 *wbuf[2]; int c = 0;
    for (int i = 0; c < 2; ++i) if (i != h->psi_slot) wbuf[c++] = h->pool[i];
    double2 *basis = h->d_basis;
    for (int i = 0; i < n; ++i) {
        const double *ef = h->d_etab + (size_t)i * B;
        // one fused pass per Krylov vector: v_p formed on load, g_p = H v_p, <v_p|g_p> and ||v_p||^2 reduced
        for (int p = 0; p < K; ++p) {
            EpiLanczosF a{};
            a.psi = psi; a.g_in = wbuf[(p + 1) & 1];
            a.v1 = (p >= 1) ? basis + (size_t)(p - 1) * h->n_state : nullptr;
            a.v2 = (p >= 2) ? basis + (size_t)(p - 2) * h->n_state : nullptr;
            a.v_out = basis + (size_t)p * h->n_state;
            a.g_out = (p < K - 1) ? wbuf[p & 1] : nullptr;
            a.ef = ef; a.alpha = h->d_alpha; a.beta = h->d_beta; a.sc = h->d_inv; a.nrm = h->d_nrm; a.m_used = h->d_m;
            a.p = p; a.K = K; a.tol = h->beta_tol;
            if (h->lanczos_tma && (h->grid.n_r & 7) == 0 && tma_available()) {
                // sources fetched by TMA (tdse_tile_tma.cuh); the maps are copied by value into the launch
                const int tiles_r = (h->grid.n_r + kTtTW - 1) / kTtTW, tiles_l = (h->grid.n_l + kTtTL - 1) / kTtTL;
                const int n_items = tiles_r * tiles_l * B;
                CUtensorMap tm[3] = {};
                bool ok = true;
                for (int i = 0; i < 3 && ok; ++i) {
                    const double2 *src = (i == 0) ? (p == 0 ? psi : a.g_in) : (i == 1 ? a.v1 : a.v2);
                    if (!src) continue;
                    ok = tile_tensor_map(&tm[i], src, h->grid.n_r, h->grid.n_l, B);
                }
                if (ok) {
                    static DeviceOnce attr_once;
                    if (attr_once.first()) {
                        CU(cudaFuncSetAttribute(tile_tma3_kernel<3, EpiLanczosF>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTt3Smem));
                        CU(cudaFuncSetAttribute(tile_tma3_kernel<5, EpiLanczosF>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTt3Smem));
                        CU(cudaFuncSetAttribute(tile_tma3_kernel<3, EpiLanczosF, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTt3Smem));
                        CU(cudaFuncSetAttribute(tile_tma3_kernel<5, EpiLanczosF, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTt3Smem));
                    }
                    RedCtx rc{h->d_partials, h->d_counter, tiles_r * tiles_l};
                    const int grid = std::min(n_items, h->n_sm * 2);
                    if (h->grid.gauge == 1) {
                        if (h->grid.fd_order == 3)
                            tile_tma3_kernel<3, EpiLanczosF, true><<<grid, 256, kTt3Smem, s>>>(h->gd, a, rc, tm[0], tm[1], tm[2], tiles_r, tiles_l, n_items);
                        else
                            tile_tma3_kernel<5, EpiLanczosF, true><<<grid, 256, kTt3Smem, s>>>(h->gd, a, rc, tm[0], tm[1], tm[2], tiles_r, tiles_l, n_items);
                    } else if (h->grid.fd_order == 3)
                        tile_tma3_kernel<3, EpiLanczosF><<<grid, 256, kTt3Smem, s>>>(h->gd, a, rc, tm[0], tm[1], tm[2], tiles_r, tiles_l, n_items);
                    else
                        tile_tma3_kernel<5, EpiLanczosF><<<grid, 256, kTt3Smem, s>>>(h->gd, a, rc, tm[0], tm[1], tm[2], tiles_r, tiles_l, n_items);
                    count(h);
                    CU(cudaGetLastError());
                    continue;
                }
            }
            RC(launch_tile(h, a, s));
        }
        small_exp_kernel<<<B, 32, 0, s>>>(h->d_alpha, h->d_beta, h->d_m, &h->d_ctl->dt, K, order, h->d_coef, h->d_nsub);
        count(h);
        OpCombine oc{};
        oc.psi = psi; oc.q = basis; oc.q_stride = h->n_state; oc.coef = h->d_coef; oc.nrm = h->d_nrm; oc.sc = h->d_inv;
        oc.m_used = h->d_m; oc.K = K;
        RC(launch_ew(h, oc, s));
        RC(enqueue_mask(h, psi, s));
        if (obs) RC(enqueue_obs(h, psi, i, 1, 0, 0.0, h->d_rows, s));
    }
    ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, n);
    count(h);
    CU(cudaGetLastError());
    return TDSE_OK;
}

// The adaptive run as ONE graph launch: a WHILE node whose body is G attempted Dormand-Prince steps followed by the
// condition kernel (go on while the device controller has not set `done`).  No host poll inside the run (the paper
// enqueues kernels asynchronously to keep the device busy; its kernel boundaries exist only for global
// synchronisation, P:484 -- the accept / reject decision is taken by the last CTA of the last stage on the device).
int build_rk45_loop(tdse_handle *h, int G) {
    if (h->rk45_loop && h->rk45_loop_G == G) return TDSE_OK;
    if (h->rk45_loop) { cudaGraphExecDestroy(h->rk45_loop); h->rk45_loop = nullptr; }
    cudaGraph_t g = nullptr;
    CU(cudaGraphCreate(&g, 0));
    auto fail = [&](int rc) { cudaGraphDestroy(g); cudaGetLastError(); return rc; };
    cudaGraphConditionalHandle handle;
    if (cudaGraphConditionalHandleCreate(&handle, g, 1, cudaGraphCondAssignDefault) != cudaSuccess) return fail(TDSE_ERR_CUDA);
    cudaGraphNodeParams np{};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    if (cudaGraphAddNode(&node, g, nullptr, 0, &np) != cudaSuccess) return fail(TDSE_ERR_CUDA);
    cudaGraph_t body = np.conditional.phGraph_out[0];
    if (cudaStreamBeginCaptureToGraph(h->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed) != cudaSuccess)
        return fail(TDSE_ERR_CUDA);
    h->pending = 0;
    int rc = enqueue_rk45_block(h, G, 1, h->cap_stream);
    rk45_cond_kernel<<<1, 32, 0, h->cap_stream>>>(h->d_ctl, handle);
    ++h->pending;
    cudaGraph_t captured = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(h->cap_stream, &captured);
    if (rc != TDSE_OK || ce != cudaSuccess) return fail(rc != TDSE_OK ? rc : TDSE_ERR_CUDA);
    cudaGraphExec_t ex = nullptr;
    if (cudaGraphInstantiate(&ex, g, 0) != cudaSuccess) return fail(TDSE_ERR_CUDA);
    cudaGraphDestroy(g);
    h->rk45_loop = ex; h->rk45_loop_G = G; h->rk45_loop_nodes = h->pending;
    ++h->graph_inst;
    return TDSE_OK;
}

// ---- graph-captured time loop (row a7; NS: "the time loop is captured in a CUDA graph") ------------------
}  // namespace
namespace tdse { int launch_rk45_persist(const RkpArgs &a, const RkpPlan &p, cudaStream_t s); bool rk45_persist_fits(int fd, int gauge, const RkpPlan &p); }
namespace {
enum Kind { KIND_TAYLOR = 1, KIND_RK4 = 2, KIND_LANCZOS = 3, KIND_RK45 = 4, KIND_RKGEN = 5 };

int enqueue_block(tdse_handle *h, int kind, int p1, int p2, int n, int obs, cudaStream_t s) {
    switch (kind) {
        case KIND_TAYLOR: return enqueue_taylor_block(h, p1, n, obs, s);
        case KIND_RK4: return enqueue_rk4_block(h, n, obs, s);
        case KIND_LANCZOS: return enqueue_lanczos_block(h, p1, p2, n, obs, s);
        case KIND_RK45: return enqueue_rk45_block(h, n, 1, s);
        case KIND_RKGEN: return enqueue_rk_generic_block(h, p1, n, obs, s);
    }
    return TDSE_ERR_ARG;
}

// Run `nblocks` blocks of `n` steps each on `stream`, through a cached graph when enabled.
int run_blocks(tdse_handle *h, int kind, int p1, int p2, int n, int obs, long nblocks, cudaStream_t stream) {
    if (nblocks <= 0) return TDSE_OK;
    if (!h->use_graph) {
        for (long i = 0; i < nblocks; ++i) {
            h->pending = 0;
            RC(enqueue_block(h, kind, p1, p2, n, obs, stream));
            h->launches += h->pending;
        }
        return TDSE_OK;
    }
    const auto key = std::make_tuple(kind, p1, p2, n, obs + 2 * h->taylor_blocked_last + 256 * (h->rpp.variant + 1) + 8192 * h->rpp.tma + 16384 * h->rk4_fused + 32768 * h->imag + 65536 * (int)obs_fused_now(h, obs) + 131072 * h->rpp.persist + 16777216 * (h->rpp.H & 127), h->psi_slot);
    auto it = h->graphs.find(key);
    if (it == h->graphs.end()) {
        cudaGraph_t g = nullptr;
        CU(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
        h->pending = 0;
        const int rc = enqueue_block(h, kind, p1, p2, n, obs, h->cap_stream);
        const cudaError_t ce = cudaStreamEndCapture(h->cap_stream, &g);
        if (rc != TDSE_OK) { if (g) cudaGraphDestroy(g); return rc; }
        CU(ce);
        cudaGraphExec_t ex = nullptr;
        const cudaError_t ie = cudaGraphInstantiate(&ex, g, 0);
        cudaGraphDestroy(g);
        CU(ie);
        h->graph_nodes[key] = h->pending;
        ++h->graph_inst;
        it = h->graphs.emplace(key, ex).first;
    }
    const long nodes = h->graph_nodes[key];
    for (long i = 0; i < nblocks; ++i) {
        CU(cudaGraphLaunch(it->second, stream));
        h->launches += nodes;
    }
    return TDSE_OK;
}

int run_fixed(tdse_handle *h, int kind, int p1, int p2, double t0, double dt, long nsteps, int obs_every,
              cudaStream_t stream) {
    const int B = h->grid.batch;
    int G = std::max(1, h->graph_steps);
    // small grids whose launches take several steps: a graph of four times as many steps (the field-table and counter
    // kernels and the graph launch itself weigh 15 % of a 16-step block there)
    if (kind == KIND_TAYLOR && h->taylor_blocked_last && h->rpp.persist > 1) G *= 4;
    if (h->taylor_blocked_last) G = (G + 1) & ~1;       // ping-pong needs an even block
    RC(ensure_buf(h, &h->d_etab, &h->etab_cap, (size_t)G * 7 * B));
    RC(ensure_rows(h, nsteps, obs_every));
    if (h->taylor_blocked_last) RC(ensure_rp_obs(h, obs_every));
    CtlInit v{};
    v.t0 = t0; v.dt = dt; v.obs_every = obs_every; v.field_sample = h->field_sample;
    h->pending = 0;
    RC(init_ctl(h, v, stream));
    if (h->vg_quad) {                   // A(t0) of the pulses given by their field (reading R-V4)
        vecpot_init_kernel<<<B, 256, 0, stream>>>(h->d_ctl, h->d_pulse, h->d_arun);
        count(h);
        CU(cudaGetLastError());
    }
    h->launches += h->pending;
    const int obs = obs_every > 0 ? 1 : 0;
    RC(run_blocks(h, kind, p1, p2, G, obs, nsteps / G, stream));
    const int rem = (int)(nsteps % G);
    if (rem) {
        const int ug = h->use_graph; h->use_graph = 0;
        const int rc = run_blocks(h, kind, p1, p2, rem, obs, 1, stream);
        h->use_graph = ug;
        RC(rc);
    }
    h->log_rows = obs ? nsteps / obs_every : 0;
    return TDSE_OK;
}

// ---- the persistent on-chip Runge-Kutta kernel (tdse_rk45_persist.cuh) -------------------------------------------------
// its plan on the current device (ok = 0: the grid does not fit on chip, or the device cannot hold the grid at once)
RkpPlan rkp_plan_for(tdse_handle *h) {
    RkpPlan pp{};
    int dev = 0, max_smem = 0, coop = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop)
        pp = rkp_plan(h->grid, h->n_sm, std::min(max_smem - 2048, kRkpMaxSmem));
    if (pp.ok && !rk45_persist_fits(h->grid.fd_order, h->grid.gauge, pp)) pp.ok = 0;     // (a partitioned or shared device)
    return pp;
}

// workspace of the packets (cleared: no packet of an earlier launch may carry a sequence number of this one) and the
// arguments every mode shares
int rkp_prepare(tdse_handle *h, const RkpPlan &pp, RkpArgs &a, cudaStream_t s) {
    const size_t part_off = (pp.halo_bytes + 255) & ~(size_t)255, ws_bytes = part_off + pp.part_bytes;
    if (h->rkp_ws_cap < ws_bytes) {
        CU(cudaStreamSynchronize(s));
        if (h->d_rkp_ws) cudaFree(h->d_rkp_ws);
        h->d_rkp_ws = nullptr; h->rkp_ws_cap = 0;
        CU(cudaMalloc(&h->d_rkp_ws, ws_bytes));
        h->rkp_ws_cap = ws_bytes;
    }
    char *ws = (char *)h->d_rkp_ws;
    a = RkpArgs{};
    a.g = h->gd; a.psi = h->pool[h->psi_slot]; a.ctl = h->d_ctl; a.pulse = h->d_pulse; a.replay = h->d_replay;
    a.dt_log = h->d_dtlog; a.err_log = h->d_errlog;
    a.halo = (unsigned long long *)ws; a.part = (unsigned long long *)(ws + part_off);
    a.G = pp.G; a.Wc = pp.Wc; a.R = pp.R; a.pitch = pp.pitch;
    CU(cudaMemsetAsync(ws, 0, ws_bytes, s));
    return TDSE_OK;
}

bool grid_valid(const tdse_grid *g) {
    return g && g->n_r >= 1 && g->n_l >= 1 && g->dr > 0.0 && g->batch >= 1 && g->batch <= 65535 &&
           (long long)g->n_r * g->n_l * g->batch < (1LL << 31) * 8;
}

}  // namespace

// =========================================================================================================
extern "C" {

const char *tdse_version(void) { return "tdse_b200 0.1 (sm_100a)"; }

const char *tdse_strerror(int code) {
    switch (code) {
        case TDSE_OK: return "ok";
        case TDSE_ERR_ARG: return "invalid argument";
        case TDSE_ERR_ALLOC: return "allocation failed";
        case TDSE_ERR_CUDA: return "CUDA error (no device or launch failure)";
        case TDSE_ERR_NONFINITE: return "non-finite norm logged (unstable step size?)";
        case TDSE_ERR_UNSUPPORTED: return "unsupported configuration";
        case TDSE_ERR_TOO_LARGE: return "size beyond the fixed scratch array of the no-allocation entry point";
    }
    return "unknown error";
}

int tdse_create(const tdse_grid *grid, tdse_handle **out) {
    if (!out) return TDSE_ERR_ARG;
    *out = nullptr;
    if (!grid_valid(grid)) return TDSE_ERR_ARG;
    if ((grid->gauge != 0 && grid->gauge != 1) || (grid->fd_order != 3 && grid->fd_order != 5)) return TDSE_ERR_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return TDSE_ERR_CUDA; }
    tdse_handle *h = new (std::nothrow) tdse_handle();
    if (!h) return TDSE_ERR_ALLOC;
    h->grid = *grid;
    {
        int dev = 0, n_sm = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n_sm > 0)
            h->n_sm = n_sm;
    }
    if ((grid->fd_order == 3 ? rp_init_fd3() : rp_init_fd5()) != TDSE_OK) { delete h; return TDSE_ERR_CUDA; }
    const int N = grid->n_r, L = grid->n_l, B = grid->batch;
    h->n_state = (size_t)N * L * B;
    auto fail = [&](int rc) { tdse_destroy(h); return rc; };
    auto body = [&]() -> int {
        // tables of the diagonal of h_l (Eq. 7) and the coupling (Eq. 9)
        std::vector<double> vj(N), cen(N), cl(L);
        const double dr2 = grid->dr * grid->dr;
        const double kd = (grid->fd_order == 3) ? 1.0 / dr2 : 30.0 / (24.0 * dr2);
        for (int j = 0; j < N; ++j) {
            const double r = (j + 1) * grid->dr;
            vj[j] = kd - grid->z_nuc / r;
            cen[j] = 1.0 / (2.0 * r * r);
        }
        for (int l = 0; l < L; ++l) cl[l] = (l + 1) / std::sqrt((2.0 * l + 1.0) * (2.0 * l + 3.0));
        CU(cudaMalloc(&h->d_vj, sizeof(double) * N));
        CU(cudaMalloc(&h->d_cen, sizeof(double) * N));
        CU(cudaMalloc(&h->d_cl, sizeof(double) * L));
        CU(cudaMemcpy(h->d_vj, vj.data(), sizeof(double) * N, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(h->d_cen, cen.data(), sizeof(double) * N, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(h->d_cl, cl.data(), sizeof(double) * L, cudaMemcpyHostToDevice));
        GridDev &g = h->gd;
        g.n_r = N; g.n_l = L; g.batch = B; g.fd = grid->fd_order; g.gauge = grid->gauge; g.dr = grid->dr; g.z = grid->z_nuc;
        if (grid->fd_order == 3) { g.c1 = -0.5 / dr2; g.c2 = 0.0; }
        else { g.c1 = -16.0 / (24.0 * dr2); g.c2 = 1.0 / (24.0 * dr2); }
        g.vj = h->d_vj; g.cen = h->d_cen; g.cl = h->d_cl;
        CU(cudaMalloc(&h->d_pulse, sizeof(tdse_pulse) * B));
        CU(cudaMemset(h->d_pulse, 0, sizeof(tdse_pulse) * B));
        CU(cudaMalloc(&h->d_ctl, sizeof(Ctl)));
        CU(cudaMemset(h->d_ctl, 0, sizeof(Ctl)));
        CU(cudaMalloc(&h->d_bufs, sizeof(double2 *) * kRkRoles));
        CU(cudaMalloc(&h->d_counter, sizeof(unsigned int)));
        CU(cudaMemset(h->d_counter, 0, sizeof(unsigned int)));
        CU(cudaMalloc(&h->d_eapply, sizeof(double) * B));
        // reduction partials: the larger of the tile grid and the element-wise grid, 4 values per CTA
        const size_t ctas = std::max((size_t)tile_ctas_per_member(h), (size_t)ew_grid(h).x) * B;
        size_t cap = 0;
        RC(ensure_buf(h, &h->d_partials, &cap, ctas * 4));
        CU(cudaMalloc(&h->d_obs_partials, sizeof(double) * 3 * obs_chunks(h) * B));
        CU(cudaMalloc(&h->d_obs_counters, sizeof(unsigned int) * B));
        CU(cudaMemset(h->d_obs_counters, 0, sizeof(unsigned int) * B));
        CU(cudaMalloc(&h->d_row_direct, sizeof(double) * 3 * B));
        CU(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
        RC(ensure_pool(h, 1));
        return TDSE_OK;
    };
    const int rc = body();
    if (rc != TDSE_OK) return fail(rc);
    *out = h;
    return TDSE_OK;
}

void tdse_destroy(tdse_handle *h) {
    if (!h) return;
    cudaDeviceSynchronize();
    free_graphs(h);
    for (double2 *p : h->pool) cudaFree(p);
    void *ptrs[] = {h->d_vj, h->d_cen, h->d_cl, h->d_pulse, h->d_bufs, h->d_ctl, h->d_etab, h->d_eapply, h->d_partials,
                    h->d_counter, h->d_phi, h->d_lstate, h->d_obs_partials, h->d_obs_counters, h->d_elog, h->d_imag_inv, h->d_mask, h->d_pb, h->d_sigma, h->d_j0, h->d_arun, h->d_loff, h->d_slist, h->d_yield, h->d_rp_part, h->d_rp_counter, h->d_rows, h->d_row_direct,
                    h->d_dtlog, h->d_errlog, h->d_replay, h->d_alpha, h->d_beta, h->d_nrm, h->d_inv, h->d_coef,
                    h->d_m, h->d_nsub, h->d_basis, h->d_rkp_ws};
    for (void *p : ptrs) if (p) cudaFree(p);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    cudaGetLastError();
    delete h;
}

int tdse_set_option(tdse_handle *h, const char *key, double value) {
    if (!h || !key) return TDSE_ERR_ARG;
    const std::string k(key);
    if (k == "field_sample") { if (value != 0.0 && value != 1.0) return TDSE_ERR_ARG; h->field_sample = (int)value; }
    else if (k == "use_graph") h->use_graph = value != 0.0;
    else if (k == "graph_steps") { if (value < 1 || value > 4096) return TDSE_ERR_ARG; h->graph_steps = (int)value; }
    else if (k == "taylor_block") { if (value != 0.0 && value != 1.0) return TDSE_ERR_ARG; h->taylor_block = (int)value; }
    else if (k == "taylor_rp_variant") { if (value < -1 || value >= kNumRpVariants) return TDSE_ERR_ARG; h->rp_variant = (int)value; free_graphs(h); }
    else if (k == "apply_tma") { if (value < 0 || value > 2) return TDSE_ERR_ARG; h->apply_tma = (int)value; }
    else if (k == "lanczos_tma") { if (value < 0 || value > 1) return TDSE_ERR_ARG; h->lanczos_tma = (int)value; free_graphs(h); }
    else if (k == "obs_fused") { if (value != 0.0 && value != 1.0 && value != 2.0) return TDSE_ERR_ARG; h->obs_fused = (int)value; free_graphs(h); }
    else if (k == "persist") { if (value < 0 || value > 64) return TDSE_ERR_ARG; h->persist = (int)value; free_graphs(h); }
    else if (k == "rk4_block") { if (value < 0 || value > 1) return TDSE_ERR_ARG; h->rk4_block = (int)value; free_graphs(h); }
    else if (k == "taylor_rp_tma") { if (value < -1 || value > 1) return TDSE_ERR_ARG; h->rp_tma = (int)value; free_graphs(h); }
    else if (k == "lanczos_beta_tol") { if (!(value >= 0.0)) return TDSE_ERR_ARG; h->beta_tol = value; free_graphs(h); }
    else if (k == "rk45_dt_max") { if (!(value >= 0.0)) return TDSE_ERR_ARG; h->rk45_dt_max = value; }
    else if (k == "rk45_check_every") { if (value < 1 || value > 1024) return TDSE_ERR_ARG; h->rk45_check_every = (int)value; }
    else if (k == "rk4_persist") { if (value != 0.0 && value != 1.0) return TDSE_ERR_ARG; h->rk4_persist = (int)value; }
    else if (k == "rk45_persist") { if (value != 0.0 && value != 1.0) return TDSE_ERR_ARG; h->rk45_persist = (int)value; }
    else if (k == "rk45_loop") { if (value != 0.0 && value != 1.0) return TDSE_ERR_ARG; h->rk45_use_loop = (int)value; }
    else return TDSE_ERR_ARG;
    return TDSE_OK;
}

int tdse_set_pulse(tdse_handle *h, const tdse_pulse *p) {
    if (!h || !p) return TDSE_ERR_ARG;
    bool quad = false;                  // velocity gauge + a pulse given by its field: A(t) by the running quadrature
    if (h->grid.gauge == 1)
        for (int b = 0; b < h->grid.batch; ++b) {
            if (p[b].kind != 0 && p[b].kind != 1) return TDSE_ERR_ARG;
            if (p[b].omega != 0.0 && p[b].kind == 0) quad = true;
        }
    CU(cudaDeviceSynchronize());
    if (quad != h->vg_quad) free_graphs(h);
    h->vg_quad = quad;
    if (quad && !h->d_arun) {
        CU(cudaMalloc(&h->d_arun, sizeof(double) * h->grid.batch));
        CU(cudaMemset(h->d_arun, 0, sizeof(double) * h->grid.batch));
    }
    CU(cudaMemcpy(h->d_pulse, p, sizeof(tdse_pulse) * h->grid.batch, cudaMemcpyHostToDevice));
    return TDSE_OK;
}

int tdse_set_bound_states(tdse_handle *h, int n_states, const int *l_of_state, const double *phi) {
    if (!h || n_states < 0 || (n_states > 0 && (!l_of_state || !phi))) return TDSE_ERR_ARG;
    for (int s = 0; s < n_states; ++s) if (l_of_state[s] < 0 || l_of_state[s] >= h->grid.n_l) return TDSE_ERR_ARG;
    CU(cudaDeviceSynchronize());
    free_graphs(h);
    if (h->d_phi) { cudaFree(h->d_phi); h->d_phi = nullptr; }
    if (h->d_lstate) { cudaFree(h->d_lstate); h->d_lstate = nullptr; }
    if (h->d_loff) { cudaFree(h->d_loff); h->d_loff = nullptr; }
    if (h->d_slist) { cudaFree(h->d_slist); h->d_slist = nullptr; }
    if (h->d_rows) { cudaFree(h->d_rows); h->d_rows = nullptr; h->rows_cap = 0; }
    if (h->d_row_direct) { cudaFree(h->d_row_direct); h->d_row_direct = nullptr; }
    h->n_states = n_states;
    h->log_rows = 0;
    CU(cudaMalloc(&h->d_row_direct, sizeof(double) * (3 + n_states) * h->grid.batch));
    if (n_states > 0) {
        CU(cudaMalloc(&h->d_phi, sizeof(double) * (size_t)n_states * h->grid.n_r));
        CU(cudaMalloc(&h->d_lstate, sizeof(int) * n_states));
        // states grouped by partial wave for pop_kernel: l_off[l] .. l_off[l+1] indexes state_list
        std::vector<int> loff(h->grid.n_l + 1, 0), slist(n_states);
        for (int s = 0; s < n_states; ++s) ++loff[l_of_state[s] + 1];
        for (int l = 0; l < h->grid.n_l; ++l) loff[l + 1] += loff[l];
        std::vector<int> fill(loff.begin(), loff.end() - 1);
        for (int s = 0; s < n_states; ++s) slist[fill[l_of_state[s]]++] = s;
        CU(cudaMalloc(&h->d_loff, sizeof(int) * loff.size()));
        CU(cudaMalloc(&h->d_slist, sizeof(int) * n_states));
        CU(cudaMemcpy(h->d_loff, loff.data(), sizeof(int) * loff.size(), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(h->d_slist, slist.data(), sizeof(int) * n_states, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(h->d_phi, phi, sizeof(double) * (size_t)n_states * h->grid.n_r, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(h->d_lstate, l_of_state, sizeof(int) * n_states, cudaMemcpyHostToDevice));
    }
    return TDSE_OK;
}

// psi <- P psi on the handle's state (no-op without a cut-off)
static int project_state(tdse_handle *h, cudaStream_t s) {
    if (!h->d_j0) return TDSE_OK;
    OpProject op{};
    op.psi = h->pool[h->psi_slot]; op.j0 = h->d_j0; op.n_r = h->grid.n_r; op.n_l = h->grid.n_l;
    h->pending = 0;
    RC(launch_ew(h, op, s));
    h->launches += h->pending;
    return TDSE_OK;
}

int tdse_set_state(tdse_handle *h, const void *psi, int is_device, void *stream) {
    if (!h || !psi) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (is_device < 0 || is_device > 2) return TDSE_ERR_ARG;
    CU(cudaMemcpyAsync(h->pool[h->psi_slot], psi, h->n_state * sizeof(double2),
                       is_device == 1 ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    if (is_device == 0) CU(cudaStreamSynchronize(s));
    RC(project_state(h, s));                          // centrifugal cut-off (if set): the held points are zero from here on
    return TDSE_OK;
}

int tdse_get_state(tdse_handle *h, void *psi, int is_device, void *stream) {
    if (!h || !psi) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (is_device < 0 || is_device > 2) return TDSE_ERR_ARG;
    CU(cudaMemcpyAsync(psi, h->pool[h->psi_slot], h->n_state * sizeof(double2),
                       is_device == 1 ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
    if (is_device == 0) CU(cudaStreamSynchronize(s));
    return TDSE_OK;
}

int tdse_apply_H(tdse_handle *h, const void *psi_dev, void *out_dev, const double *e_field_host, void *stream) {
    if (!h || !psi_dev || !out_dev || !e_field_host || psi_dev == out_dev) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const int B = h->grid.batch;
    if (!h->eapply_valid || std::memcmp(h->eapply_host.data(), e_field_host, sizeof(double) * B) != 0) {
        // the staging copy must not race with an earlier launch still reading d_eapply
        CU(cudaStreamSynchronize(s));
        h->eapply_host.assign(e_field_host, e_field_host + B);
        CU(cudaMemcpy(h->d_eapply, h->eapply_host.data(), sizeof(double) * B, cudaMemcpyHostToDevice));
        h->eapply_valid = true;
    }
    EpiApply e{};
    e.in = (const double2 *)psi_dev; e.ef = h->d_eapply; e.out = (double2 *)out_dev;
    h->pending = 0;
    // tiles fetched by TMA (zero fill outside the index box by the hardware) when the layout allows it
    // (and the grid is many rounds of resident CTAs: small, L2-resident grids measured 8 % slower this way)
    const long apply_items = (long)((h->grid.n_r + kTtTW - 1) / kTtTW) * ((h->grid.n_l + kTtTL - 1) / kTtTL) * B;
    if (h->apply_tma && (h->grid.n_r & 7) == 0 && ((uintptr_t)psi_dev & 15) == 0 &&
        (h->apply_tma == 2 || apply_items >= 6L * h->n_sm * kTtMinB)) {
        CUtensorMap tmv{};
        const CUtensorMap *tm = &tmv;
        if (tile_tensor_map(&tmv, psi_dev, h->grid.n_r, h->grid.n_l, B)) {
            const int tiles_r = (h->grid.n_r + kTtTW - 1) / kTtTW, tiles_l = (h->grid.n_l + kTtTL - 1) / kTtTL;
            const int n_items = tiles_r * tiles_l * B;
            const int smem = kTtStages * (int)kTtStageBytes + 64;
            const int grid = std::min(n_items, h->n_sm * kTtMinB);
            static DeviceOnce attr_once;
            if (attr_once.first()) {
                CU(cudaFuncSetAttribute(tile_tma_kernel<3, EpiApply>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
                CU(cudaFuncSetAttribute(tile_tma_kernel<5, EpiApply>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
                CU(cudaFuncSetAttribute(tile_tma_kernel<3, EpiApply, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
                CU(cudaFuncSetAttribute(tile_tma_kernel<5, EpiApply, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            }
            const bool vg = h->grid.gauge == 1;
            if (vg) {
                if (h->grid.fd_order == 3) tile_tma_kernel<3, EpiApply, true><<<grid, 256, smem, s>>>(h->gd, e, *tm, tiles_r, tiles_l, n_items);
                else tile_tma_kernel<5, EpiApply, true><<<grid, 256, smem, s>>>(h->gd, e, *tm, tiles_r, tiles_l, n_items);
            } else if (h->grid.fd_order == 3) tile_tma_kernel<3, EpiApply><<<grid, 256, smem, s>>>(h->gd, e, *tm, tiles_r, tiles_l, n_items);
            else tile_tma_kernel<5, EpiApply><<<grid, 256, smem, s>>>(h->gd, e, *tm, tiles_r, tiles_l, n_items);
            count(h);
            CU(cudaGetLastError());
            h->launches += h->pending;
            return TDSE_OK;
        }
    }
    RC(launch_tile(h, e, s));
    h->launches += h->pending;
    return TDSE_OK;
}

static int step_taylor_impl(tdse_handle *h, int order, double t0, double dt, long nsteps, int obs_every, void *stream);

int tdse_step_taylor(tdse_handle *h, int order, double t0, double dt, long nsteps, int obs_every, void *stream) {
    if (!h || order < 1 || order > 64 || nsteps < 0 || obs_every < 0 || !(dt == dt)) return TDSE_ERR_ARG;
    h->imag = 0;
    return step_taylor_impl(h, order, t0, dt, nsteps, obs_every, stream);
}

int tdse_step_imag(tdse_handle *h, int order, double dt, long nsteps, void *stream) {
    if (!h || order < 1 || order > 64 || nsteps < 0 || !(dt > 0.0)) return TDSE_ERR_ARG;
    const size_t need = (size_t)std::max(1L, nsteps) * h->grid.batch;
    RC(ensure_buf(h, &h->d_elog, &h->elog_cap, need));
    if (!h->d_imag_inv) CU(cudaMalloc(&h->d_imag_inv, sizeof(double) * h->grid.batch));
    h->imag = 1;
    const int rc = step_taylor_impl(h, order, 0.0, dt, nsteps, 0, stream);
    h->imag = 0;
    if (rc == TDSE_OK) h->elog_rows = nsteps;
    return rc;
}

int tdse_energy_log(tdse_handle *h, double *energy_host, long max_rows, void *stream) {
    if (!h || !energy_host || max_rows < 0) return TDSE_ERR_ARG;
    const long rows = std::min(max_rows, h->elog_rows);
    if (rows > 0) {
        CU(cudaMemcpyAsync(energy_host, h->d_elog, sizeof(double) * rows * h->grid.batch, cudaMemcpyDeviceToHost,
                           (cudaStream_t)stream));
        CU(cudaStreamSynchronize((cudaStream_t)stream));
    }
    return TDSE_OK;
}

static int step_taylor_impl(tdse_handle *h, int order, double t0, double dt, long nsteps, int obs_every, void *stream) {
    RC(ensure_pool(h, 4));
    // taylor_block: 0 one kernel per order; 1 all orders in one pass (persistent register-patch kernel) when
    // the grid allows it (n_l <= 128), else one kernel per order
    h->taylor_blocked_last = 0;
    h->rk4_fused = 0;
    h->rpp = RpPlan{};
    // (the all-orders-in-one-pass kernel implements the length-gauge coupling only; imaginary time has no field)
    const bool lg = (h->grid.gauge == 0 || h->imag) && !(h->imag && h->d_j0);      // (imaginary time with a cut-off: per order)
    if (lg && h->taylor_block == 1) {
        // (persistent steps: real-time Taylor on grids one CTA per member can hold, logged rows fused or none)
        // (several steps per launch: real-time Taylor on SMALL grids -- at most one wave of CTAs --, no cut-off, logged
        // rows fusable or none; the deepest blocking that keeps the interior of a tile at least half of it)
        h->rpp = RpPlan{};
        const bool may_persist = h->persist > 1 && h->rp_tma != 1 && !h->imag && !h->d_j0 &&
                                 (obs_every == 0 || (h->obs_fused && h->n_states <= kRpObsStates));
        for (int k = may_persist ? h->persist : 0; k > 1 && !h->rpp.ok; k /= 2) {
            RpPlan p = rp_plan(h->grid, order, h->n_sm, h->rp_variant, 0, 0, k);
            if (p.ok && (long)p.n_items * p.cl <= h->n_sm) h->rpp = p;
        }
        if (!h->rpp.ok) h->rpp = rp_plan(h->grid, order, h->n_sm, h->rp_variant, h->rp_tma, h->imag ? 2 : 0);
        if (h->rpp.ok) h->taylor_blocked_last = 3;
    }
    return run_fixed(h, KIND_TAYLOR, order, 0, t0, dt, nsteps, obs_every, (cudaStream_t)stream);
}

int tdse_step_rk4(tdse_handle *h, double t0, double dt, long nsteps, int obs_every, void *stream) {
    if (!h || nsteps < 0 || obs_every < 0) return TDSE_ERR_ARG;
    h->rk45_persist_last = 0;
    // Grids that fit on chip, no logged rows, no absorber: the whole call runs in the persistent Runge-Kutta kernel, classic
    // RK4 written as an FSAL scheme of five stage vectors (the fifth is psi_new, its k the k_1 of the next step); field
    // values of all stage times from a table, a launch per 2048 steps.
    if (h->rk4_persist && obs_every == 0 && nsteps > 0 && !h->d_mask && !h->vg_quad) {
        const RkpPlan pp = rkp_plan_for(h);
        if (pp.ok) {
            cudaStream_t s = (cudaStream_t)stream;
            const int B = h->grid.batch, NS = 5;
            const long chunk = 2048;
            RC(ensure_pool(h, 1));
            RC(ensure_buf(h, &h->d_etab, &h->etab_cap, (size_t)std::min(chunk, nsteps) * NS * B));
            h->taylor_blocked_last = 0; h->rk4_fused = 0; h->rpp = RpPlan{};
            CtlInit v{};
            v.t0 = t0; v.dt = dt; v.obs_every = 0; v.field_sample = h->field_sample;
            h->pending = 0;
            RC(init_ctl(h, v, s));
            StageTimes cs{};
            cs.c[0] = 0.0; cs.c[1] = 0.5; cs.c[2] = 0.5; cs.c[3] = 1.0; cs.c[4] = 1.0;
            for (long done = 0; done < nsteps;) {
                const long n = std::min(chunk, nsteps - done);
                field_table_rk_kernel<<<(unsigned)((n * NS * B + 255) / 256), 256, 0, s>>>(h->d_ctl, h->d_pulse, B, (int)n, NS, cs,
                                                                                         h->d_etab, h->gd.gauge);
                count(h);
                RkpArgs a{};
                RC(rkp_prepare(h, pp, a, s));
                a.n_stage = NS; a.fixed = 1; a.n_fixed = n; a.e_tab = h->d_etab;
                for (int i = 1; i < 4; ++i)
                    for (int j = 0; j < i; ++j) a.a[i][j] = RK4_A[i][j];
                for (int j = 0; j < 4; ++j) a.a[4][j] = RK4_B[j];
                RC(launch_rk45_persist(a, pp, s));
                count(h);
                ctl_advance_kernel<<<1, 32, 0, s>>>(h->d_ctl, (int)n);
                count(h);
                done += n;
            }
            CU(cudaGetLastError());
            h->launches += h->pending;
            h->log_rows = 0;
            h->rk45_persist_last = 1;
            return TDSE_OK;
        }
    }
    RC(ensure_pool(h, 6));
    h->taylor_blocked_last = 0;
    h->rk4_fused = 0;
    h->rpp = RpPlan{};
    if (h->rk4_block && h->grid.gauge == 0) {           // all four stages in one pass (register-patch kernel in RK mode) when it applies
        h->rpp = rp_plan(h->grid, 4, h->n_sm, -1, h->rp_tma, 1);
        if (h->rpp.ok) { h->rk4_fused = 1; h->taylor_blocked_last = 3; }
        else h->rpp = RpPlan{};
    }
    rk_roles(h);
    RC(upload_bufs(h, 6, (cudaStream_t)stream));
    return run_fixed(h, KIND_RK4, 0, 0, t0, dt, nsteps, obs_every, (cudaStream_t)stream);
}

int tdse_step_lanczos(tdse_handle *h, int K, int order, double t0, double dt, long nsteps, int obs_every, void *stream) {
    if (!h || K < 1 || order < 1 || nsteps < 0 || obs_every < 0) return TDSE_ERR_ARG;
    if (K > kMaxKrylov) return TDSE_ERR_UNSUPPORTED;
    RC(ensure_pool(h, 3));
    h->taylor_blocked_last = 0;
    const int B = h->grid.batch;
    if (h->lz_K != K) {
        CU(cudaDeviceSynchronize());
        free_graphs(h);
        void *old[] = {h->d_alpha, h->d_beta, h->d_nrm, h->d_inv, h->d_coef, h->d_m, h->d_nsub, h->d_basis};
        for (void *p : old) if (p) cudaFree(p);
        h->d_alpha = h->d_beta = h->d_nrm = h->d_inv = nullptr; h->d_coef = nullptr; h->d_m = h->d_nsub = nullptr;
        h->d_basis = nullptr; h->lz_K = 0;
        CU(cudaMalloc(&h->d_alpha, sizeof(double) * B * K));
        CU(cudaMalloc(&h->d_beta, sizeof(double) * B * K));
        CU(cudaMalloc(&h->d_nrm, sizeof(double) * B));
        CU(cudaMalloc(&h->d_inv, sizeof(double) * B * K));
        CU(cudaMalloc(&h->d_coef, sizeof(double2) * B * K));
        CU(cudaMalloc(&h->d_m, sizeof(int) * B));
        CU(cudaMalloc(&h->d_nsub, sizeof(int) * B));
        CU(cudaMalloc(&h->d_basis, sizeof(double2) * h->n_state * K));
        h->lz_K = K;
    }
    CU(cudaMemsetAsync(h->d_alpha, 0, sizeof(double) * B * K, (cudaStream_t)stream));
    CU(cudaMemsetAsync(h->d_beta, 0, sizeof(double) * B * K, (cudaStream_t)stream));
    return run_fixed(h, KIND_LANCZOS, K, order, t0, dt, nsteps, obs_every, (cudaStream_t)stream);
}

int tdse_step_rk(tdse_handle *h, int method, double t0, double dt, long nsteps, int obs_every, void *stream) {
    if (!h || method < 0 || method > 5 || nsteps < 0 || obs_every < 0) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->d_sigma) CU(cudaMalloc(&h->d_sigma, sizeof(double) * h->grid.batch));
    CU(cudaMemsetAsync(h->d_sigma, 0, sizeof(double) * h->grid.batch, s));
    if (method == 0) return tdse_step_rk4(h, t0, dt, nsteps, obs_every, stream);      // (fused kernel when it applies)
    RC(ensure_pool(h, kRkRoles));
    h->taylor_blocked_last = 0;
    h->rk4_fused = 0;
    h->imag = 0;
    rk_roles(h);
    RC(upload_bufs(h, kRkRoles, s));
    return run_fixed(h, KIND_RKGEN, method, 0, t0, dt, nsteps, obs_every, s);
}

int tdse_rk_sigma(tdse_handle *h, double *sigma_host, void *stream) {
    if (!h || !sigma_host) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->d_sigma) { for (int b = 0; b < h->grid.batch; ++b) sigma_host[b] = 0.0; return TDSE_OK; }
    CU(cudaMemcpyAsync(sigma_host, h->d_sigma, sizeof(double) * h->grid.batch, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return TDSE_OK;
}

int tdse_step_rk45(tdse_handle *h, double t0, double t_end, double dt_init, double rtol, const double *dt_replay,
                   long n_replay, long *n_accept, long *n_reject, void *stream) {
    if (!h || !(rtol > 0.0)) return TDSE_ERR_ARG;
    if (h->d_mask) return TDSE_ERR_UNSUPPORTED;      // the per-step mask of Eq. 18 presumes a fixed dt
    if (h->vg_quad) return TDSE_ERR_UNSUPPORTED;     // (the running quadrature of A(t) is built for the fixed-step propagators)
    const bool replay = dt_replay != nullptr;
    if (replay ? (n_replay < 0) : (!(dt_init > 0.0) || !(t_end > t0))) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const int B = h->grid.batch;
    // grids that fit the shared memory of the machine: the whole run is one persistent kernel (tdse_rk45_persist.cuh)
    RkpPlan pp{};
    if (h->rk45_persist) pp = rkp_plan_for(h);
    h->rk45_persist_last = pp.ok;
    h->taylor_blocked_last = 0;
    if (!pp.ok) {
        RC(ensure_pool(h, kRkRoles));
        rk_roles(h);
        RC(upload_bufs(h, kRkRoles, s));
        RC(ensure_buf(h, &h->d_etab, &h->etab_cap, (size_t)std::max(1, h->graph_steps) * 7 * B));
    }
    // logs
    const long want_log = replay ? std::max(1L, n_replay) : (1L << 20);
    if (h->log_cap < want_log) {
        CU(cudaDeviceSynchronize());
        free_graphs(h);
        if (h->d_dtlog) cudaFree(h->d_dtlog);
        if (h->d_errlog) cudaFree(h->d_errlog);
        h->d_dtlog = h->d_errlog = nullptr; h->log_cap = 0;
        CU(cudaMalloc(&h->d_dtlog, sizeof(double) * want_log));
        CU(cudaMalloc(&h->d_errlog, sizeof(double) * want_log));
        h->log_cap = want_log;
    }
    if (replay && n_replay > 0) {
        if (h->replay_cap < n_replay) {
            CU(cudaDeviceSynchronize());
            free_graphs(h);
            if (h->d_replay) cudaFree(h->d_replay);
            h->d_replay = nullptr; h->replay_cap = 0;
            CU(cudaMalloc(&h->d_replay, sizeof(double) * n_replay));
            h->replay_cap = n_replay;
        }
        CU(cudaMemcpy(h->d_replay, dt_replay, sizeof(double) * n_replay, cudaMemcpyHostToDevice));
    }
    h->last_accept = 0;
    if (n_accept) *n_accept = 0;
    if (n_reject) *n_reject = 0;
    if (replay && n_replay == 0) return TDSE_OK;
    CtlInit v{};
    v.t = t0; v.t_end = t_end; v.rtol = rtol; v.dt_max = h->rk45_dt_max; v.replay = replay ? 1 : 0;
    v.n_replay = n_replay; v.max_log = h->log_cap;
    v.h = dt_init;
    if (!replay && v.dt_max > 0.0 && v.h > v.dt_max) v.h = v.dt_max;
    h->pending = 0;
    RC(init_ctl(h, v, s));
    if (pp.ok) {
        RkpArgs a{};
        RC(rkp_prepare(h, pp, a, s));
        a.n_stage = 7;
        for (int i = 0; i < 7; ++i) {
            for (int j = 0; j < 7; ++j) a.a[i][j] = DP_A[i][j];
            a.d_err[i] = DP_B[i] - DP_BH[i];
        }
        RC(launch_rk45_persist(a, pp, s));
        count(h);
        h->launches += h->pending;
        Ctl hc{};
        CU(cudaMemcpyAsync(&hc, h->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        if (!hc.done) return TDSE_ERR_NONFINITE;            // the run stopped on a step that is no positive number
        h->last_accept = (long)hc.n_accept;
        if (n_accept) *n_accept = (long)hc.n_accept;
        if (n_reject) *n_reject = (long)hc.n_reject;
        return TDSE_OK;
    }
    // the first attempted step needs k_1 (no FSAL yet): run it eagerly with stage 0 included
    RC(enqueue_rk45_block(h, 1, 0, s));
    h->launches += h->pending;
    const int G = std::max(1, h->rk45_check_every);
    Ctl hc{};
    if (h->rk45_use_loop && h->use_graph && build_rk45_loop(h, G) == TDSE_OK) {
        // device-driven: one graph launch runs blocks of G attempted steps until the controller is done
        CU(cudaGraphLaunch(h->rk45_loop, s));
        CU(cudaMemcpyAsync(&hc, h->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        h->launches += h->rk45_loop_nodes * ((hc.n_attempt - 1 + G - 1) / G);
        h->psi_slot = h->role_slot[hc.perm[R_PSI]];
        if (!hc.done) return TDSE_ERR_NONFINITE;            // the loop stopped on a step that is no positive number
        h->last_accept = (long)hc.n_accept;
        if (n_accept) *n_accept = (long)hc.n_accept;
        if (n_reject) *n_reject = (long)hc.n_reject;
        return TDSE_OK;
    }
    for (;;) {
        CU(cudaMemcpyAsync(&hc, h->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        if (hc.done) break;
        if (!(hc.h > 0.0) || hc.n_attempt > (1LL << 40)) {
            h->psi_slot = h->role_slot[hc.perm[R_PSI]];       // the state follows the device's role swaps even on failure
            return TDSE_ERR_NONFINITE;
        }
        RC(run_blocks(h, KIND_RK45, 0, 0, G, 0, 1, s));
    }
    // the device swapped roles on every accept: make the host's view of "the state" follow
    h->psi_slot = h->role_slot[hc.perm[R_PSI]];
    h->last_accept = (long)hc.n_accept;
    if (n_accept) *n_accept = (long)hc.n_accept;
    if (n_reject) *n_reject = (long)hc.n_reject;
    return TDSE_OK;
}

int tdse_observables(tdse_handle *h, double t, double *out_host, void *stream) {
    if (!h || !out_host) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    h->pending = 0;
    RC(enqueue_obs(h, h->pool[h->psi_slot], 0, 0, 1, t, h->d_row_direct, s));
    h->launches += h->pending;
    CU(cudaMemcpyAsync(out_host, h->d_row_direct, sizeof(double) * (3 + h->n_states) * h->grid.batch,
                       cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return TDSE_OK;
}

int tdse_obs_log(tdse_handle *h, double *out_host, long max_rows, long *rows) {
    if (!h || !rows || max_rows < 0 || (max_rows > 0 && !out_host)) return TDSE_ERR_ARG;
    CU(cudaDeviceSynchronize());
    *rows = h->log_rows;
    const long n = std::min(max_rows, h->log_rows);
    const size_t W = 3 + h->n_states, per = W * h->grid.batch;
    if (n > 0) {
        CU(cudaMemcpy(out_host, h->d_rows, sizeof(double) * per * n, cudaMemcpyDeviceToHost));
        for (long r = 0; r < n; ++r)
            for (int b = 0; b < h->grid.batch; ++b)
                if (!std::isfinite(out_host[r * per + b * W])) return TDSE_ERR_NONFINITE;
    }
    return TDSE_OK;
}

int tdse_dt_log(tdse_handle *h, double *dt_host, double *err_host, long max, long *n) {
    if (!h || !n || max < 0 || (max > 0 && !dt_host)) return TDSE_ERR_ARG;
    CU(cudaDeviceSynchronize());
    *n = h->last_accept;
    const long c = std::min(std::min(max, h->last_accept), h->log_cap);
    if (c > 0) {
        CU(cudaMemcpy(dt_host, h->d_dtlog, sizeof(double) * c, cudaMemcpyDeviceToHost));
        if (err_host) CU(cudaMemcpy(err_host, h->d_errlog, sizeof(double) * c, cudaMemcpyDeviceToHost));
    }
    return TDSE_OK;
}

int tdse_lanczos_info(tdse_handle *h, double *alpha, double *beta, double *coef, int *m_used, int *n_sub) {
    if (!h) return TDSE_ERR_ARG;
    if (h->lz_K == 0) return TDSE_ERR_ARG;
    CU(cudaDeviceSynchronize());
    const size_t n = (size_t)h->grid.batch * h->lz_K;
    if (alpha) CU(cudaMemcpy(alpha, h->d_alpha, sizeof(double) * n, cudaMemcpyDeviceToHost));
    if (beta) CU(cudaMemcpy(beta, h->d_beta, sizeof(double) * n, cudaMemcpyDeviceToHost));
    if (coef) CU(cudaMemcpy(coef, h->d_coef, sizeof(double2) * n, cudaMemcpyDeviceToHost));
    if (m_used) CU(cudaMemcpy(m_used, h->d_m, sizeof(int) * h->grid.batch, cudaMemcpyDeviceToHost));
    if (n_sub) CU(cudaMemcpy(n_sub, h->d_nsub, sizeof(int) * h->grid.batch, cudaMemcpyDeviceToHost));
    return TDSE_OK;
}

long tdse_launch_count(tdse_handle *h) { return h ? h->launches : 0; }
long tdse_graph_instantiations(tdse_handle *h) { return h ? h->graph_inst : 0; }

int tdse_ionisation_yield(tdse_handle *h, double *out_host, void *stream) {
    if (!h || !out_host) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->d_yield) CU(cudaMalloc(&h->d_yield, sizeof(double) * h->grid.batch));
    h->pending = 0;
    RC(enqueue_obs(h, h->pool[h->psi_slot], 0, 0, 1, 0.0, h->d_row_direct, s));
    yield_kernel<<<h->grid.batch, 32, 0, s>>>(h->d_row_direct, h->n_states, h->d_yield);
    count(h);
    CU(cudaGetLastError());
    h->launches += h->pending;
    CU(cudaMemcpyAsync(out_host, h->d_yield, sizeof(double) * h->grid.batch, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return TDSE_OK;
}

int tdse_set_absorber(tdse_handle *h, double r_b, int p) {
    if (!h || (r_b > 0.0 && p < 1)) return TDSE_ERR_ARG;
    CU(cudaDeviceSynchronize());
    free_graphs(h);                                   // captured kernels hold the grid description by value
    if (!(r_b > 0.0)) {
        if (h->d_mask) cudaFree(h->d_mask);
        h->d_mask = nullptr; h->gd.mask = nullptr;
        return TDSE_OK;
    }
    const int N = h->grid.n_r;
    std::vector<double> m(N);
    for (int j = 0; j < N; ++j) {                      // exp(-i W(r_j) dt) of P:146 Eq. 18 = 1 - cos^p[(pi/2)(1 - r/r_b)]
        const double r = (j + 1) * h->grid.dr;
        m[j] = (r >= r_b) ? 0.0 : 1.0 - std::pow(std::cos(0.5 * 3.14159265358979323846 * (1.0 - r / r_b)), (double)p);
    }
    if (!h->d_mask) CU(cudaMalloc(&h->d_mask, sizeof(double) * N));
    CU(cudaMemcpy(h->d_mask, m.data(), sizeof(double) * N, cudaMemcpyHostToDevice));
    h->gd.mask = h->d_mask;
    return TDSE_OK;
}

int tdse_set_cutoff(tdse_handle *h, double lambda) {
    if (!h || !(lambda >= 0.0)) return TDSE_ERR_ARG;
    CU(cudaDeviceSynchronize());
    free_graphs(h);                                   // captured kernels hold the grid description by value
    h->cutoff = lambda;
    if (!(lambda > 0.0)) {
        if (h->d_j0) cudaFree(h->d_j0);
        h->d_j0 = nullptr; h->gd.j0 = nullptr; h->gd.j0_max = 0;
        return TDSE_OK;
    }
    const int N = h->grid.n_r, L = h->grid.n_l;
    std::vector<int> j0(L, 0);
    int jmax = 0;
    for (int l = 0; l < L; ++l) {
        // point (l, j) is held iff l(l+1) > (2 Lambda) r_j^2 with r_j = (j+1) dr, in exactly this operation order
        int j = 0;
        while (j < N) {
            const double r = (double)(j + 1) * h->grid.dr;
            if (!((double)(l * (l + 1)) > (2.0 * lambda) * (r * r))) break;
            ++j;
        }
        j0[l] = j;
        jmax = std::max(jmax, j);
    }
    if (!h->d_j0) CU(cudaMalloc(&h->d_j0, sizeof(int) * L));
    CU(cudaMemcpy(h->d_j0, j0.data(), sizeof(int) * L, cudaMemcpyHostToDevice));
    h->gd.j0 = h->d_j0; h->gd.j0_max = jmax;
    RC(project_state(h, nullptr));
    CU(cudaDeviceSynchronize());
    return TDSE_OK;
}

int tdse_bound_population(tdse_handle *h, double r_b, double *out_host, void *stream) {
    if (!h || !out_host || !(r_b >= 0.0)) return TDSE_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->d_pb) CU(cudaMalloc(&h->d_pb, sizeof(double) * h->grid.batch));
    OpBoundPop op{};
    op.psi = h->pool[h->psi_slot]; op.n_r = h->grid.n_r; op.dr = h->grid.dr; op.out = h->d_pb;
    int jm = 0;
    while (jm < h->grid.n_r && (jm + 1) * h->grid.dr <= r_b) ++jm;      // r_j = (j+1) dr <= r_b  (R-G27)
    op.j_max = jm;
    h->pending = 0;
    RC(launch_ew(h, op, s));
    h->launches += h->pending;
    CU(cudaMemcpyAsync(out_host, h->d_pb, sizeof(double) * h->grid.batch, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return TDSE_OK;
}

int tdse_taylor_was_blocked(tdse_handle *h) { return h ? h->taylor_blocked_last + ((h->taylor_blocked_last == 3 && h->rpp.tma) ? 1 : 0) : 0; }
int tdse_rk45_was_persistent(tdse_handle *h) { return h ? h->rk45_persist_last : 0; }
int tdse_taylor_plan(tdse_handle *h, int *variant, int *steps_per_launch, int *ctas) {
    if (!h) return TDSE_ERR_ARG;
    const bool used = h->taylor_blocked_last == 3 || h->rk4_fused;
    if (variant) *variant = (used && h->rpp.ok) ? h->rpp.variant : -1;
    if (steps_per_launch) *steps_per_launch = (used && h->rpp.ok && h->rpp.persist > 1) ? h->rpp.persist : 1;
    if (ctas) *ctas = (used && h->rpp.ok) ? h->rpp.grid : 0;
    return TDSE_OK;
}

}  // extern "C"
