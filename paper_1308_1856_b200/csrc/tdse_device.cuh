// tdse_device.cuh -- device-side data structures and helpers shared by all kernels of libtdse_b200.
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tdse.h"

namespace tdse {

constexpr int kMaxKrylov = 32;     // one lane per Krylov coefficient in the small exponential
constexpr int kRkRoles   = 10;     // PSI, G0, G1, K0..K6

// Grid description and device tables handed to every kernel by value.
struct GridDev {
    int n_r, n_l, batch, fd;
    int gauge;              // 0 length gauge (Eq. 11), 1 velocity gauge (Eq. 12 in reading R-V2)
    double dr, z;
    double c1, c2;          // off-diagonal stencil weights of -1/2 D2: 3-point c1 = -1/(2dr^2); 5-point c1 = -16/(24dr^2), c2 = +1/(24dr^2)
    const double *vj;       // [n_r]  kinetic diagonal - Z/r_j          (Eq. 7, Eq. 15)
    const double *cen;      // [n_r]  1/(2 r_j^2)                       (centrifugal factor, Eq. 7)
    const double *cl;       // [n_l]  c_l = (l+1)/sqrt((2l+1)(2l+3))    (Eq. 9, m = 0)
    const int *j0;          // [n_l]  centrifugal inner cut-off (an extension beyond the paper, tdse_set_cutoff): the points
                            //        (l, j < j0[l]) are HELD at zero, H acts as its principal sub-matrix on the others;
                            //        nullptr: no cut-off
    int j0_max;             //        max_l j0[l]: columns >= j0_max are untouched by the cut-off
    const double *mask;     // [n_r]  absorbing-boundary factor exp(-i W(r_j) dt) of P:146 Eq. 18 applied after every
                            //        step, or nullptr (no absorber)
};

// Device-resident control block: everything a captured graph must be able to re-read at launch time.
struct Ctl {
    // fixed-step propagators
    double t0, dt;
    long long step_base;            // index (within this call) of the first step of the running block
    int obs_every, field_sample;
    // adaptive / replayed Dormand-Prince
    double t, h, t_end, rtol, dt_max;
    int done, last, after_reject, replay;
    long long n_accept, n_reject, n_attempt, n_replay, max_log;
    int perm[kRkRoles];             // role -> buffer index (swapped on accept: psi <-> psi_new, k1 <-> k7)
};

struct CtlInit {
    double t0, dt; int obs_every, field_sample;
    double t, h, t_end, rtol, dt_max; int replay; long long n_replay, max_log;
};

// Reduction context of a kernel launch: per-CTA partial sums, a ticket counter, and the CTA count.
struct RedCtx {
    double *partials;               // [ctas][NRED]
    unsigned int *counter;          // zero before the launch; reset by the last CTA
    int ctas_per_member;
};

// is point (l, j) (0-based column) held at zero by the centrifugal cut-off?  (rows outside 0..n_l-1 are zero anyway)
__device__ __forceinline__ bool held_pt(const GridDev &g, int l, int j) {
    return g.j0 != nullptr && l >= 0 && l < g.n_l && j < __ldg(g.j0 + l);
}

__device__ __forceinline__ double2 ldcg2(const double2 *p) { return __ldcg(p); }

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
// a + s*b, s real
__device__ __forceinline__ double2 caxpy_r(double s, double2 b, double2 a) {
    return make_double2(fma(s, b.x, a.x), fma(s, b.y, a.y));
}

// E(t) of one member (Eq. 19 with the Hann envelope of P:166; reading R-G8).  The time bookkeeping uses
// explicitly rounded operations so that t itself carries no contraction-dependent bits.
__device__ inline double pulse_E(const tdse_pulse &p, double t) {
    if (p.omega == 0.0) return p.e0;
    const double T = __ddiv_rn(__dmul_rn(2.0 * 3.14159265358979323846, p.n_cycles), p.omega);
    if (t < 0.0 || t > T) return 0.0;
    const double wt = __dmul_rn(p.omega, t);
    const double hw = __ddiv_rn(wt, __dmul_rn(2.0, p.n_cycles));
    if (p.kind == 1) {      // E = -dA/dt of the Hann-shaped vector potential (R-V3)
        const double Om = __ddiv_rn(p.omega, __dmul_rn(2.0, p.n_cycles));
        const double s = sin(hw), c = cos(hw), ph = __dadd_rn(wt, p.cep);
        return (p.e0 / p.omega) * s * (2.0 * Om * c * sin(ph) + p.omega * s * cos(ph));
    }
    const double s = sin(hw);
    return __dmul_rn(__dmul_rn(__dmul_rn(p.e0, s), s), cos(__dadd_rn(wt, p.cep)));
}

// A(t) of a kind-1 pulse (R-V3); the static test aid (omega = 0) has A = e0; kind 0 has no closed form here
__device__ inline double pulse_A(const tdse_pulse &p, double t) {
    if (p.omega == 0.0) return p.e0;
    if (p.kind != 1) return nan("");
    const double T = __ddiv_rn(__dmul_rn(2.0 * 3.14159265358979323846, p.n_cycles), p.omega);
    if (t < 0.0 || t > T) return 0.0;
    const double wt = __dmul_rn(p.omega, t);
    const double s = sin(__ddiv_rn(wt, __dmul_rn(2.0, p.n_cycles)));
    return -(p.e0 / p.omega) * s * s * sin(__dadd_rn(wt, p.cep));
}

// Velocity gauge with a pulse given by its FIELD (kind 0): A(t) exists only as the running quadrature of P:186-188,
// A(t_{n+1}) = A(t_n) - int_{t_n}^{t_n + h} E dtau "using a standard 5-point Gaussian quadrature" (c dropped), and
// A(t_n + c_i h) = A(t_n) - int_{t_n}^{t_n + c_i h} E dtau inside a step.
__device__ __forceinline__ bool pulse_needs_quadrature(const tdse_pulse &p, int gauge) {
    return gauge == 1 && p.omega != 0.0 && p.kind == 0;
}
// int_{ta}^{tb} E dtau by ONE 5-point Gauss-Legendre rule
__device__ inline double gl5_field(const tdse_pulse &p, double ta, double tb) {
    const double x1 = 0.5384693101056831, x2 = 0.9061798459386640;          // nodes on [-1, 1] (0, +-x1, +-x2)
    const double w0 = 0.5688888888888889, w1 = 0.4786286704993665, w2 = 0.2369268850561891;
    const double half = 0.5 * (tb - ta), mid = 0.5 * (tb + ta);
    double s = w2 * pulse_E(p, mid - half * x2);
    s += w1 * pulse_E(p, mid - half * x1);
    s += w0 * pulse_E(p, mid);
    s += w1 * pulse_E(p, mid + half * x1);
    s += w2 * pulse_E(p, mid + half * x2);
    return half * s;
}

// the time-dependent factor of the coupling: E(t) in the length gauge, A(t) in the velocity gauge
__device__ inline double pulse_field(const tdse_pulse &p, double t, int gauge) {
    return gauge == 1 ? pulse_A(p, t) : pulse_E(p, t);
}

// t0 + x*dt with two roundings (never contracted)
__device__ __forceinline__ double time_at(double t0, double x, double dt) { return __dadd_rn(t0, __dmul_rn(x, dt)); }

// Deterministic block reduction of NRED doubles per thread: warp shuffle tree, then a fixed-order pass over
// the per-warp results.  Result valid in thread 0.  scratch: NRED * (NT/32) doubles of shared memory.
template <int NT, int NRED>
__device__ __forceinline__ void block_reduce(double (&v)[NRED], double *scratch) {
    constexpr int NW = NT / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int r = 0; r < NRED; ++r) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v[r] += __shfl_down_sync(0xffffffffu, v[r], off);
    }
    __syncthreads();   // scratch may still be in use by a previous call
    if (lane == 0) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) scratch[r * NW + warp] = v[r];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) {
            double x = (lane < NW) ? scratch[r * NW + lane] : 0.0;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) x += __shfl_down_sync(0xffffffffu, x, off);
            v[r] = x;
        }
    }
}

// Two-stage grid reduction with a "last CTA finishes" second stage (replaces the paper's redundant
// per-work-group second stage).  Every CTA of the launch must call this exactly once.
// cta_linear = member * ctas_per_member + tile.  The last CTA sums the partials of every member in a fixed
// order and calls fin.finish_member(b, sums) for each, then fin.finish_all(), from thread 0.
template <int NT, int NRED, class Fin>
__device__ __forceinline__ void grid_reduce_finish(double (&red)[NRED], const RedCtx &rc, int cta_linear,
                                                   int total_ctas, int n_members, Fin &fin, double *scratch,
                                                   int *flag) {
    block_reduce<NT, NRED>(red, scratch);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) rc.partials[(size_t)cta_linear * NRED + r] = red[r];
        __threadfence();
        const unsigned int ticket = atomicAdd(rc.counter, 1u);
        *flag = (ticket == (unsigned int)(total_ctas - 1));
    }
    __syncthreads();
    if (!*flag) return;
    __threadfence();
    for (int b = 0; b < n_members; ++b) {
        double s[NRED];
#pragma unroll
        for (int r = 0; r < NRED; ++r) s[r] = 0.0;
        const double *p = rc.partials + (size_t)b * rc.ctas_per_member * NRED;
        for (int i = threadIdx.x; i < rc.ctas_per_member; i += NT) {
#pragma unroll
            for (int r = 0; r < NRED; ++r) s[r] += __ldcg(p + (size_t)i * NRED + r);
        }
        block_reduce<NT, NRED>(s, scratch);
        if (threadIdx.x == 0) fin.finish_member(b, s);
    }
    if (threadIdx.x == 0) {
        fin.finish_all();
        *rc.counter = 0u;
    }
}

// The same in two parts for persistent kernels: a CTA stores one partial per WORK ITEM (slot = member *
// items_per_member + item), and signs off once at its end; the last CTA to sign off finishes as above.
template <int NT, int NRED>
__device__ __forceinline__ void grid_store_partial(double (&red)[NRED], const RedCtx &rc, size_t slot, double *scratch) {
    block_reduce<NT, NRED>(red, scratch);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) rc.partials[slot * NRED + r] = red[r];
    }
}
template <int NT, int NRED, class Fin>
__device__ __forceinline__ void grid_finish(const RedCtx &rc, int total_ctas, int n_members, Fin &fin, double *scratch,
                                            int *flag) {
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int ticket = atomicAdd(rc.counter, 1u);
        *flag = (ticket == (unsigned int)(total_ctas - 1));
    }
    __syncthreads();
    if (!*flag) return;
    __threadfence();
    for (int b = 0; b < n_members; ++b) {
        double s[NRED];
#pragma unroll
        for (int r = 0; r < NRED; ++r) s[r] = 0.0;
        const double *p = rc.partials + (size_t)b * rc.ctas_per_member * NRED;
        for (int i = threadIdx.x; i < rc.ctas_per_member; i += NT) {
#pragma unroll
            for (int r = 0; r < NRED; ++r) s[r] += __ldcg(p + (size_t)i * NRED + r);
        }
        block_reduce<NT, NRED>(s, scratch);
        if (threadIdx.x == 0) fin.finish_member(b, s);
    }
    if (threadIdx.x == 0) {
        fin.finish_all();
        *rc.counter = 0u;
    }
}

// (H f)_{l,j} from the five/seven neighbouring values (Eq. 11).  d = l(l+1)/(2r^2) - Z/r + kinetic diagonal.
template <int FD>
__device__ __forceinline__ double2 h_point(const GridDev &g, double d, double er, double cm, double cp,
                                           double2 f, double2 fm1, double2 fp1, double2 fm2, double2 fp2,
                                           double2 lo, double2 up) {
    double2 h;
    double kx = g.c1 * (fp1.x + fm1.x), ky = g.c1 * (fp1.y + fm1.y);
    if (FD == 5) {
        kx = fma(g.c2, fp2.x + fm2.x, kx);
        ky = fma(g.c2, fp2.y + fm2.y, ky);
    }
    const double cx = fma(cp, up.x, cm * lo.x), cy = fma(cp, up.y, cm * lo.y);
    h.x = fma(er, cx, fma(d, f.x, kx));
    h.y = fma(er, cy, fma(d, f.y, ky));
    return h;
}

// Velocity-gauge coupling added to h (Eq. 12 in reading R-V2; afield = A(t)):
//   -i A [ c_{l-1} (d/dr - l/r) f_{l-1} + c_l (d/dr + (l+1)/r) f_{l+1} ],  d/dr by P:119 Eq. 14 (R-V1).
// c points at (l, j) of a shared-memory tile with row pitch `pitch` that holds the rows l-1 and l+1 with their radial halo.
template <int FD>
__device__ __forceinline__ void vg_couple(const GridDev &g, const double2 *c, int pitch, int l, double rinv, double cm,
                                          double cp, double afield, double2 lo, double2 up, double2 &h) {
    const double2 *cl_ = c - pitch, *cu_ = c + pitch;
    double dlx, dly, dux, duy;
    if (FD == 3) {
        const double w = 0.5 / g.dr;
        dlx = w * (cl_[1].x - cl_[-1].x); dly = w * (cl_[1].y - cl_[-1].y);
        dux = w * (cu_[1].x - cu_[-1].x); duy = w * (cu_[1].y - cu_[-1].y);
    } else {
        const double w = 1.0 / (12.0 * g.dr);
        dlx = w * (8.0 * (cl_[1].x - cl_[-1].x) - (cl_[2].x - cl_[-2].x));
        dly = w * (8.0 * (cl_[1].y - cl_[-1].y) - (cl_[2].y - cl_[-2].y));
        dux = w * (8.0 * (cu_[1].x - cu_[-1].x) - (cu_[2].x - cu_[-2].x));
        duy = w * (8.0 * (cu_[1].y - cu_[-1].y) - (cu_[2].y - cu_[-2].y));
    }
    const double sx = cm * (dlx - (double)l * rinv * lo.x) + cp * (dux + (double)(l + 1) * rinv * up.x);
    const double sy = cm * (dly - (double)l * rinv * lo.y) + cp * (duy + (double)(l + 1) * rinv * up.y);
    h.x = fma(afield, sy, h.x);              // -i (sx + i sy) = sy - i sx
    h.y = fma(-afield, sx, h.y);
}

}  // namespace tdse
