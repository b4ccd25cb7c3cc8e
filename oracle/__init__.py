"""CPU oracle for the CLTDSE hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front-end of oracle/tdse_oracle.cpp (see tdse_oracle.h for the citations).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package; it imports nothing from paper_1308_1856_b200.
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = None


class Grid(C.Structure):
    _fields_ = [("n_r", C.c_int), ("dr", C.c_double), ("n_l", C.c_int), ("fd_order", C.c_int),
                ("z_nuc", C.c_double), ("batch", C.c_int), ("r_offset", C.c_double), ("gauge", C.c_int),
                ("cutoff_lambda", C.c_double)]


class Pulse(C.Structure):
    _fields_ = [("e0", C.c_double), ("omega", C.c_double), ("n_cycles", C.c_double), ("cep", C.c_double),
                ("kind", C.c_int)]


class Obs(C.Structure):
    _fields_ = [("n_states", C.c_int), ("l_of_state", C.POINTER(C.c_int)), ("phi", C.POINTER(C.c_double)),
                ("obs_every", C.c_int), ("obs_out", C.POINTER(C.c_double))]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_pulse_E.restype = C.c_double
        _lib.oracle_pulse_E.argtypes = [C.POINTER(Pulse), C.c_double]
        _lib.oracle_pulse_A.restype = C.c_double
        _lib.oracle_pulse_A.argtypes = [C.POINTER(Pulse), C.c_double]
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_grid(n_r, dr, n_l, fd_order, z_nuc=1.0, batch=1, r_offset=0.0, gauge=0, cutoff_lambda=0.0):
    """cutoff_lambda > 0: centrifugal inner cut-off (an extension beyond the paper, see tdse_oracle.h)."""
    return Grid(int(n_r), float(dr), int(n_l), int(fd_order), float(z_nuc), int(batch), float(r_offset), int(gauge),
                float(cutoff_lambda))


def _pulses(g, pulses):
    """pulses: iterable of (e0, omega, n_cycles, cep[, kind]) per member (or one tuple for all)."""
    if isinstance(pulses, tuple) and not isinstance(pulses[0], (tuple, list)):
        pulses = [pulses] * g.batch
    assert len(pulses) == g.batch
    arr = (Pulse * g.batch)()
    for i, p in enumerate(pulses):
        arr[i] = Pulse(float(p[0]), float(p[1]), float(p[2]), float(p[3]), int(p[4]) if len(p) > 4 else 0)
    return arr


def _state(g, psi):
    psi = np.ascontiguousarray(psi, dtype=np.complex128).reshape(g.batch, g.n_l, g.n_r).copy()
    return psi


def _obs(g, states, obs_every, nsteps):
    """states: None or (l_of_state int array, phi [n][n_r]) -> (Obs struct or None, out array, keepalive)."""
    if not obs_every:
        return None, None, None
    if states is None:
        l_arr = np.zeros(0, dtype=np.int32)
        phi = np.zeros((0, g.n_r))
    else:
        l_arr = np.ascontiguousarray(states[0], dtype=np.int32)
        phi = np.ascontiguousarray(states[1], dtype=np.float64).reshape(len(l_arr), g.n_r)
    n_blocks = nsteps // obs_every
    out = np.zeros((n_blocks, g.batch, 3 + len(l_arr)))
    o = Obs(len(l_arr), l_arr.ctypes.data_as(C.POINTER(C.c_int)), _dp(phi), int(obs_every), _dp(out))
    return o, out, (l_arr, phi)


def set_threads(n):
    lib().oracle_set_threads(int(n))


def _pulse1(pulse):
    return Pulse(float(pulse[0]), float(pulse[1]), float(pulse[2]), float(pulse[3]), int(pulse[4]) if len(pulse) > 4 else 0)


def pulse_E(pulse, t):
    p = _pulse1(pulse)
    return lib().oracle_pulse_E(C.byref(p), float(t))


def pulse_A(pulse, t):
    """A(t) with E = -dA/dt (kind 1 pulses; NaN for kind 0)."""
    p = _pulse1(pulse)
    return lib().oracle_pulse_A(C.byref(p), float(t))


def gl5_field_integral(pulse, ta, tb):
    """int_ta^tb E dtau by one 5-point Gauss-Legendre rule."""
    p = _pulse1(pulse)
    f = lib().oracle_gl5_field_integral
    f.restype = C.c_double
    f.argtypes = [C.POINTER(Pulse), C.c_double, C.c_double]
    return f(C.byref(p), float(ta), float(tb))


def vecpot_running(pulse, t0, dt, nsteps):
    """A(t0 + n dt), n = 0..nsteps, by the running quadrature of P:188 on the field of `pulse`."""
    p = _pulse1(pulse)
    out = np.zeros(int(nsteps) + 1)
    rc = lib().oracle_vecpot_running(C.byref(p), C.c_double(t0), C.c_double(dt), C.c_long(nsteps), _dp(out))
    assert rc == 0, rc
    return out


def coupling(n_l):
    c = np.zeros(n_l)
    lib().oracle_coupling(int(n_l), _dp(c))
    return c


def apply_H(g, psi, e_field):
    psi = _state(g, psi)
    e = np.ascontiguousarray(np.broadcast_to(np.asarray(e_field, dtype=np.float64), (g.batch,)))
    out = np.empty_like(psi)
    rc = lib().oracle_apply_H(C.byref(g), _dp(psi.view(np.float64)), _dp(e), _dp(out.view(np.float64)))
    assert rc == 0, rc
    return out


def held_mask(g):
    """[n_l][n_r] bool: the points the centrifugal cut-off holds at zero."""
    m = np.zeros((g.n_l, g.n_r), dtype=bool)
    for l in range(g.n_l):
        for j in range(1, g.n_r + 1):
            if not lib().oracle_is_held(C.byref(g), l, j):
                break                      # held points of a row are its first ones
            m[l, j - 1] = True
    return m


def project(g, psi):
    psi = _state(g, psi)
    rc = lib().oracle_project(C.byref(g), _dp(psi.view(np.float64)))
    assert rc == 0, rc
    return psi


def dense_H(g, e_field):
    n = g.n_r * g.n_l
    h = np.zeros((n, n))
    rc = lib().oracle_dense_H(C.byref(g), C.c_double(e_field), _dp(h))
    assert rc == 0, rc
    return h


def bound_states(g, l, n_want, only_negative=False):
    en = np.zeros(n_want)
    phi = np.zeros((n_want, g.n_r))
    n = lib().oracle_bound_states(C.byref(g), int(l), int(n_want), int(bool(only_negative)), _dp(en), _dp(phi))
    assert n >= 0, n
    return en[:n].copy(), phi[:n].copy()


def observables(g, psi, e_now, states=None):
    psi = _state(g, psi)
    e = np.ascontiguousarray(np.broadcast_to(np.asarray(e_now, dtype=np.float64), (g.batch,)))
    if states is None:
        l_arr, phi = np.zeros(0, dtype=np.int32), np.zeros((0, g.n_r))
    else:
        l_arr = np.ascontiguousarray(states[0], dtype=np.int32)
        phi = np.ascontiguousarray(states[1], dtype=np.float64).reshape(len(l_arr), g.n_r)
    out = np.zeros((g.batch, 3 + len(l_arr)))
    rc = lib().oracle_observables(C.byref(g), _dp(psi.view(np.float64)), _dp(e), len(l_arr),
                                  l_arr.ctypes.data_as(C.POINTER(C.c_int)), _dp(phi), _dp(out))
    assert rc == 0, rc
    return out


def step_taylor(g, pulses, psi, order, t0, dt, nsteps, field_sample=0, states=None, obs_every=0):
    psi = _state(g, psi)
    pa = _pulses(g, pulses)
    o, out, keep = _obs(g, states, obs_every, nsteps)
    rc = lib().oracle_step_taylor(C.byref(g), pa, _dp(psi.view(np.float64)), int(order), C.c_double(t0),
                                  C.c_double(dt), C.c_long(nsteps), int(field_sample),
                                  C.byref(o) if o else None)
    assert rc == 0, rc
    return psi, out


def step_imag(g, psi, order, dt, nsteps):
    """Imaginary-time propagation with re-normalisation. Returns psi, energy[nsteps][batch]."""
    psi = _state(g, psi)
    en = np.zeros((max(nsteps, 1), g.batch))
    rc = lib().oracle_step_imag(C.byref(g), _dp(psi.view(np.float64)), int(order), C.c_double(dt), C.c_long(nsteps),
                                _dp(en))
    assert rc == 0, rc
    return psi, en[:nsteps]


def step_rk_fixed(g, pulses, psi, tableau, t0, dt, nsteps, states=None, obs_every=0):
    """tableau: 0 = ClassicRK4, 1 = DormandPrince (5th-order weights). Returns psi, err[nsteps], obs."""
    psi = _state(g, psi)
    pa = _pulses(g, pulses)
    o, out, keep = _obs(g, states, obs_every, nsteps)
    err = np.zeros(max(nsteps, 1))
    rc = lib().oracle_step_rk_fixed(C.byref(g), pa, _dp(psi.view(np.float64)), int(tableau), C.c_double(t0),
                                    C.c_double(dt), C.c_long(nsteps), _dp(err), C.byref(o) if o else None)
    assert rc == 0, rc
    return psi, err[:nsteps], out


RK_METHODS = {"rk4": 0, "dormandprince": 1, "euler": 2, "rkf": 3, "cashkarp": 4, "merson": 5}


def step_rk_method(g, pulses, psi, method, t0, dt, nsteps, states=None, obs_every=0):
    """Fixed-step propagation with one of the tableaux of P:796 and the passive error sum sigma[batch]."""
    psi = _state(g, psi)
    pa = _pulses(g, pulses)
    o, out, keep = _obs(g, states, obs_every, nsteps)
    sigma = np.zeros(g.batch)
    rc = lib().oracle_step_rk_sigma(C.byref(g), pa, _dp(psi.view(np.float64)), int(RK_METHODS[method]), C.c_double(t0),
                                    C.c_double(dt), C.c_long(nsteps), _dp(sigma), C.byref(o) if o else None)
    assert rc == 0, rc
    return psi, sigma, out


def step_rk4(g, pulses, psi, t0, dt, nsteps, states=None, obs_every=0):
    psi, _, out = step_rk_fixed(g, pulses, psi, 0, t0, dt, nsteps, states, obs_every)
    return psi, out


def step_rk45(g, pulses, psi, t0, t_end, dt_init, rtol, dt_max=0.0, dt_replay=None, max_log=1 << 20):
    """Returns psi, dict(n_accept, n_reject, dt[], err[])."""
    psi = _state(g, psi)
    pa = _pulses(g, pulses)
    na, nr = C.c_long(0), C.c_long(0)
    if dt_replay is not None:
        rep = np.ascontiguousarray(dt_replay, dtype=np.float64)
        max_log = max(len(rep), 1)
    dt_log, err_log = np.zeros(max_log), np.zeros(max_log)
    rc = lib().oracle_step_rk45(C.byref(g), pa, _dp(psi.view(np.float64)), C.c_double(t0), C.c_double(t_end),
                                C.c_double(dt_init), C.c_double(rtol), C.c_double(dt_max),
                                _dp(rep) if dt_replay is not None else None,
                                C.c_long(len(rep) if dt_replay is not None else 0),
                                C.byref(na), C.byref(nr), _dp(dt_log), _dp(err_log), C.c_long(max_log))
    assert rc == 0, rc
    n = min(na.value, max_log)
    return psi, {"n_accept": na.value, "n_reject": nr.value, "dt": dt_log[:n].copy(), "err": err_log[:n].copy()}


def step_lanczos(g, pulses, psi, krylov_dim, taylor_order, t0, dt, nsteps, field_sample=0, beta_tol=1e-12,
                 states=None, obs_every=0):
    psi = _state(g, psi)
    pa = _pulses(g, pulses)
    o, out, keep = _obs(g, states, obs_every, nsteps)
    rc = lib().oracle_step_lanczos(C.byref(g), pa, _dp(psi.view(np.float64)), int(krylov_dim), int(taylor_order),
                                   C.c_double(t0), C.c_double(dt), C.c_long(nsteps), int(field_sample),
                                   C.c_double(beta_tol), C.byref(o) if o else None)
    assert rc == 0, rc
    return psi, out


def lanczos_internals(g, psi, e_field, krylov_dim, taylor_order, dt, beta_tol=1e-12):
    """One member. Returns dict(m, q[K][L][N], alpha[K], beta[K], coef[K] complex, n_sub)."""
    assert g.batch == 1
    psi = _state(g, psi)
    K = int(krylov_dim)
    q = np.zeros((K, g.n_l, g.n_r), dtype=np.complex128)
    alpha, beta = np.zeros(K), np.zeros(K)
    coef = np.zeros(K, dtype=np.complex128)
    n_sub = C.c_int(0)
    m = lib().oracle_lanczos_internals(C.byref(g), _dp(psi.view(np.float64)), C.c_double(e_field), K,
                                       int(taylor_order), C.c_double(dt), C.c_double(beta_tol),
                                       _dp(q.view(np.float64)), _dp(alpha), _dp(beta),
                                       _dp(coef.view(np.float64)), C.byref(n_sub))
    assert m >= 1, m
    return {"m": m, "q": q, "alpha": alpha, "beta": beta, "coef": coef, "n_sub": n_sub.value}


# ---------------------------------------------------------------------------------------------------------------
# Absorbing boundary and spatial yields (plain numpy; Eq. 18, Eq. 26, Eq. 27-28)
# ---------------------------------------------------------------------------------------------------------------
def absorber_W(g, r_b, p, dt):
    """W(r_j) of P:146 Eq. 18, literally: (i/dt) ln{1 - cos^p[(pi/2)(1 - r/r_b)]} on r_j = j dr (complex)."""
    r = g.dr * np.arange(1, g.n_r + 1)
    arg = 1.0 - np.cos(0.5 * np.pi * (1.0 - r / r_b)) ** p
    with np.errstate(divide="ignore", invalid="ignore"):
        return (1j / dt) * np.log(arg.astype(np.complex128))


def absorber_mask(g, r_b, p):
    """exp(-i W dt) of Eq. 18 = 1 - cos^p[(pi/2)(1 - r/r_b)]: the factor one step of the imaginary potential
    multiplies the wavefunction by (reading R-G26: W enters as a split step after each propagator step, which is
    what the (i/dt) ln{...} form of Eq. 18 is built for); 0 for r >= r_b."""
    r = g.dr * np.arange(1, g.n_r + 1)
    m = 1.0 - np.cos(0.5 * np.pi * (1.0 - r / r_b)) ** p
    m[r >= r_b] = 0.0
    return m


def step_masked(step_fn, g, psi, mask, t0, dt, nsteps):
    """nsteps steps of `step_fn(psi, t_start, 1) -> psi`, each followed by psi *= mask (absorbing boundary)."""
    psi = np.array(psi, dtype=np.complex128, copy=True)
    for n in range(nsteps):
        psi = step_fn(psi, t0 + n * dt, 1)
        psi *= mask[None, None, :]
    return psi


def bound_population(g, psi, r_b):
    """p_b = sum_l int_0^{r_b} |f_l|^2 dr (Eq. 26; rectangle rule over r_j <= r_b, reading R-G27); the spatial
    ionisation yield is p_i = 1 - p_b (Eq. 27-28) when no absorber removes norm."""
    r = g.dr * np.arange(1, g.n_r + 1)
    psi = np.asarray(psi).reshape(g.batch, g.n_l, g.n_r)
    return g.dr * np.sum(np.abs(psi[:, :, r <= r_b]) ** 2, axis=(1, 2))
