"""Thin ctypes binding of libtdse_b200.so (include/tdse.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used here for device memory and
streams only.  There is no CPU fallback: if the library is missing or a call fails, this module raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libtdse_b200.so")

TDSE_OK = 0
ERRORS = {-1: "TDSE_ERR_ARG", -2: "TDSE_ERR_ALLOC", -3: "TDSE_ERR_CUDA", -4: "TDSE_ERR_NONFINITE",
          -5: "TDSE_ERR_UNSUPPORTED", -6: "TDSE_ERR_TOO_LARGE"}

# every symbol include/tdse.h declares
SYMBOLS = ["tdse_create", "tdse_destroy", "tdse_set_option", "tdse_set_pulse", "tdse_set_bound_states",
           "tdse_set_cutoff", "tdse_set_state", "tdse_get_state", "tdse_apply_H", "tdse_set_absorber", "tdse_bound_population", "tdse_step_taylor", "tdse_step_imag", "tdse_energy_log", "tdse_step_rk4", "tdse_step_rk", "tdse_rk_sigma",
           "tdse_step_lanczos", "tdse_step_rk45", "tdse_observables", "tdse_obs_log", "tdse_dt_log",
           "tdse_lanczos_info", "tdse_ionisation_yield", "tdse_graph_instantiations", "tdse_launch_count", "tdse_taylor_was_blocked", "tdse_rk45_was_persistent", "tdse_taylor_plan", "tdse_observables_noalloc", "tdse_strerror", "tdse_version"]


class TdseError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__(f"{what}: {ERRORS.get(code, code)} ({strerror(code)})")


class Grid(C.Structure):
    _fields_ = [("n_r", C.c_int), ("dr", C.c_double), ("n_l", C.c_int), ("fd_order", C.c_int), ("gauge", C.c_int),
                ("z_nuc", C.c_double), ("batch", C.c_int)]


class Pulse(C.Structure):
    _fields_ = [("e0", C.c_double), ("omega", C.c_double), ("n_cycles", C.c_double), ("cep", C.c_double),
                ("kind", C.c_int)]


_lib = None


def lib():
    """Load the CUDA library; fail loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1308_1856_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, dp, ip, lp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_long)
        L.tdse_create.argtypes = [C.POINTER(Grid), C.POINTER(vp)]
        L.tdse_destroy.argtypes = [vp]
        L.tdse_destroy.restype = None
        L.tdse_set_option.argtypes = [vp, C.c_char_p, C.c_double]
        L.tdse_set_pulse.argtypes = [vp, C.POINTER(Pulse)]
        L.tdse_set_bound_states.argtypes = [vp, C.c_int, ip, dp]
        L.tdse_set_state.argtypes = [vp, vp, C.c_int, vp]
        L.tdse_get_state.argtypes = [vp, vp, C.c_int, vp]
        L.tdse_apply_H.argtypes = [vp, vp, vp, dp, vp]
        L.tdse_step_taylor.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_long, C.c_int, vp]
        L.tdse_step_imag.argtypes = [vp, C.c_int, C.c_double, C.c_long, vp]
        L.tdse_step_rk.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_long, C.c_int, vp]
        L.tdse_rk_sigma.argtypes = [vp, C.POINTER(C.c_double), vp]
        L.tdse_set_absorber.argtypes = [vp, C.c_double, C.c_int]
        L.tdse_set_cutoff.argtypes = [vp, C.c_double]
        L.tdse_bound_population.argtypes = [vp, C.c_double, C.POINTER(C.c_double), vp]
        L.tdse_energy_log.argtypes = [vp, C.POINTER(C.c_double), C.c_long, vp]
        L.tdse_step_rk4.argtypes = [vp, C.c_double, C.c_double, C.c_long, C.c_int, vp]
        L.tdse_step_lanczos.argtypes = [vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_long, C.c_int, vp]
        L.tdse_step_rk45.argtypes = [vp, C.c_double, C.c_double, C.c_double, C.c_double, dp, C.c_long, lp, lp, vp]
        L.tdse_observables.argtypes = [vp, C.c_double, dp, vp]
        L.tdse_obs_log.argtypes = [vp, dp, C.c_long, lp]
        L.tdse_dt_log.argtypes = [vp, dp, dp, C.c_long, lp]
        L.tdse_lanczos_info.argtypes = [vp, dp, dp, dp, ip, ip]
        L.tdse_launch_count.argtypes = [vp]
        L.tdse_launch_count.restype = C.c_long
        L.tdse_graph_instantiations.argtypes = [vp]
        L.tdse_graph_instantiations.restype = C.c_long
        L.tdse_ionisation_yield.argtypes = [vp, dp, vp]
        L.tdse_observables_noalloc.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, vp, vp, vp]
        L.tdse_taylor_plan.argtypes = [vp, ip, ip, ip]
        L.tdse_rk45_was_persistent.argtypes = [vp]
        L.tdse_rk45_was_persistent.restype = C.c_int
        L.tdse_taylor_was_blocked.argtypes = [vp]
        L.tdse_strerror.argtypes = [C.c_int]
        L.tdse_strerror.restype = C.c_char_p
        L.tdse_version.restype = C.c_char_p
        _lib = L
    return _lib


def strerror(code):
    return lib().tdse_strerror(int(code)).decode()


def version():
    return lib().tdse_version().decode()


def observables_noalloc(psi_dev, dr, z_nuc, e_now_dev, out_dev, stream=None):
    """{norm, <z>, <z''>} of psi_dev (torch complex128 CUDA tensor [batch][n_l][n_r]) into out_dev (float64 CUDA tensor
    [batch][3]) through the entry point that allocates nothing; e_now_dev: float64 CUDA tensor [batch] or None."""
    batch, n_l, n_r = psi_dev.shape
    assert psi_dev.is_cuda and psi_dev.is_contiguous() and out_dev.is_cuda and out_dev.is_contiguous()
    assert out_dev.numel() == 3 * batch and (e_now_dev is None or (e_now_dev.is_cuda and e_now_dev.numel() == batch))
    _check(lib().tdse_observables_noalloc(C.c_void_p(psi_dev.data_ptr()), int(n_r), int(n_l), int(batch), float(dr),
                                          float(z_nuc), C.c_void_p(e_now_dev.data_ptr() if e_now_dev is not None else None),
                                          C.c_void_p(out_dev.data_ptr()), _stream(stream)), "tdse_observables_noalloc")
    return out_dev


def _check(rc, what):
    if rc != TDSE_OK:
        raise TdseError(rc, what)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _stream(stream):
    """torch stream / raw int / None -> void*."""
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


class Tdse:
    """One handle = one grid (n_r, dr, n_l, fd_order, batch) with its state resident on the GPU."""

    def __init__(self, n_r, dr, n_l, fd_order, z_nuc=1.0, batch=1, gauge=0):
        self.grid = Grid(int(n_r), float(dr), int(n_l), int(fd_order), int(gauge), float(z_nuc), int(batch))
        self._h = C.c_void_p()
        self.n_states = 0
        _check(lib().tdse_create(C.byref(self.grid), C.byref(self._h)), "tdse_create")

    # -- lifetime
    def close(self):
        if self._h:
            lib().tdse_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def shape(self):
        return (self.grid.batch, self.grid.n_l, self.grid.n_r)

    # -- configuration
    def set_option(self, key, value):
        _check(lib().tdse_set_option(self._h, key.encode(), float(value)), f"tdse_set_option({key})")

    def set_pulse(self, pulses):
        """pulses: one (e0, omega, n_cycles, cep[, kind]) tuple for all members, or a list of batch tuples."""
        b = self.grid.batch
        if isinstance(pulses, tuple) and not isinstance(pulses[0], (tuple, list)):
            pulses = [pulses] * b
        if len(pulses) != b:
            raise ValueError("need one pulse per member")
        arr = (Pulse * b)()
        for i, p in enumerate(pulses):
            arr[i] = Pulse(float(p[0]), float(p[1]), float(p[2]), float(p[3]), int(p[4]) if len(p) > 4 else 0)
        _check(lib().tdse_set_pulse(self._h, arr), "tdse_set_pulse")

    def set_bound_states(self, l_of_state, phi):
        l_arr = np.ascontiguousarray(l_of_state, dtype=np.int32)
        phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(len(l_arr), self.grid.n_r)
        _check(lib().tdse_set_bound_states(self._h, len(l_arr), l_arr.ctypes.data_as(C.POINTER(C.c_int)), _dp(phi)),
               "tdse_set_bound_states")
        self.n_states = len(l_arr)

    # -- state
    def set_state(self, psi, stream=None, pinned_async=False):
        """psi: numpy complex128 array (host) or torch complex128 CUDA tensor, shape [batch][n_l][n_r].
        pinned_async: the numpy array lives in pinned memory and the copy is left asynchronous on the stream."""
        if isinstance(psi, np.ndarray):
            a = np.ascontiguousarray(psi, dtype=np.complex128)
            assert a.size == int(np.prod(self.shape))
            assert not pinned_async or a is psi or a.ctypes.data == psi.ctypes.data
            _check(lib().tdse_set_state(self._h, C.c_void_p(a.ctypes.data), 2 if pinned_async else 0, _stream(stream)),
                   "tdse_set_state")
        else:
            t = psi.contiguous()
            assert t.is_cuda and t.numel() == int(np.prod(self.shape)) and t.element_size() == 16
            _check(lib().tdse_set_state(self._h, C.c_void_p(t.data_ptr()), 1, _stream(stream)), "tdse_set_state")

    def get_state(self, out=None, stream=None, pinned_async=False):
        """Returns a numpy array (out=None or numpy) or fills the given torch CUDA tensor.
        pinned_async: `out` is a pinned numpy array; the copy is left asynchronous on the stream."""
        if out is None:
            out = np.empty(self.shape, dtype=np.complex128)
        if isinstance(out, np.ndarray):
            assert out.flags.c_contiguous and out.dtype == np.complex128
            _check(lib().tdse_get_state(self._h, C.c_void_p(out.ctypes.data), 2 if pinned_async else 0, _stream(stream)),
                   "tdse_get_state")
        else:
            assert out.is_cuda and out.is_contiguous() and out.element_size() == 16
            _check(lib().tdse_get_state(self._h, C.c_void_p(out.data_ptr()), 1, _stream(stream)), "tdse_get_state")
        return out

    # -- the hot path
    def apply_H(self, psi_dev, out_dev, e_field, stream=None):
        """out_dev = H(e_field) psi_dev; both torch complex128 CUDA tensors of shape [batch][n_l][n_r]."""
        e = np.ascontiguousarray(np.broadcast_to(np.asarray(e_field, dtype=np.float64), (self.grid.batch,)))
        assert psi_dev.is_cuda and out_dev.is_cuda and psi_dev.is_contiguous() and out_dev.is_contiguous()
        assert psi_dev.numel() == out_dev.numel() == int(np.prod(self.shape))
        _check(lib().tdse_apply_H(self._h, C.c_void_p(psi_dev.data_ptr()), C.c_void_p(out_dev.data_ptr()), _dp(e),
                                  _stream(stream)), "tdse_apply_H")
        return out_dev

    def step_taylor(self, order, t0, dt, nsteps, obs_every=0, stream=None):
        _check(lib().tdse_step_taylor(self._h, int(order), float(t0), float(dt), int(nsteps), int(obs_every),
                                      _stream(stream)), "tdse_step_taylor")

    def set_cutoff(self, lam):
        """Centrifugal inner cut-off Lambda (an extension beyond the paper); 0 removes it."""
        _check(lib().tdse_set_cutoff(self._h, float(lam)), "tdse_set_cutoff")

    def set_absorber(self, r_b, p):
        _check(lib().tdse_set_absorber(self._h, float(r_b), int(p)), "tdse_set_absorber")

    def bound_population(self, r_b, stream=None):
        out = np.zeros(self.grid.batch)
        _check(lib().tdse_bound_population(self._h, float(r_b), out.ctypes.data_as(C.POINTER(C.c_double)),
                                           _stream(stream)), "tdse_bound_population")
        return out

    def step_imag(self, order, dt, nsteps, stream=None):
        """Imaginary-time propagation with re-normalisation; returns the energy estimates [nsteps][batch]."""
        _check(lib().tdse_step_imag(self._h, int(order), float(dt), int(nsteps), _stream(stream)), "tdse_step_imag")
        en = np.zeros((max(int(nsteps), 1), self.grid.batch))
        _check(lib().tdse_energy_log(self._h, en.ctypes.data_as(C.POINTER(C.c_double)), int(nsteps), _stream(stream)),
               "tdse_energy_log")
        return en[:int(nsteps)]

    def step_rk4(self, t0, dt, nsteps, obs_every=0, stream=None):
        _check(lib().tdse_step_rk4(self._h, float(t0), float(dt), int(nsteps), int(obs_every), _stream(stream)),
               "tdse_step_rk4")

    RK_METHODS = {"rk4": 0, "dormandprince": 1, "euler": 2, "rkf": 3, "cashkarp": 4, "merson": 5}

    def step_rk(self, method, t0, dt, nsteps, obs_every=0, stream=None):
        """Fixed-step Runge-Kutta with one of the paper's methods; returns the passive error sums sigma[batch]."""
        _check(lib().tdse_step_rk(self._h, int(self.RK_METHODS[method]), float(t0), float(dt), int(nsteps), int(obs_every),
                                  _stream(stream)), "tdse_step_rk")
        sig = np.zeros(self.grid.batch)
        _check(lib().tdse_rk_sigma(self._h, sig.ctypes.data_as(C.POINTER(C.c_double)), _stream(stream)), "tdse_rk_sigma")
        return sig

    def step_lanczos(self, krylov_dim, taylor_order, t0, dt, nsteps, obs_every=0, stream=None):
        _check(lib().tdse_step_lanczos(self._h, int(krylov_dim), int(taylor_order), float(t0), float(dt),
                                       int(nsteps), int(obs_every), _stream(stream)), "tdse_step_lanczos")

    def step_rk45(self, t0, t_end, dt_init, rtol, dt_replay=None, stream=None):
        """Returns dict(n_accept, n_reject, dt[], err[])."""
        na, nr = C.c_long(0), C.c_long(0)
        rep, n_rep = None, 0
        if dt_replay is not None:
            rep_arr = np.ascontiguousarray(dt_replay, dtype=np.float64)
            rep, n_rep = _dp(rep_arr), len(rep_arr)
        _check(lib().tdse_step_rk45(self._h, float(t0), float(t_end), float(dt_init), float(rtol), rep, n_rep,
                                    C.byref(na), C.byref(nr), _stream(stream)), "tdse_step_rk45")
        n = C.c_long(0)
        dt = np.zeros(max(na.value, 1))
        err = np.zeros(max(na.value, 1))
        _check(lib().tdse_dt_log(self._h, _dp(dt), _dp(err), len(dt), C.byref(n)), "tdse_dt_log")
        k = min(n.value, len(dt))
        return {"n_accept": na.value, "n_reject": nr.value, "dt": dt[:k].copy(), "err": err[:k].copy()}

    # -- observables
    def observables(self, t, stream=None):
        out = np.zeros((self.grid.batch, 3 + self.n_states))
        _check(lib().tdse_observables(self._h, float(t), _dp(out), _stream(stream)), "tdse_observables")
        return out

    def obs_log(self):
        rows = C.c_long(0)
        _check(lib().tdse_obs_log(self._h, None, 0, C.byref(rows)), "tdse_obs_log")
        out = np.zeros((max(rows.value, 1), self.grid.batch, 3 + self.n_states))
        if rows.value > 0:
            _check(lib().tdse_obs_log(self._h, _dp(out), rows.value, C.byref(rows)), "tdse_obs_log")
        return out[:rows.value]

    def lanczos_info(self, krylov_dim):
        b, k = self.grid.batch, int(krylov_dim)
        alpha, beta = np.zeros((b, k)), np.zeros((b, k))
        coef = np.zeros((b, k), dtype=np.complex128)
        m, ns = np.zeros(b, dtype=np.int32), np.zeros(b, dtype=np.int32)
        _check(lib().tdse_lanczos_info(self._h, _dp(alpha), _dp(beta), _dp(coef.view(np.float64)),
                                       m.ctypes.data_as(C.POINTER(C.c_int)), ns.ctypes.data_as(C.POINTER(C.c_int))),
               "tdse_lanczos_info")
        return {"alpha": alpha, "beta": beta, "coef": coef, "m": m, "n_sub": ns}

    def ionisation_yield(self, stream=None):
        """1 - sum of the bound-state populations of the current state, per member."""
        out = np.zeros(self.grid.batch)
        _check(lib().tdse_ionisation_yield(self._h, _dp(out), _stream(stream)), "tdse_ionisation_yield")
        return out

    def launch_count(self):
        return int(lib().tdse_launch_count(self._h))

    def graph_instantiations(self):
        return int(lib().tdse_graph_instantiations(self._h))

    def taylor_was_blocked(self):
        return bool(lib().tdse_taylor_was_blocked(self._h))

    def taylor_plan(self):
        """dict(variant, steps_per_launch, ctas) of the register-patch kernel the last step call ran with."""
        v, k, n = C.c_int(-1), C.c_int(0), C.c_int(0)
        _check(lib().tdse_taylor_plan(self._h, C.byref(v), C.byref(k), C.byref(n)), "tdse_taylor_plan")
        return {"variant": v.value, "steps_per_launch": k.value, "ctas": n.value}

    def rk45_was_persistent(self):
        return bool(lib().tdse_rk45_was_persistent(self._h))

    def taylor_kernel(self):
        """0: one kernel per order, 3 / 4: all orders in one pass (direct loads / TMA tile fetches)."""
        return int(lib().tdse_taylor_was_blocked(self._h))
