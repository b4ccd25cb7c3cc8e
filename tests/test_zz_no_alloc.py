"""GPU test of tdse_observables_noalloc, the entry point that allocates nothing (scratch in a file-scope device array):
its output against the existing path (tdse_observables of a handle) on the same state, on two calls in a row -- the
second with another state, so that a stale counter or partial sum left in the shared scratch by the first would show.
Collected last on purpose (the suite runs with pytest -x).  Run with `-m gpu` on the B200 box.
"""
import numpy as np
import pytest

import oracle
from paper_1308_1856_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_OBS = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1308_1856_b200 import binding
    return binding


def existing_path(B, c, psi, pulses, t):
    h = B.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"], batch=c["batch"])
    h.set_pulse(pulses)
    h.set_state(psi)
    ref = h.observables(t)[:, :3].copy()
    h.close()
    return ref


@pytest.mark.parametrize("name,kw", [("cfg5", dict(batch=24)), ("cfg1", dict(batch=3, n_r=333, n_l=11)),
                                     ("cfg3", dict(n_r=1000))])
def test_noalloc_observables_match_the_handle_path_twice(B, name, kw):
    import torch
    c = wl.config(name, **kw)
    pulses = wl.pulses(c)
    t = 0.37 * c["t_pulse"]
    e_now = torch.tensor([oracle.pulse_E(p, t) for p in pulses], dtype=torch.float64, device="cuda")
    out = torch.full((c["batch"], 3), float("nan"), dtype=torch.float64, device="cuda")
    for call, psi in enumerate((wl.populated_state(c), wl.random_state(c, seed_extra=5))):
        ref = existing_path(B, c, psi, pulses, t)
        d_psi = torch.from_numpy(psi).cuda()
        out.fill_(float("nan"))
        mem0 = torch.cuda.memory_allocated()
        B.observables_noalloc(d_psi, c["dr"], c.get("z_nuc", 1.0), e_now, out)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == mem0
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got)), call
        assert np.max(np.abs(got[:, 0] - ref[:, 0])) <= TOL_OBS * max(1.0, float(np.max(np.abs(ref[:, 0])))), call
        for k in (1, 2):
            assert np.max(np.abs(got[:, k] - ref[:, k])) <= TOL_OBS * max(1.0, float(np.max(np.abs(ref[:, k])))), call
    # field-free: e_now = NULL drops the -E(t) term only
    B.observables_noalloc(d_psi, c["dr"], c.get("z_nuc", 1.0), None, out)
    torch.cuda.synchronize()
    free = out.cpu().numpy()
    assert np.max(np.abs(free[:, :2] - got[:, :2])) == 0.0
    assert np.max(np.abs(free[:, 2] - (got[:, 2] + e_now.cpu().numpy()))) <= 1e-12 * max(1.0, float(np.max(np.abs(got[:, 2]))))


def test_noalloc_rejects_sizes_beyond_the_scratch(B):
    import torch
    psi = torch.zeros((2, 2, 8), dtype=torch.complex128, device="cuda")
    out = torch.zeros((2, 3), dtype=torch.float64, device="cuda")
    L = B.lib()
    import ctypes as C
    args = lambda n_r, n_l, batch: (C.c_void_p(psi.data_ptr()), n_r, n_l, batch, 0.1, 1.0, C.c_void_p(None),
                                    C.c_void_p(out.data_ptr()), C.c_void_p(0))
    assert L.tdse_observables_noalloc(*args(8, 2, 4097)) == -6                 # TDSE_ERR_TOO_LARGE: members
    assert L.tdse_observables_noalloc(*args(256 * 40000, 2, 1)) == -6          # ... CTAs of one launch
    assert L.tdse_observables_noalloc(*args(8, 2, 0)) == -1                    # TDSE_ERR_ARG
    assert "scratch" in B.strerror(-6)
    torch.cuda.synchronize()
