"""GPU parity on the OUTPUTS BASELINE.json's configs name (north star: "every config matches the oracle within the
stated tolerances"): CFG1's full pulse with norm / 1s / 2p / dipole logged every step, CFG2's adaptive Dormand-Prince
run at CFG2's own size, CFG5's final ionisation yield over every bound state of the discrete h_l.  The oracle is the
checker; inputs are the seeded generators of workloads.py.  Run with `-m gpu` on the B200 box.
"""
import numpy as np
import pytest

import oracle
from paper_1308_1856_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_PSI = 1e-9
TOL_OBS = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1308_1856_b200 import binding
    oracle.set_threads(8)
    return binding


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def all_bound_states(g, n_l, n_max=64):
    """Every eigenvector of the discrete h_l, l = 0..n_l-1, with E < 0 (SURVEY C7 / reading R-G23): input data."""
    ls, phis, ens = [], [], []
    for l in range(n_l):
        en, phi = oracle.bound_states(g, l, n_max, only_negative=True)
        assert len(en) < n_max                       # the search stopped at E >= 0, not at the cap
        ls += [l] * len(en)
        phis += list(phi)
        ens += list(en)
    return np.array(ls, dtype=np.int32), np.array(phis), np.array(ens)


def test_cfg1_full_pulse_every_step(B):
    """CFG1 as BASELINE.json states it -- hydrogen from the (discrete) 1s state, 8 x 500, 3-point, the whole 2-cycle
    pulse, Taylor-4 at dt_eff (about 66 000 steps), norm, 1s / 2p populations and dipole recorded EVERY step -- against
    the oracle: final wavefunction to 1e-9, every logged norm and population to 1e-10, dipole and acceleration to
    1e-9 of their scale (Eq. 25, Eq. 34, Eq. 36; P:371 column list)."""
    c = wl.config("cfg1")
    g = oracle.make_grid(c["n_r"], c["dr"], c["n_l"], c["fd_order"])
    h = B.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"])
    _, phi0 = oracle.bound_states(g, 0, 1)
    _, phi1 = oracle.bound_states(g, 1, 1)
    st = (np.array([0, 1], dtype=np.int32), np.array([phi0[0], phi1[0]]))
    pulses = wl.pulses(c)
    h.set_pulse(pulses)
    h.set_bound_states(*st)
    psi0 = wl.ground_state(c, phi0[0])
    dt = wl.dt_eff(c)
    nsteps = int(round(c["t_pulse"] / dt))
    assert nsteps > 60000 and abs(nsteps * dt - c["t_pulse"]) < 1e-9
    h.set_state(psi0)
    h.step_taylor(c["order"], 0.0, dt, nsteps, 1)
    got, rows = h.get_state(), h.obs_log()
    ref, rrows = oracle.step_taylor(g, pulses, psi0, c["order"], 0.0, dt, nsteps, states=st, obs_every=1)
    assert rows.shape == rrows.shape == (nsteps, 1, 5)
    assert rel_l2(got, ref) <= TOL_PSI
    assert np.max(np.abs(rows[..., 0] - rrows[..., 0])) <= TOL_OBS            # norm, every step
    assert np.max(np.abs(rows[..., 3:] - rrows[..., 3:])) <= TOL_OBS          # 1s and 2p populations, every step
    for k in (1, 2):                                                          # dipole, acceleration
        assert np.max(np.abs(rows[..., k] - rrows[..., k])) <= 1e-9 * max(1.0, float(np.max(np.abs(rrows[..., k]))))
    # the run did something: the pulse moved population out of 1s and the norm stayed 1 (P10)
    assert rrows[-1, 0, 3] < 0.9999 and abs(rrows[-1, 0, 0] - 1.0) <= 1e-10
    assert np.max(np.abs(rrows[..., 1])) > 1e-2
    h.close()


@pytest.mark.parametrize("persist", [1, 0])
def test_cfg2_adaptive_rk45_full_size(B, persist):
    """CFG2's second propagator at CFG2's own size (4000 x 32, 5-point): embedded Dormand-Prince 5(4), rtol 1e-8,
    adaptive dt over a 0.05 au window at the pulse peak, as the persistent cooperative kernel (the default at this size)
    and stage by stage.  Protocol R-G20: the oracle replays the accepted-dt sequence of the CUDA run, must itself find
    err <= 1.05 on every step, and the final states agree to 1e-9."""
    c = wl.config("cfg2")
    g = oracle.make_grid(c["n_r"], c["dr"], c["n_l"], c["fd_order"])
    h = B.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"])
    h.set_option("rk45_persist", persist)
    pulses = wl.pulses(c)
    h.set_pulse(pulses)
    psi0 = wl.populated_state(c)
    t0 = 0.5 * c["t_pulse"]
    t1 = t0 + 0.05
    h.set_state(psi0)
    info = h.step_rk45(t0, t1, 1e-5, c["rtol"])
    assert h.rk45_was_persistent() == bool(persist)
    got = h.get_state()
    assert info["n_accept"] > 500 and len(info["dt"]) == info["n_accept"]     # stability-limited: dt ~ 1/rho(H)
    assert abs(np.sum(info["dt"]) - (t1 - t0)) <= 1e-12
    assert np.all(info["err"] <= 1.0)
    ref, rinfo = oracle.step_rk45(g, pulses, psi0, t0, t1, 1e-5, c["rtol"], dt_replay=info["dt"])
    assert np.max(rinfo["err"]) <= 1.05
    assert rel_l2(got, ref) <= TOL_PSI
    for l in range(c["n_l"]):
        assert np.linalg.norm(got[0, l] - ref[0, l]) <= TOL_PSI * max(np.linalg.norm(ref[0, l]), 1e-3)
    obs = h.observables(t1)
    robs = oracle.observables(g, ref, [oracle.pulse_E(pulses[0], t1)])
    assert abs(obs[0, 0] - robs[0, 0]) <= TOL_OBS
    h.close()


def test_cfg5_ionisation_yield_over_all_bound_states(B):
    """CFG5's stated output: final ionisation yield 1 - sum of bound populations per member, the sum running over EVERY
    eigenvector of the discrete h_l, l = 0..15, with E < 0 (94 vectors of length 2000 in this box; reading R-G23).  A slice
    of 8 members of the intensity scan, 300 Taylor-6 steps at the pulse peak from the populated state: every population
    and the yield against the oracle to 1e-10 (Eq. 25)."""
    c = wl.config("cfg5")
    full = wl.pulses(c)
    members = [0, 1, 31, 64, 100, 128, 200, 255]
    c8 = wl.config("cfg5", batch=len(members))
    pulses = [full[m] for m in members]
    g = oracle.make_grid(c8["n_r"], c8["dr"], c8["n_l"], c8["fd_order"], batch=len(members))
    ls, phis, ens = all_bound_states(g, c8["n_l"])
    assert 80 <= len(ls) <= 260 and np.all(ens < 0)          # 94 on this box (r_max = 200)
    h = B.Tdse(c8["n_r"], c8["dr"], c8["n_l"], c8["fd_order"], batch=len(members))
    h.set_pulse(pulses)
    h.set_bound_states(ls, phis)
    psi0 = wl.populated_state(c8)
    dt = wl.dt_eff(c)
    nsteps = 300
    t0 = wl.window(c, nsteps, dt)
    h.set_state(psi0)
    h.step_taylor(c["order"], t0, dt, nsteps, 100)          # three logged row blocks on the way (many-state log path)
    assert h.taylor_was_blocked()
    t1 = t0 + nsteps * dt
    got, rows = h.get_state(), h.obs_log()
    final = h.observables(t1)
    yld = h.ionisation_yield()
    ref, rrows = oracle.step_taylor(g, pulses, psi0, c["order"], t0, dt, nsteps, states=(ls, phis), obs_every=100)
    assert rel_l2(got, ref) <= TOL_PSI
    assert rows.shape == rrows.shape == (3, len(members), 3 + len(ls))
    assert np.max(np.abs(rows[..., 0] - rrows[..., 0])) <= TOL_OBS
    assert np.max(np.abs(rows[..., 3:] - rrows[..., 3:])) <= TOL_OBS
    assert np.max(np.abs(final[:, 3:] - rrows[-1, :, 3:])) <= TOL_OBS         # every population of every member
    ryld = 1.0 - np.sum(rrows[-1, :, 3:], axis=1)
    assert np.max(np.abs(yld - ryld)) <= TOL_OBS
    assert np.all(ryld > 1e-3) and np.all(ryld < 1.0)                         # the wavepackets are mostly continuum
    h.close()
