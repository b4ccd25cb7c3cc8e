"""Seeded synthetic workloads shaped like the paper's hydrogen set-ups.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's
tests.  It holds no arithmetic of the method (no Hamiltonian, no propagator, no observable):
only shapes, unit conversions, pulse parameters, the step-size rule and seeded input states.

Citations: P:<n> = line n of the paper text; CFGn = BASELINE.json configs[n-1];
S1..S4 = the synthetic-input recipes stated in DESIGN.md ("Input recipe").
"""
import math

import numpy as np

AU_INTENSITY_W_CM2 = 3.50944758e16      # 1 au of intensity
NM_TO_OMEGA = 45.5633525                # omega(au) = 45.5633525 / lambda(nm)
MASK64 = (1 << 64) - 1


class SplitMix64:
    """Counter-based 64-bit generator (public-domain algorithm by S. Vigna), scalar."""

    def __init__(self, seed):
        self.x = seed & MASK64

    def next_u64(self):
        self.x = (self.x + 0x9E3779B97F4A7C15) & MASK64
        z = self.x
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        return z ^ (z >> 31)

    def uniform(self):                   # [0, 1): top 53 bits / 2^53
        return (self.next_u64() >> 11) / float(1 << 53)


def splitmix64_uniform(seed, n):
    """n uniforms in [0,1) from SplitMix64(seed), vectorised (same stream as the scalar class)."""
    with np.errstate(over="ignore"):
        k = np.arange(1, n + 1, dtype=np.uint64)
        z = np.uint64(seed & MASK64) + k * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) / float(1 << 53)


def e0_of_intensity(i_w_cm2):
    return math.sqrt(i_w_cm2 / AU_INTENSITY_W_CM2)


def omega_of_nm(lam_nm):
    return NM_TO_OMEGA / lam_nm


# name -> shape and method parameters (BASELINE.json configs, shapes table of SURVEY §8)
CONFIGS = {
    "tiny": dict(index=0, n_r=100, dr=0.2, n_l=3, fd_order=3, batch=1, propagator="taylor", order=4,
                 dt_cfg=0.004, lam_nm=800.0, intensity=1e14, n_cycles=2),
    "cfg1": dict(index=1, n_r=500, dr=0.2, n_l=8, fd_order=3, batch=1, propagator="taylor", order=4,
                 dt_cfg=0.01, lam_nm=800.0, intensity=1e14, n_cycles=2),
    "cfg2": dict(index=2, n_r=4000, dr=0.1, n_l=32, fd_order=5, batch=1, propagator="rk4", order=4,
                 dt_cfg=0.002, lam_nm=800.0, intensity=1e14, n_cycles=4, rtol=1e-8),
    "cfg3": dict(index=3, n_r=20000, dr=0.1, n_l=64, fd_order=5, batch=1, propagator="taylor", order=10,
                 dt_cfg=0.005, lam_nm=800.0, intensity=2e14, n_cycles=10),
    "cfg4": dict(index=4, n_r=40000, dr=0.1, n_l=128, fd_order=3, batch=1, propagator="lanczos", order=12,
                 krylov_dim=16, dt_cfg=0.02, lam_nm=1800.0, intensity=3e14, n_cycles=6),
    "cfg5": dict(index=5, n_r=2000, dr=0.1, n_l=16, fd_order=3, batch=256, propagator="taylor", order=6,
                 dt_cfg=0.004, lam_nm=800.0, intensity=(1e13, 5e14), n_cycles=4),
}

# eta of the dt_eff rule per propagator/order
ETA = {("taylor", 4): 2.5, ("rk4", 4): 2.5, ("taylor", 6): 0.5, ("taylor", 10): 1.0, ("rk45", 5): 0.9,
       ("lanczos", 12): 4.0}


def config(name, **overrides):
    c = dict(CONFIGS[name])
    c.update(overrides)
    c["name"] = name
    c["omega"] = omega_of_nm(c["lam_nm"])
    c["t_pulse"] = 2.0 * math.pi * c["n_cycles"] / c["omega"]
    return c


def intensities(c):
    """Per-member peak intensities. CFG5: I_k = 1e13 * 50^(k/255) in a seeded Fisher-Yates order."""
    b = c["batch"]
    if not isinstance(c["intensity"], tuple):
        return [float(c["intensity"])] * b
    lo, hi = c["intensity"]
    vals = [lo * (hi / lo) ** (k / max(b - 1, 1)) for k in range(b)]
    rng = SplitMix64(5)
    for i in range(b - 1, 0, -1):
        j = rng.next_u64() % (i + 1)
        vals[i], vals[j] = vals[j], vals[i]
    return vals


def pulses(c):
    """[(e0, omega, n_cycles, cep)] per member: sin^2 envelope on E, cos carrier, cep 0 (Eq. 19)."""
    return [(e0_of_intensity(i), c["omega"], float(c["n_cycles"]), 0.0) for i in intensities(c)]


def rho_gershgorin(c, e0_max=None):
    """Upper bound of the spectral radius of H used ONLY to choose a stable step:
    kappa_G/dr^2 + (L-1)L/(2 dr^2) + E0 r_max, kappa_G = 2 (3-point) or 8/3 (5-point).  With a centrifugal inner
    cut-off c["cutoff_lambda"] > 0 (an extension beyond the paper: points with l(l+1)/(2 r^2) > Lambda are held at
    zero) the centrifugal part is at most Lambda."""
    if e0_max is None:
        e0_max = max(p[0] for p in pulses(c))
    kg = 2.0 if c["fd_order"] == 3 else 8.0 / 3.0
    dr2 = c["dr"] ** 2
    cen = (c["n_l"] - 1) * c["n_l"] / (2.0 * dr2)
    lam = c.get("cutoff_lambda", 0.0)
    if lam > 0.0:
        cen = min(cen, lam)
    return kg / dr2 + cen + e0_max * c["n_r"] * c["dr"]


def dt_eff(c, propagator=None, order=None, t_run=None):
    """dt_eff = T_run / ceil(T_run / min(dt_cfg, eta/rho_G)): the stated dt of every BASELINE config is
    outside the explicit stability region."""
    propagator = propagator or c["propagator"]
    order = order or (5 if propagator == "rk45" else c["order"])
    eta = ETA.get((propagator, order), 1.0)
    t_run = t_run or c["t_pulse"]
    dt = min(c["dt_cfg"], eta / rho_gershgorin(c))
    return t_run / math.ceil(t_run / dt)


def window(c, nsteps, dt):
    """Bounded window of nsteps steps centred on the pulse peak: returns t0."""
    return 0.5 * c["t_pulse"] - 0.5 * nsteps * dt


def radial_grid(c):
    return c["dr"] * np.arange(1, c["n_r"] + 1, dtype=np.float64)


# ---- seeded states ---------------------------------------------------------------------

def random_state(c, seed_extra=0):
    """S1: re, im of every element uniform in [-1, 1) from SplitMix64(1308e6 + 1856 + config index)."""
    n = c["batch"] * c["n_l"] * c["n_r"]
    u = splitmix64_uniform(1308 * 10 ** 6 + 1856 + c["index"] + seed_extra, 2 * n)
    v = 2.0 * u - 1.0
    return (v[0::2] + 1j * v[1::2]).reshape(c["batch"], c["n_l"], c["n_r"])


def random_fields(c):
    """S1 field values: 0.05 for a single member, 0.01 + 0.0004 b for batched."""
    if c["batch"] == 1:
        return np.array([0.05])
    return 0.01 + 0.0004 * np.arange(c["batch"], dtype=np.float64)


def hydrogen_u(n, l, r):
    """Analytic hydrogen reduced radial functions u_nl(r) = r R_nl(r) (textbook), n <= 3.
    Stand-ins for bound states where no discrete eigenvector is supplied (bench, smoke)."""
    if (n, l) == (1, 0):
        return 2.0 * r * np.exp(-r)
    if (n, l) == (2, 0):
        return (1.0 / (2.0 * math.sqrt(2.0))) * r * (2.0 - r) * np.exp(-r / 2.0)
    if (n, l) == (2, 1):
        return (1.0 / (2.0 * math.sqrt(6.0))) * r * r * np.exp(-r / 2.0)
    if (n, l) == (3, 0):
        return (2.0 / (81.0 * math.sqrt(3.0))) * r * (27.0 - 18.0 * r + 2.0 * r * r) * np.exp(-r / 3.0)
    if (n, l) == (3, 1):
        return (8.0 / (27.0 * math.sqrt(6.0))) * r * r * (1.0 - r / 6.0) * np.exp(-r / 3.0)
    if (n, l) == (3, 2):
        return (4.0 / (81.0 * math.sqrt(30.0))) * r ** 3 * np.exp(-r / 3.0)
    raise ValueError((n, l))


def grid_normalised(u, dr):
    return u / math.sqrt(dr * float(np.sum(u * u)))


def ground_state(c, phi_1s=None):
    """S2: phi_1s in l = 0, zeros elsewhere, same for every member."""
    r = radial_grid(c)
    if phi_1s is None:
        phi_1s = grid_normalised(hydrogen_u(1, 0, r), c["dr"])
    psi = np.zeros((c["batch"], c["n_l"], c["n_r"]), dtype=np.complex128)
    psi[:, 0, :] = phi_1s
    return psi


def populated_state(c, phi_1s=None):
    """S4: normalise(1s (+) sum_l a_l exp(-(r-r_l)^2/(2 sigma^2)) e^{i k_l r}) -- one smooth wavepacket in every
    l block, sigma = 5 au, a_l in [0.05,0.15], r_l in [0.2,0.6] r_max, k_l in [-1,1]; SplitMix64(1856 + index)."""
    r = radial_grid(c)
    psi = ground_state(c, phi_1s)
    rng = SplitMix64(1856 + c["index"])
    r_max = c["n_r"] * c["dr"]
    for b in range(c["batch"]):
        for l in range(c["n_l"]):
            a = 0.05 + 0.10 * rng.uniform()
            rl = (0.2 + 0.4 * rng.uniform()) * r_max
            k = -1.0 + 2.0 * rng.uniform()
            psi[b, l, :] += a * np.exp(-(r - rl) ** 2 / (2.0 * 25.0)) * np.exp(1j * k * r)
        nrm = math.sqrt(c["dr"] * float(np.sum(np.abs(psi[b]) ** 2)))
        psi[b] /= nrm
    return psi
