"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

Every oracle function is checked against something other than itself: values the paper prints
(tests/golden/), closed forms, LAPACK on a dense matrix, brute force on the tiny grid, invariants.
Pin numbers P1..P10 refer to DESIGN.md "Oracle pins".
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.linalg as sla

import oracle
from paper_1308_1856_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def read_golden(name):
    rows = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            rows.append(line.split())
    return rows


def tiny(fd_order, n_l=3, n_r=100, dr=0.2):
    return oracle.make_grid(n_r, dr, n_l, fd_order)


def rand_state(shape, seed):
    u = wl.splitmix64_uniform(seed, 2 * int(np.prod(shape)))
    v = 2 * u - 1
    return (v[0::2] + 1j * v[1::2]).reshape(shape)


def dense_propagate(h, psi, dt):
    """exp(-i H dt) psi by LAPACK eigen-decomposition of the dense real-symmetric H."""
    w, v = np.linalg.eigh(h)
    return v @ (np.exp(-1j * w * dt) * (v.T @ psi))


# ---------------------------------------------------------------- coupling, pulse
def test_coupling_is_cos_theta_matrix_element():
    """c_l = <l 0|cos(theta)|l+1 0> (Eq. 9): Gauss-Legendre quadrature of normalised Legendre polynomials."""
    x, w = np.polynomial.legendre.leggauss(80)
    c = oracle.coupling(12)
    for l in range(12):
        pl = np.polynomial.legendre.Legendre.basis(l)(x) * math.sqrt((2 * l + 1) / 2)
        pn = np.polynomial.legendre.Legendre.basis(l + 1)(x) * math.sqrt((2 * l + 3) / 2)
        assert abs(np.sum(w * pl * x * pn) - c[l]) < 1e-13
    assert abs(c[0] - 1 / math.sqrt(3)) < 1e-16


def test_pulse_properties():
    """E(t) = e0 sin^2(w t/2n_c) cos(w t + cep) on [0, T] (Eq. 19): zero at the ends and outside,
    |E(T/2)| = e0 for integer n_c, zero time integral, carrier at omega."""
    e0, om, nc = 0.0534, 0.057, 4.0
    T = 2 * math.pi * nc / om
    p = (e0, om, nc, 0.0)
    assert oracle.pulse_E(p, 0.0) == 0.0
    assert abs(oracle.pulse_E(p, T)) < 1e-15
    assert oracle.pulse_E(p, -1e-9) == 0.0 and oracle.pulse_E(p, T * (1 + 1e-12) + 1e-9) == 0.0
    assert abs(abs(oracle.pulse_E(p, T / 2)) - e0) < 1e-15
    t = np.linspace(0, T, 20001)
    e = np.array([oracle.pulse_E(p, x) for x in t])
    assert abs(np.trapezoid(e, t)) < 1e-9 * e0 * T           # no DC component for n_c >= 2
    # the spectrum peaks at the carrier
    f = np.abs(np.fft.rfft(e, 8 * len(e)))
    om_peak = 2 * math.pi * np.argmax(f) / (8 * len(e) * (t[1] - t[0]))
    assert abs(om_peak - om) < 0.02 * om
    # cep shifts the carrier: cep = pi/2 makes the centre a zero crossing
    assert abs(oracle.pulse_E((e0, om, nc, math.pi / 2), T / 2)) < 1e-15
    # test aid: omega = 0 is a static field
    assert oracle.pulse_E((0.05, 0.0, 1.0, 0.0), 123.4) == 0.05


# ---------------------------------------------------------------- P1: Hermiticity, dense == matrix-free
@pytest.mark.parametrize("fd", [3, 5])
def test_P1_dense_H_symmetric_and_equals_matrix_free(fd):
    g = tiny(fd)
    h = oracle.dense_H(g, 0.05)
    assert np.array_equal(h, h.T)                               # exactly symmetric
    psi = rand_state((1, g.n_l, g.n_r), 11 + fd)
    ref = (h @ psi.reshape(-1)).reshape(psi.shape)
    out = oracle.apply_H(g, psi, 0.05)
    assert np.linalg.norm(out - ref) <= 1e-14 * np.linalg.norm(ref)


@pytest.mark.parametrize("fd", [3, 5])
def test_P1_band_structure(fd):
    """P:134/Fig. 1: diagonal blocks are (2w+1)-diagonal, length-gauge off-diagonal blocks are diagonal,
    blocks with |l-l'| > 1 vanish; off-diagonal blocks scale linearly with E and vanish at E = 0."""
    g = tiny(fd)
    n, L, w = g.n_r, g.n_l, (1 if fd == 3 else 2)
    h = oracle.dense_H(g, 0.05).reshape(L, n, L, n)
    h0 = oracle.dense_H(g, 0.0).reshape(L, n, L, n)
    jj = np.abs(np.arange(n)[:, None] - np.arange(n)[None, :])
    for l in range(L):
        for lp in range(L):
            blk = h[l, :, lp, :]
            if l == lp:
                assert np.all(blk[jj > w] == 0) and np.all(blk[jj <= w] != 0)
                assert np.array_equal(blk, h0[l, :, lp, :])
            elif abs(l - lp) == 1:
                assert np.all(blk[jj > 0] == 0) and np.all(np.diag(blk) != 0)
                assert np.all(h0[l, :, lp, :] == 0)
                r = 0.2 * np.arange(1, n + 1)
                assert np.allclose(np.diag(blk), 0.05 * r * oracle.coupling(L)[min(l, lp)], rtol=1e-15)
            else:
                assert np.all(blk == 0)


@pytest.mark.parametrize("shape", [(500, 0.2, 8, 3, 1), (700, 0.1, 5, 5, 1), (64, 0.1, 4, 3, 3), (257, 0.1, 7, 5, 2)])
def test_P1_matrix_free_hermitian(shape):
    n_r, dr, n_l, fd, b = shape
    g = oracle.make_grid(n_r, dr, n_l, fd, batch=b)
    x = rand_state((b, n_l, n_r), 3)
    y = rand_state((b, n_l, n_r), 4)
    e = 0.01 + 0.0004 * np.arange(b)
    hx, hy = oracle.apply_H(g, x, e), oracle.apply_H(g, y, e)
    for m in range(b):
        lhs, rhs = np.vdot(x[m], hy[m]), np.vdot(hx[m], y[m])
        assert abs(lhs - rhs) <= 1e-13 * abs(lhs)
    # batched call == per-member calls
    g1 = oracle.make_grid(n_r, dr, n_l, fd, batch=1)
    for m in range(b):
        assert np.array_equal(oracle.apply_H(g1, x[m], e[m])[0], hx[m])


# ---------------------------------------------------------------- P2/P3: energies
def test_P2_closed_form_3point_ground_state():
    for dr_s, e_s in read_golden("closed_form_energies.txt"):
        dr, e_gold = float(dr_s), float(e_s)
        assert abs(e_gold + 1 / (1 + math.sqrt(1 + dr * dr))) < 1e-12
        g = oracle.make_grid(int(round(100 / dr)), dr, 1, 3)
        en, phi = oracle.bound_states(g, 0, 1)
        assert abs(en[0] - e_gold) < 1e-11
        # the eigenvector is j q^j
        q = math.sqrt(1 + dr * dr) - dr
        j = np.arange(1, g.n_r + 1)
        ref = wl.grid_normalised(j * q ** j, dr)
        assert np.max(np.abs(phi[0] - ref)) < 1e-9
        assert abs(dr * np.sum(phi[0] ** 2) - 1) < 1e-13 and phi[0, 0] > 0
        # H phi = E phi with the matrix-free operator (pins kinetic sign, Coulomb term, grid origin)
        res = oracle.apply_H(g, phi[0][None, None, :], 0.0)[0, 0] - en[0] * phi[0]
        assert np.linalg.norm(res) < 1e-10
    # O(dr^2) convergence to -0.5 (NS)
    errs = [abs(-1 / (1 + math.sqrt(1 + d * d)) + 0.5) for d in (0.2, 0.1, 0.05)]
    assert 3.9 < errs[0] / errs[1] < 4.1 and 3.9 < errs[1] / errs[2] < 4.1


@pytest.mark.parametrize("fd,dr,l", [(3, 0.2, 0), (3, 0.2, 1), (3, 0.1, 3), (5, 0.2, 0), (5, 0.2, 1), (5, 0.1, 2)])
def test_P2b_eigensolver_vs_lapack(fd, dr, l):
    """Bound states of h_l against LAPACK on the same band (scipy.linalg.eig_banded)."""
    n = 600
    g = oracle.make_grid(n, dr, l + 1, fd)
    r = dr * np.arange(1, n + 1)
    v = l * (l + 1) / (2 * r * r) - 1 / r
    if fd == 3:
        band = np.zeros((2, n)); band[0] = 1 / dr ** 2 + v; band[1, :-1] = -0.5 / dr ** 2
    else:
        band = np.zeros((3, n)); band[0] = 30 / (24 * dr ** 2) + v
        band[1, :-1] = -16 / (24 * dr ** 2); band[2, :-2] = 1 / (24 * dr ** 2)
    w, vec = sla.eig_banded(band, lower=True, select="i", select_range=(0, 3))
    en, phi = oracle.bound_states(g, l, 4)
    assert np.max(np.abs(en - w)) < 1e-10
    for k in range(4):
        ref = vec[:, k] / math.sqrt(dr) * np.sign(vec[0, k])
        assert np.max(np.abs(phi[k] - ref)) < 1e-7
    # the oracle's own H agrees: ||H phi - E phi|| small for block l
    psi = np.zeros((1, l + 1, n), dtype=complex); psi[0, l] = phi[0]
    res = oracle.apply_H(g, psi, 0.0)[0, l] - en[0] * phi[0]
    assert np.linalg.norm(res) < 1e-9
    # only_negative stops at the continuum
    en_neg, _ = oracle.bound_states(g, l, 40, only_negative=True)
    assert len(en_neg) < 40 and np.all(en_neg < 0)
    w_all = sla.eig_banded(band, lower=True, eigvals_only=True)
    assert len(en_neg) == int(np.sum(w_all < 0))


def test_P3_paper_printed_energies_5point():
    """E_1s ~ -0.47 on (R = 800, dr = 0.2) and ~ -0.5 with Offset -0.02: pins the 5-point coefficients and
    the zero-extension inner boundary (reading G4); odd extension would give -0.4896 / -0.5241."""
    for n_r, dr, fd, off, e_print, tol in read_golden("paper_energies.txt"):
        g = oracle.make_grid(int(n_r), float(dr), 1, int(fd), r_offset=float(off))
        en, _ = oracle.bound_states(g, 0, 1)
        assert abs(en[0] - float(e_print)) < float(tol), en
    g = oracle.make_grid(4000, 0.2, 1, 5)
    assert abs(oracle.bound_states(g, 0, 1)[0][0] - (-0.4714542027)) < 1e-9


# ---------------------------------------------------------------- P6: structural zeros / reality
@pytest.mark.parametrize("fd", [3, 5])
def test_P6_structural_zeros_and_reality(fd):
    g = oracle.make_grid(120, 0.2, 6, fd)
    psi = np.zeros((1, 6, 120), dtype=complex)
    psi[0, 0] = rand_state((120,), 5).real
    cur = psi
    for k in range(1, 5):
        cur = oracle.apply_H(g, cur, 0.07)
        assert np.all(cur[0, k + 1:] == 0)                     # coupling only l <-> l +- 1
        assert np.any(cur[0, k] != 0)
        assert np.all(cur.imag == 0)                           # H real: real in, real out
    # i * real in -> purely imaginary out
    out = oracle.apply_H(g, 1j * psi, 0.07)
    assert np.all(out.real == 0)


# ---------------------------------------------------------------- P4: dense exponential on the tiny grid
STATIC = lambda e: (e, 0.0, 1.0, 0.0)       # omega = 0: static field


@pytest.mark.parametrize("fd", [3, 5])
@pytest.mark.parametrize("order", [2, 4, 6, 10])
def test_P4_taylor_vs_dense_exponential(fd, order):
    g = tiny(fd)
    h = oracle.dense_H(g, 0.05)
    rho = np.max(np.abs(np.linalg.eigvalsh(h)))
    dt = 0.004
    y = dt * rho
    psi = rand_state((1, g.n_l, g.n_r), 21)
    psi /= np.linalg.norm(psi)
    exact = dense_propagate(h, psi.reshape(-1), dt)
    got, _ = oracle.step_taylor(g, STATIC(0.05), psi, order, 0.0, dt, 1)
    err = np.linalg.norm(got.reshape(-1) - exact)
    bound = 1.01 * y ** (order + 1) / math.factorial(order + 1)
    assert err <= bound + 1e-15
    # ... and it IS of order P: the error is the first dropped term (next one is y/(P+2) smaller)
    lead = psi.reshape(-1).copy()
    for k in range(order + 1):
        lead = dt * (h @ lead)
    lead = np.linalg.norm(lead) / math.factorial(order + 1)
    assert 0.7 * lead - 2e-15 <= err <= 1.3 * lead + 2e-15
    # exact polynomial: sum_k (-i H dt)^k / k!
    acc, term = psi.reshape(-1).copy(), psi.reshape(-1).copy()
    for k in range(1, order + 1):
        term = (-1j * dt / k) * (h @ term); acc = acc + term
    assert np.linalg.norm(got.reshape(-1) - acc) < 1e-14


@pytest.mark.parametrize("fd", [3, 5])
def test_P4_rk4_and_dp5_stability_polynomials(fd):
    """Constant field: RK4 == Taylor-4 polynomial; DP5 == sum_{k<=5} z^k/k! + z^6/600 (its stability function)."""
    g = tiny(fd)
    h = oracle.dense_H(g, 0.05)
    dt = 0.004
    psi = rand_state((1, g.n_l, g.n_r), 22); psi /= np.linalg.norm(psi)
    v = psi.reshape(-1)
    pw = [v]
    for k in range(1, 7):
        pw.append(-1j * dt * (h @ pw[-1]))
    t4 = sum(pw[k] / math.factorial(k) for k in range(5))
    r5 = sum(pw[k] / math.factorial(k) for k in range(6)) + pw[6] / 600
    got4, _ = oracle.step_rk4(g, STATIC(0.05), psi, 0.0, dt, 1)
    assert np.linalg.norm(got4.reshape(-1) - t4) < 2e-15
    got5, err, _ = oracle.step_rk_fixed(g, STATIC(0.05), psi, 1, 0.0, dt, 1)
    assert np.linalg.norm(got5.reshape(-1) - r5) < 2e-15
    # embedded 4th-order solution: R4hat = sum_{k<=4} z^k/k! + (1097/120000) z^5 + (161/120000) z^6 + z^7/24000
    pw.append(-1j * dt * (h @ pw[-1]))
    r4 = sum(pw[k] / math.factorial(k) for k in range(5)) + 1097 / 120000 * pw[5] + 161 / 120000 * pw[6] + pw[7] / 24000
    want = np.linalg.norm(r5 - r4) / np.linalg.norm(r5)
    assert abs(err[0] - want) < 1e-3 * want


def test_dormand_prince_order_conditions():
    """The tableau satisfies the order conditions in exact rational arithmetic: row sums = c; b up to order 5."""
    F = Fraction
    c = [F(0), F(1, 5), F(3, 10), F(4, 5), F(8, 9), F(1), F(1)]
    a = [[], [F(1, 5)], [F(3, 40), F(9, 40)], [F(44, 45), F(-56, 15), F(32, 9)],
         [F(19372, 6561), F(-25360, 2187), F(64448, 6561), F(-212, 729)],
         [F(9017, 3168), F(-355, 33), F(46732, 5247), F(49, 176), F(-5103, 18656)],
         [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84)]]
    b = [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84), F(0)]
    bh = [F(5179, 57600), F(0), F(7571, 16695), F(393, 640), F(-92097, 339200), F(187, 2100), F(1, 40)]
    for i in range(7):
        assert sum(a[i]) == c[i]
    for q in range(1, 6):                                       # quadrature conditions
        assert sum(bi * ci ** (q - 1) for bi, ci in zip(b, c)) == F(1, q)
    for q in range(1, 5):
        assert sum(bi * ci ** (q - 1) for bi, ci in zip(bh, c)) == F(1, q)
    assert sum(bi * ci ** 4 for bi, ci in zip(bh, c)) != F(1, 5)
    ac = [sum(aij * c[j] for j, aij in enumerate(a[i])) for i in range(7)]
    assert sum(bi * x for bi, x in zip(b, ac)) == F(1, 6)        # order 3
    assert sum(bi * ci * x for bi, ci, x in zip(b, c, ac)) == F(1, 8)   # order 4
    # the stability function the oracle is pinned to in test_P4: coefficient of z^6 is 1/600
    # (b . A^5 . 1 = 1/600)
    vec = [F(1)] * 7
    for _ in range(5):
        vec = [sum(aij * vec[j] for j, aij in enumerate(a[i])) for i in range(7)]
    assert sum(bi * x for bi, x in zip(b, vec)) == F(1, 600)


@pytest.mark.parametrize("fd", [3, 5])
def test_P4_lanczos_vs_dense_exponential(fd):
    g = tiny(fd)
    h = oracle.dense_H(g, 0.05)
    dt = 0.004
    psi = rand_state((1, g.n_l, g.n_r), 23); psi /= np.linalg.norm(psi)
    exact = dense_propagate(h, psi.reshape(-1), dt)
    got, _ = oracle.step_lanczos(g, STATIC(0.05), psi, 16, 12, 0.0, dt, 1)
    assert np.linalg.norm(got.reshape(-1) - exact) < 1e-12
    # several steps, against the dense propagator applied repeatedly
    got, _ = oracle.step_lanczos(g, STATIC(0.05), psi, 16, 12, 0.0, dt, 25)
    assert np.linalg.norm(got.reshape(-1) - dense_propagate(h, psi.reshape(-1), 25 * dt)) < 1e-11


# ---------------------------------------------------------------- P9: Lanczos internals
@pytest.mark.parametrize("fd", [3, 5])
def test_P9_lanczos_internals(fd):
    g = tiny(fd)
    h = oracle.dense_H(g, 0.05)
    psi = rand_state((1, g.n_l, g.n_r), 24)
    K = 16
    r = oracle.lanczos_internals(g, psi, 0.05, K, 12, 0.004)
    assert r["m"] == K
    Q = r["q"].reshape(K, -1)
    # three-term recurrence in the order of reading G16:  H q_p = beta_{p-1} q_{p-1} + alpha_p q_p + beta_p q_{p+1}
    hn = np.max(np.abs(np.linalg.eigvalsh(h)))
    for p in range(K - 1):
        lhs = h @ Q[p]
        rhs = r["alpha"][p] * Q[p] + r["beta"][p] * Q[p + 1] + (r["beta"][p - 1] * Q[p - 1] if p else 0)
        assert np.linalg.norm(lhs - rhs) < 1e-13 * hn
        assert abs(r["alpha"][p] - np.vdot(Q[p], lhs).real) < 1e-12 * hn
    G = Q.conj() @ Q.T
    assert np.max(np.abs(np.diag(G) - 1)) < 1e-13                   # unit vectors
    assert np.max(np.abs(np.diag(G, 1))) < 1e-12 and np.max(np.abs(np.diag(G, 2))) < 1e-12   # local orthogonality
    # no re-orthogonalisation in the paper: global orthogonality decays as Ritz values converge, but stays small
    assert np.max(np.abs(G[:8, :8] - np.eye(8))) < 1e-11 and np.max(np.abs(G - np.eye(K))) < 1e-6
    T = Q.conj() @ (h @ Q.T)
    Tref = np.diag(r["alpha"]) + np.diag(r["beta"][:K - 1], 1) + np.diag(r["beta"][:K - 1], -1)
    assert np.max(np.abs(T - Tref)) < 1e-6 * np.max(np.abs(Tref))  # Q^H H Q = tridiag(beta, alpha, beta)
    assert abs(np.vdot(Q[0], psi.reshape(-1)) - np.linalg.norm(psi)) < 1e-12
    # coefficients = exp(-i T dt) e_1 (LAPACK), sub-stepping per the Gershgorin rule
    w, v = np.linalg.eigh(Tref)
    cref = v @ (np.exp(-1j * w * 0.004) * v[0])
    assert np.max(np.abs(r["coef"] - cref)) < 1e-13
    gr = max(abs(r["alpha"][i]) + (r["beta"][i - 1] if i else 0) + (r["beta"][i] if i < K - 1 else 0) for i in range(K))
    assert r["n_sub"] == max(1, math.ceil(0.004 * gr / 3.0))
    # K = 1: psi * R(-i alpha dt), R the truncated exponential
    r1 = oracle.lanczos_internals(g, psi, 0.05, 1, 12, 0.004)
    a = np.vdot(psi, (h @ psi.reshape(-1)).reshape(psi.shape)).real / np.vdot(psi, psi).real
    assert abs(r1["alpha"][0] - a) < 1e-12 * abs(a)
    z = -1j * a * 0.004 / r1["n_sub"]
    R = sum(z ** k / math.factorial(k) for k in range(13)) ** r1["n_sub"]
    assert abs(r1["coef"][0] - R) < 1e-14
    got, _ = oracle.step_lanczos(g, STATIC(0.05), psi, 1, 12, 0.0, 0.004, 1)
    assert np.linalg.norm(got - psi * R) < 1e-13 * np.linalg.norm(psi)


def test_lanczos_substepping_large_dt():
    """Reading G18: with Ritz values * dt above the Taylor-12 stability limit the small system is sub-stepped;
    the step stays unitary in the Krylov space (|c| = 1) and exact for a state inside an invariant subspace."""
    g = tiny(3)
    h = oracle.dense_H(g, 0.0)
    w, v = np.linalg.eigh(h)
    # state spanned by 3 eigenvectors with large eigenvalues: Krylov space closes at m = 3
    idx = [len(w) - 1, len(w) - 7, 5]
    psi = (v[:, idx] @ np.array([0.6, 0.5 + 0.2j, 0.3j])).reshape(1, g.n_l, g.n_r)
    dt = 0.5
    assert dt * w[-1] > 3.4
    r = oracle.lanczos_internals(g, psi, 0.0, 8, 12, dt, beta_tol=1e-9)
    assert r["m"] == 3 and r["n_sub"] > 1
    # each sub-step has y <= 3: Taylor-12 is stable there (|R| <= 1) and accurate to y^13/13! ~ 2.6e-4
    assert 1 - 1e-3 * r["n_sub"] < np.linalg.norm(r["coef"]) <= 1 + 1e-12
    got, _ = oracle.step_lanczos(g, STATIC(0.0), psi, 8, 12, 0.0, dt, 1, beta_tol=1e-9)
    assert np.linalg.norm(got.reshape(-1) - dense_propagate(h, psi.reshape(-1), dt)) < 1e-3 * r["n_sub"]
    # without sub-stepping the same step would blow up: |R_12(-i y)| > 1 for y = dt * lambda_max
    y = dt * w[-1]
    assert abs(sum((-1j * y) ** k / math.factorial(k) for k in range(13))) > 1.0 + 1e-3


# ---------------------------------------------------------------- P5: field-free eigenstate phase
@pytest.mark.parametrize("prop", ["taylor4", "taylor6", "rk4", "dp5", "lanczos"])
def test_P5_field_free_phase(prop):
    dr, n_r = 0.2, 500
    g = oracle.make_grid(n_r, dr, 3, 3)
    e1s = -1 / (1 + math.sqrt(1 + dr * dr))                       # closed form, not the oracle's eigenvalue
    en, phi = oracle.bound_states(g, 0, 1)
    psi0 = np.zeros((1, 3, n_r), dtype=complex); psi0[0, 0] = phi[0]
    dt, n = 0.01, 200
    off = (0.0, 0.057, 2.0, 0.0)
    trunc = lambda z, p: sum(z ** k / math.factorial(k) for k in range(p + 1))
    z = -1j * e1s * dt
    if prop.startswith("taylor"):
        p = int(prop[6:]); psi, _ = oracle.step_taylor(g, off, psi0, p, 0.0, dt, n); R = trunc(z, p)
    elif prop == "rk4":
        psi, _ = oracle.step_rk4(g, off, psi0, 0.0, dt, n); R = trunc(z, 4)
    elif prop == "dp5":
        psi, _, _ = oracle.step_rk_fixed(g, off, psi0, 1, 0.0, dt, n); R = trunc(z, 5) + z ** 6 / 600
    else:
        psi, _ = oracle.step_lanczos(g, off, psi0, 16, 12, 0.0, dt, n); R = trunc(z, 12)
    amp = dr * np.sum(phi[0] * psi[0, 0])
    assert abs(amp - R ** n) < 1e-12
    assert abs(amp - np.exp(-1j * e1s * dt * n)) < 1e-6          # e^{-i E0 t} phase (NS)
    obs = oracle.observables(g, psi, 0.0, ([0], phi[:1]))
    assert abs(obs[0, 0] - abs(R) ** (2 * n)) < 1e-12            # norm = |R|^{2n}
    assert abs(obs[0, 3] - abs(R) ** (2 * n)) < 1e-12            # 1s population
    assert np.all(np.abs(psi[0, 1:]) < 1e-300)                   # no field: other blocks stay empty


# ---------------------------------------------------------------- time-dependent H: order of convergence
def _td_reference(g, pulse, psi, t0, t1, n):
    """Independent reference for time-dependent H: product of dense midpoint exponentials, Richardson-extrapolated."""
    def run(m):
        v = psi.reshape(-1).copy()
        dt = (t1 - t0) / m
        h0 = oracle.dense_H(g, 0.0)
        h1 = oracle.dense_H(g, 1.0) - h0
        for k in range(m):
            e = oracle.pulse_E(pulse, t0 + (k + 0.5) * dt)
            v = dense_propagate(h0 + e * h1, v, dt)
        return v
    a, b = run(n), run(2 * n)
    return (4 * b - a) / 3                                       # midpoint rule is O(dt^2)


def test_time_dependent_convergence_orders():
    g = oracle.make_grid(40, 0.4, 3, 3)                            # small so that dense references are cheap
    pulse = (0.3, 1.5, 2.0, 0.3)                                   # strong, fast pulse: time dependence matters
    t0, t1 = 1.0, 3.0
    psi = rand_state((1, 3, 40), 31); psi /= np.linalg.norm(psi)
    ref = _td_reference(g, pulse, psi, t0, t1, 400)
    def err(fn, n):
        return np.linalg.norm(fn(n).reshape(-1) - ref)
    rk4 = lambda n: oracle.step_rk4(g, pulse, psi, t0, (t1 - t0) / n, n)[0]
    dp5 = lambda n: oracle.step_rk_fixed(g, pulse, psi, 1, t0, (t1 - t0) / n, n)[0]
    tay = lambda n: oracle.step_taylor(g, pulse, psi, 8, t0, (t1 - t0) / n, n)[0]
    lan = lambda n: oracle.step_lanczos(g, pulse, psi, 12, 12, t0, (t1 - t0) / n, n)[0]
    tay_start = lambda n: oracle.step_taylor(g, pulse, psi, 8, t0, (t1 - t0) / n, n, field_sample=1)[0]
    e1, e2 = err(rk4, 400), err(rk4, 800)
    assert 14 < e1 / e2 < 18, (e1, e2)                           # 4th order: pins the stage times c_i
    e1, e2 = err(dp5, 200), err(dp5, 400)
    assert 27 < e1 / e2 < 37, (e1, e2)                           # 5th order
    for fn in (tay, lan):                                        # midpoint-frozen H: 2nd order
        e1, e2 = err(fn, 400), err(fn, 800)
        assert 3.8 < e1 / e2 < 4.2, (e1, e2)
    e1, e2 = err(tay_start, 400), err(tay_start, 800)
    assert 1.9 < e1 / e2 < 2.1                                   # start-frozen H: 1st order
    assert err(dp5, 800) < 1e-7 and err(rk4, 800) < 1e-6


# ---------------------------------------------------------------- RK45 controller
def test_rk45_controller_and_replay():
    g = oracle.make_grid(200, 0.2, 4, 5)
    pulse = (0.05, 0.057, 2.0, 0.0)
    en, phi = oracle.bound_states(g, 0, 1)
    psi0 = np.zeros((1, 4, 200), dtype=complex); psi0[0, 0] = phi[0]
    t0, t1 = 100.0, 101.0
    psi, info = oracle.step_rk45(g, pulse, psi0, t0, t1, 1e-4, 1e-8)
    assert info["n_accept"] == len(info["dt"]) and info["n_accept"] > 10
    assert abs(np.sum(info["dt"]) - (t1 - t0)) < 1e-12          # lands on t_end
    assert np.all(info["err"] <= 1.0)
    assert np.all(info["dt"][1:] <= 5.0 * info["dt"][:-1] * (1 + 1e-12))
    # replaying the accepted steps reproduces the state bit for bit and never exceeds err 1
    psi_r, info_r = oracle.step_rk45(g, pulse, psi0, t0, t1, 1e-4, 1e-8, dt_replay=info["dt"])
    assert np.array_equal(psi_r, psi)
    assert np.allclose(info_r["err"], info["err"], rtol=1e-12)
    # against a fine fixed-step RK4 run: error ~ n_accept * rtol (tolerance is per step)
    n = 40000
    ref, _ = oracle.step_rk4(g, pulse, psi0, t0, (t1 - t0) / n, n)
    assert np.linalg.norm(psi - ref) < 5 * info["n_accept"] * 1e-8
    # dt_max caps every step
    _, info_c = oracle.step_rk45(g, pulse, psi0, t0, t1, 1e-4, 1e-8, dt_max=2e-3)
    assert np.max(info_c["dt"]) <= 2e-3 * (1 + 1e-15)
    # fixed-step DP5 reports the same error estimate as the adaptive call's first step
    _, err, _ = oracle.step_rk_fixed(g, pulse, psi0, 1, t0, 1e-4, 1)
    assert abs(err[0] / 1e-8 - info["err"][0]) < 1e-9 * info["err"][0] + 1e-30


# ---------------------------------------------------------------- observables
def test_observables_textbook_matrix_elements():
    """<z> and <z''> of a 1s + 2p0 superposition of analytic hydrogen functions against the textbook integrals."""
    gold = {k: float(v) for k, v in read_golden("hydrogen_matrix_elements.txt")}
    dr, n_r = 0.01, 6000
    g = oracle.make_grid(n_r, dr, 3, 3)
    r = dr * np.arange(1, n_r + 1)
    u1s, u2p = wl.hydrogen_u(1, 0, r), wl.hydrogen_u(2, 1, r)
    a, b = 0.8, 0.6 * np.exp(0.4j)
    psi = np.zeros((1, 3, n_r), dtype=complex); psi[0, 0] = a * u1s; psi[0, 1] = b * u2p
    e_now = 0.0123
    obs = oracle.observables(g, psi, e_now, ([0, 1, 2], np.stack([u1s, u2p, wl.hydrogen_u(3, 2, r)])))
    re_ab = (np.conj(a) * b).real
    assert abs(obs[0, 0] - 1.0) < 1e-6                                    # norm
    assert abs(obs[0, 1] - 2 * re_ab * gold["z_1s_2p"]) < 1e-6            # P:294 Eq. 34
    assert abs(obs[0, 2] - (-e_now - 2 * re_ab * gold["acc_1s_2p"])) < 1e-5   # P:302 Eq. 36
    assert abs(obs[0, 3] - 0.64) < 1e-6 and abs(obs[0, 4] - 0.36) < 1e-6   # P:227 Eq. 25 (|.|^2)
    assert obs[0, 5] < 1e-20
    # Z scales the acceleration's Coulomb term (R-G14)
    g2 = oracle.make_grid(n_r, dr, 3, 3, z_nuc=2.0)
    obs2 = oracle.observables(g2, psi, e_now)
    assert abs((obs2[0, 2] + e_now) - 2 * (obs[0, 2] + e_now)) < 1e-12
    # batch rows are independent
    g3 = oracle.make_grid(n_r, dr, 3, 3, batch=2)
    two = np.concatenate([psi, 0.5 * psi])
    o3 = oracle.observables(g3, two, [e_now, 0.0])
    assert abs(o3[1, 0] - 0.25 * obs[0, 0]) < 1e-15 and abs(o3[0, 1] - obs[0, 1]) < 1e-15


# ---------------------------------------------------------------- P7: first-order perturbation theory
def test_P7_resonant_1s_2p_perturbation_theory():
    dr, n_r = 0.2, 500
    g = oracle.make_grid(n_r, dr, 3, 3)
    e1s, p1s = oracle.bound_states(g, 0, 1)
    e2p, p2p = oracle.bound_states(g, 1, 1)
    om = e2p[0] - e1s[0]
    assert abs(om - 0.369992762914) < 1e-9
    r = dr * np.arange(1, n_r + 1)
    d = (1 / math.sqrt(3)) * dr * np.sum(p2p[0] * r * p1s[0])    # textbook c_0 = 1/sqrt 3
    nc = 10.0
    T = 2 * math.pi * nc / om
    nsteps = int(round(T / 0.0035))
    dt = T / nsteps
    psi0 = np.zeros((1, 3, n_r), dtype=complex); psi0[0, 0] = p1s[0]
    res = {}
    for e0 in (1e-4, 1e-3):
        pulse = (e0, om, nc, 0.0)
        psi, _ = oracle.step_taylor(g, pulse, psi0, 4, 0.0, dt, nsteps)
        pop = oracle.observables(g, psi, 0.0, ([0, 1], np.stack([p1s[0], p2p[0]])))[0, 4]
        t = np.linspace(0, T, 400001)
        et = e0 * np.sin(om * t / (2 * nc)) ** 2 * np.cos(om * t)   # independent quadrature of the pulse
        pt = d * d * abs(np.trapezoid(et * np.exp(1j * om * t), t)) ** 2
        res[e0] = (pop - pt) / pt
    assert abs(res[1e-4]) < 1e-5, res
    assert 50 < res[1e-3] / res[1e-4] < 200, res                    # deviation is the E0^2 correction


# ---------------------------------------------------------------- P8 / P10: Ehrenfest, norm conservation
def test_P8_ehrenfest_and_P10_norm():
    c = wl.config("cfg1", n_l=4)
    g = oracle.make_grid(c["n_r"], c["dr"], c["n_l"], c["fd_order"])
    en, phi = oracle.bound_states(g, 0, 1)
    psi0 = wl.ground_state(c, phi[0])
    pulse = wl.pulses(c)[0]
    dt = wl.dt_eff(c)
    t0 = 0.25 * c["t_pulse"]
    n = 6000
    psi, obs = oracle.step_taylor(g, pulse, psi0, 4, t0, dt, n, states=([0], phi[:1]), obs_every=1)
    norm, z, acc = obs[:, 0, 0], obs[:, 0, 1], obs[:, 0, 2]
    assert np.max(np.abs(norm - 1)) < 1e-11                        # P10
    s = 50                                                         # second difference on a coarser stride
    zz = z[::s]
    d2 = (zz[2:] - 2 * zz[1:-1] + zz[:-2]) / (s * dt) ** 2
    a = acc[::s][1:-1]
    assert np.max(np.abs(d2 - a)) < 0.02 * np.max(np.abs(a))      # P8 (soft): signs/factors of Eq. 34/36
    assert np.max(np.abs(a)) > 1e-3


# ------------------------------------------------------------------------------------------- imaginary time (P11)
def _h_l_banded(n_r, dr, l):
    """diagonal and off-diagonal of the 3-point h_l (Eq. 7, reading R-G5), written out here independently."""
    r = dr * np.arange(1, n_r + 1)
    d = 1.0 / dr ** 2 + l * (l + 1) / (2 * r ** 2) - 1.0 / r
    e = np.full(n_r - 1, -0.5 / dr ** 2)
    return d, e


@pytest.mark.parametrize("l", [0, 1])
def test_P11_imaginary_time_converges_to_lowest_state_of_l(l):
    """with -i -> 1 and re-normalisation the state settles into the lowest eigenstate of the populated l
    block, and -ln<psi|psi>/(2 dt) (Eq. 24, reading R-G25) is its energy: closed form for l = 0, LAPACK for l = 1."""
    dr, n_r, dt, order = 0.2, 400, 0.01, 4
    g = oracle.make_grid(n_r, dr, 3, 3)
    r = dr * np.arange(1, n_r + 1)
    psi = np.zeros((1, 3, n_r), dtype=np.complex128)
    psi[0, l] = r ** (l + 1) * np.exp(-r / (l + 1)) * (1 + 0.3j)          # analytic guess with an arbitrary phase
    psi /= math.sqrt(dr * np.sum(np.abs(psi) ** 2))
    out, en = oracle.step_imag(g, psi, order, dt, 12000)
    d, e = _h_l_banded(n_r, dr, l)
    w, v = sla.eigh_tridiagonal(d, e, select="i", select_range=(0, 0))
    if l == 0:
        closed = -1.0 / (1.0 + math.sqrt(1.0 + dr * dr))                # golden/closed_form_energies.txt
        assert abs(w[0] - closed) < 1e-9                                 # (finite box: 80 au)
    assert abs(en[-1, 0] - w[0]) < 1e-9
    assert np.all(np.diff(en[:, 0]) < 1e-11)                              # the estimate decreases monotonically (up to rounding / dt)
    assert abs(dr * np.sum(np.abs(out) ** 2) - 1.0) < 1e-13              # re-normalised
    assert np.count_nonzero(out[0, [k for k in range(3) if k != l]]) == 0  # no field: blocks stay uncoupled
    ov = abs(np.vdot(v[:, 0], out[0, l])) * math.sqrt(dr)
    assert abs(ov - 1.0) < 1e-9                                           # the state is the LAPACK eigenvector


def test_P11_imaginary_time_step_on_an_eigenvector():
    """One step from an exact eigenvector of the discrete h_0: the state is unchanged and the estimate is
    -ln(R_P(-E dt)^2)/(2 dt) with R_P the truncated exponential: pins the sign, the 1/k factors and the factor 2."""
    dr, n_r = 0.2, 300
    g = oracle.make_grid(n_r, dr, 2, 3)
    d, e = _h_l_banded(n_r, dr, 0)
    w, v = sla.eigh_tridiagonal(d, e, select="i", select_range=(0, 1))
    for dt, order in ((0.02, 3), (0.05, 6)):
        for idx in (0, 1):
            psi = np.zeros((1, 2, n_r), dtype=np.complex128)
            psi[0, 0] = v[:, idx] / math.sqrt(dr)
            out, en = oracle.step_imag(g, psi, order, dt, 1)
            rp = sum((-w[idx] * dt) ** k / math.factorial(k) for k in range(order + 1))
            assert abs(en[0, 0] - (-math.log(rp * rp) / (2 * dt))) < 1e-11
            assert np.linalg.norm(out - psi) < 1e-11 * np.linalg.norm(psi)


# ------------------------------------------------------------------------------------ absorber and yields (P12)
def test_P12_absorber_mask_is_one_step_of_eq18():
    """exp(-i W dt) with W of Eq. 18 written out literally equals the real mask 1 - cos^p(...), for any dt; the
    limits of P:148 (no absorption at r -> 0, complete at r_b) and monotonic decrease hold."""
    g = oracle.make_grid(500, 0.2, 2, 3)
    for r_b, p in ((100.0, 8), (80.0, 2), (100.0, 40)):
        m = oracle.absorber_mask(g, r_b, p)
        r = g.dr * np.arange(1, g.n_r + 1)
        inside = r < r_b
        for dt in (0.01, 0.3):
            w = oracle.absorber_W(g, r_b, p, dt)
            assert np.allclose(np.exp(-1j * w[inside] * dt), m[inside], rtol=1e-13, atol=1e-15)
            assert np.all(w[inside].imag <= 0)                       # absorbing, never amplifying
        assert abs(m[0] - 1.0) < (0.5 * np.pi * r[0] / r_b) ** p * 1.01 + 1e-15   # 1 - M ~ (pi r / 2 r_b)^p at small r
        assert np.all(np.diff(m[inside]) <= 0) and m[inside][-1] < (1 - np.cos(0.5 * np.pi * g.dr / r_b) ** p) + 1e-12
        assert np.all(m[~inside] == 0.0)


def test_P12_absorber_removes_the_reflection_and_yields_add_up():
    """A free-ish outgoing wavepacket in l = 3 (weak Coulomb tail) hits the wall at r_max: without absorber the norm
    stays 1 and the packet comes back (p_b recovers); with it the outgoing flux is removed.  p_i + p_b = 1 (Eq. 28)."""
    g = oracle.make_grid(600, 0.25, 4, 3)
    r = g.dr * np.arange(1, g.n_r + 1)
    psi = np.zeros((1, 4, g.n_r), dtype=np.complex128)
    psi[0, 3] = np.exp(-(r - 60.0) ** 2 / 50.0) * np.exp(2.0j * r)           # k = 2 au outwards
    psi /= math.sqrt(g.dr * np.sum(np.abs(psi) ** 2))
    pulse = [(0.0, 0.057, 2.0, 0.0)]                                         # no field
    dt, nsteps = 0.01, 9000                                                  # travels 180 au: to the wall (150) and back

    def step(x, t, n):
        return oracle.step_taylor(g, pulse, x, 8, t, dt, n)[0]
    free = step(psi, 0.0, nsteps)
    assert abs(g.dr * np.sum(np.abs(free) ** 2) - 1.0) < 1e-9
    pb = oracle.bound_population(g, free, 100.0)
    assert abs(pb[0] + (g.dr * np.sum(np.abs(free[0][:, r > 100.0]) ** 2)) - 1.0) < 1e-9   # Eq. 28
    assert pb[0] > 0.5                                                        # reflected: back inside r < 100
    # p = 200 confines the absorbing layer to the last tenth of the box (1 - M = cos^200 < 1e-9 for r < 0.6 r_b)
    mask = oracle.absorber_mask(g, g.dr * (g.n_r + 1), 200)
    early = oracle.step_masked(step, g, psi, mask, 0.0, dt, 1500)            # packet at r ~ 90: not yet in the layer
    assert abs(g.dr * np.sum(np.abs(early) ** 2) - 1.0) < 1e-6
    absd = oracle.step_masked(step, g, early, mask, 1500 * dt, dt, nsteps - 1500)
    assert g.dr * np.sum(np.abs(absd) ** 2) < 0.02                            # the outgoing flux was absorbed
    assert oracle.bound_population(g, absd, 100.0)[0] < 0.02                  # ... and did not come back


# ------------------------------------------------------------------------------------ velocity gauge (P13, NEXT f1)
def _dense_velocity_H(n_r, dr, n_l, fd, a_field):
    """H of P:106 Eq. 12 (1/r terms in reading R-V2) built entry by entry in numpy, independently of the oracle."""
    r = dr * np.arange(1, n_r + 1)
    n = n_r * n_l
    h = np.zeros((n, n), dtype=np.complex128)
    if fd == 3:
        d2 = {0: -2.0, 1: 1.0, -1: 1.0}; s2 = 1.0 / dr ** 2
        d1 = {1: 1.0, -1: -1.0}; s1 = 1.0 / (2 * dr)
    else:
        d2 = {0: -30.0, 1: 16.0, -1: 16.0, 2: -1.0, -2: -1.0}; s2 = 1.0 / (12 * dr ** 2)
        d1 = {1: 8.0, -1: -8.0, 2: -1.0, -2: 1.0}; s1 = 1.0 / (12 * dr)
    kap = lambda l: l / math.sqrt(4.0 * l * l - 1.0) if l > 0 else 0.0     # kappa_l = k_{l,l-1}(m = 0), Eq. 9
    for l in range(n_l):
        for j in range(n_r):
            row = l * n_r + j
            for k, w in d2.items():
                if 0 <= j + k < n_r:
                    h[row, l * n_r + j + k] += -0.5 * w * s2
            h[row, row] += l * (l + 1) / (2 * r[j] ** 2) - 1.0 / r[j]
            for lp, kp, sgn in ((l - 1, kap(l), -l), (l + 1, kap(l + 1), +(l + 1))):      # reading R-V2
                if 0 <= lp < n_l:
                    for k, w in d1.items():
                        if 0 <= j + k < n_r:
                            h[row, lp * n_r + j + k] += -1j * a_field * kp * w * s1
                    h[row, lp * n_r + j] += -1j * a_field * kp * sgn / r[j]
    return h


@pytest.mark.parametrize("fd", [3, 5])
def test_P13_velocity_gauge_operator(fd):
    """The oracle's matrix-free velocity-gauge H equals the dense matrix written out from Eq. 12 / Eq. 14 column by
    column, is Hermitian, and reduces to the field-free h_l at A = 0."""
    n_r, dr, n_l, a = 14, 0.2, 4, 0.37
    g = oracle.make_grid(n_r, dr, n_l, fd, gauge=1)
    h = _dense_velocity_H(n_r, dr, n_l, fd, a)
    assert np.max(np.abs(h - h.conj().T)) < 1e-12
    cols = np.zeros((n_r * n_l, n_r * n_l), dtype=np.complex128)
    for c in range(n_r * n_l):
        e = np.zeros(n_r * n_l, dtype=np.complex128); e[c] = 1.0
        cols[:, c] = oracle.apply_H(g, e.reshape(1, n_l, n_r), a).ravel()
    assert np.max(np.abs(cols - h)) < 1e-12 * np.max(np.abs(h))
    x = rand_state((1, n_l, n_r), 77)
    g0 = oracle.make_grid(n_r, dr, n_l, fd, gauge=0)
    assert np.max(np.abs(oracle.apply_H(g, x, 0.0) - oracle.apply_H(g0, x, 0.0))) == 0.0


def test_P13_velocity_gauge_propagators_against_dense_exponential():
    """Static A (test aid): Taylor, RK4 and Lanczos steps against scipy's expm of the independently built dense H."""
    n_r, dr, n_l, a, dt = 40, 0.2, 3, 0.25, 0.004
    g = oracle.make_grid(n_r, dr, n_l, 5, gauge=1)
    u = sla.expm(-1j * dt * _dense_velocity_H(n_r, dr, n_l, 5, a))
    psi = rand_state((1, n_l, n_r), 5)
    ref = (u @ psi.ravel()).reshape(psi.shape)
    static = [(a, 0.0, 1.0, 0.0, 1)]
    assert np.linalg.norm(oracle.step_taylor(g, static, psi, 14, 0.0, dt, 1)[0] - ref) < 1e-12 * np.linalg.norm(ref)
    assert np.linalg.norm(oracle.step_lanczos(g, static, psi, 30, 14, 0.0, dt, 1)[0] - ref) < 1e-9 * np.linalg.norm(ref)
    y = float(np.max(np.abs(np.linalg.eigvalsh(_dense_velocity_H(n_r, dr, n_l, 5, a))))) * dt
    assert np.linalg.norm(oracle.step_rk4(g, static, psi, 0.0, dt, 1)[0] - ref) < 1.01 * y ** 5 / 120 * np.linalg.norm(ref)


def test_P13_vector_potential_pulse_and_gauge_agreement():
    """Kind-1 pulse (Hann shape on A, R-V3): E = -dA/dt, A vanishes at both ends, peak field ~ e0; and a
    short pulse gives the same ground-state depletion in both gauges up to the discretisation (it differs between
    the gauges at finite dr and l truncation; the paper quotes 0.27145 vs 0.27144 on a converged grid)."""
    p = (0.0534, 0.057, 4.0, 0.3, 1)
    T = 2 * math.pi * p[2] / p[1]
    ts = np.linspace(0.01, T - 0.01, 301)
    hh = 1e-5
    num = np.array([-(oracle.pulse_A(p, t + hh) - oracle.pulse_A(p, t - hh)) / (2 * hh) for t in ts])
    ana = np.array([oracle.pulse_E(p, t) for t in ts])
    assert np.max(np.abs(num - ana)) < 1e-8
    assert oracle.pulse_A(p, 0.0) == 0.0 and abs(oracle.pulse_A(p, T)) < 1e-15 and oracle.pulse_A(p, T + 1.0) == 0.0
    assert 0.9 * p[0] < np.max(np.abs(ana)) <= 1.05 * p[0]
    assert math.isnan(oracle.pulse_A((0.05, 0.057, 2.0, 0.0, 0), 1.0))          # kind 0: no closed form here (running quadrature, P16)
    # depletion of 1s by a one-cycle pulse at omega = 0.6 au (one-photon ionisation), both gauges
    n_r, dr, n_l, dt = 400, 0.2, 6, 0.004
    pulse = [(0.15, 0.6, 3.0, 0.0, 1)]
    Tp = 2 * math.pi * 3.0 / 0.6
    nsteps = int(math.ceil(Tp / dt)); dt = Tp / nsteps
    dep = []
    for gauge in (0, 1):
        g = oracle.make_grid(n_r, dr, n_l, 5, gauge=gauge)
        _, phi = oracle.bound_states(oracle.make_grid(n_r, dr, n_l, 5), 0, 1)
        psi = np.zeros((1, n_l, n_r), dtype=np.complex128); psi[0, 0] = phi[0]
        out, _ = oracle.step_taylor(g, pulse, psi, 4, 0.0, dt, nsteps)
        assert abs(dr * np.sum(np.abs(out) ** 2) - 1.0) < 1e-8
        dep.append(1.0 - abs(np.vdot(phi[0], out[0, 0]) * dr) ** 2)
    assert dep[0] > 0.01                                                         # the pulse does ionise
    assert abs(dep[0] - dep[1]) < 0.05 * dep[0]


# ------------------------------------------------------------------------------- the other RK methods of P:796 (P14)
def _order_conditions(c, a, b, order):
    """Rooted-tree order conditions up to `order` (<= 5) in exact rationals; a as a list of rows."""
    F = Fraction
    s = len(c)
    A = [[a[i][j] if j < len(a[i]) else F(0) for j in range(s)] for i in range(s)]
    dot = lambda u, v: sum(x * y for x, y in zip(u, v))
    Av = lambda v: [dot(A[i], v) for i in range(s)]
    mul = lambda u, v: [x * y for x, y in zip(u, v)]
    one = [F(1)] * s
    c2, c3 = mul(c, c), mul(mul(c, c), c)
    Ac, Ac2, Ac3 = Av(c), Av(c2), Av(c3)
    AAc, AAc2 = Av(Ac), Av(Ac2)
    conds = {1: [(one, F(1))],
             2: [(c, F(1, 2))],
             3: [(c2, F(1, 3)), (Ac, F(1, 6))],
             4: [(c3, F(1, 4)), (mul(c, Ac), F(1, 8)), (Ac2, F(1, 12)), (AAc, F(1, 24))],
             5: [(mul(c3, c), F(1, 5)), (mul(c2, Ac), F(1, 10)), (mul(c, Ac2), F(1, 15)), (mul(c, AAc), F(1, 30)),
                 (mul(Ac, Ac), F(1, 20)), (Ac3, F(1, 20)), (Av(mul(c, Ac)), F(1, 40)), (AAc2, F(1, 60)),
                 (Av(AAc), F(1, 120))]}
    ok = True
    for q in range(1, order + 1):
        for vec, rhs in conds[q]:
            ok = ok and dot(b, vec) == rhs
    return ok


def test_P14_rk_tableaux_order_conditions():
    """RKF 4(5), Cash-Karp 5(4) and Kutta-Merson 4(3) as typed into the oracle: row sums = c and ALL order conditions of
    the stated orders for both weight rows, in exact rationals; the lower-order row fails the next order."""
    F = Fraction
    tabs = {
        "rkf": ([F(0), F(1, 4), F(3, 8), F(12, 13), F(1), F(1, 2)],
                [[], [F(1, 4)], [F(3, 32), F(9, 32)], [F(1932, 2197), F(-7200, 2197), F(7296, 2197)],
                 [F(439, 216), F(-8), F(3680, 513), F(-845, 4104)],
                 [F(-8, 27), F(2), F(-3544, 2565), F(1859, 4104), F(-11, 40)]],
                [F(16, 135), F(0), F(6656, 12825), F(28561, 56430), F(-9, 50), F(2, 55)], 5,
                [F(25, 216), F(0), F(1408, 2565), F(2197, 4104), F(-1, 5), F(0)], 4),
        "cashkarp": ([F(0), F(1, 5), F(3, 10), F(3, 5), F(1), F(7, 8)],
                     [[], [F(1, 5)], [F(3, 40), F(9, 40)], [F(3, 10), F(-9, 10), F(6, 5)],
                      [F(-11, 54), F(5, 2), F(-70, 27), F(35, 27)],
                      [F(1631, 55296), F(175, 512), F(575, 13824), F(44275, 110592), F(253, 4096)]],
                     [F(37, 378), F(0), F(250, 621), F(125, 594), F(0), F(512, 1771)], 5,
                     [F(2825, 27648), F(0), F(18575, 48384), F(13525, 55296), F(277, 14336), F(1, 4)], 4),
        "merson": ([F(0), F(1, 3), F(1, 3), F(1, 2), F(1)],
                   [[], [F(1, 3)], [F(1, 6), F(1, 6)], [F(1, 8), F(0), F(3, 8)], [F(1, 2), F(0), F(-3, 2), F(2)]],
                   [F(1, 6), F(0), F(0), F(2, 3), F(1, 6)], 4,
                   [F(1, 10), F(0), F(3, 10), F(2, 5), F(1, 5)], 3),
    }
    for name, (c, a, b, pb, bh, pbh) in tabs.items():
        for i in range(len(c)):
            assert sum(a[i], F(0)) == c[i], name
        assert _order_conditions(c, a, b, pb), name
        assert _order_conditions(c, a, bh, pbh), name
        assert not _order_conditions(c, a, bh, pbh + 1), name
        if pb < 5:
            assert not _order_conditions(c, a, b, pb + 1), name


def test_P14_rk_methods_convergence_and_sigma():
    """Every method of P:796 on the tiny grid against a converged Taylor step: the error falls with its order when dt
    halves (pins the oracle's typed-in coefficients and stage times); Euler is Taylor order 1 exactly; sigma is the
    sum over steps of sqrt(|F2 - F1|^2 / M), zero for the methods without a pair."""
    g = tiny(5)
    psi = rand_state((1, g.n_l, g.n_r), 3); psi /= math.sqrt(g.dr * np.sum(np.abs(psi) ** 2))
    pulse = [(0.3, 2.0, 1.0, 0.2)]                                        # fast field: the stage times matter
    t0, span = 0.4, 0.02
    ref = oracle.step_taylor(g, pulse, psi, 8, t0, span / 400, 400)[0]
    order = {"euler": 1, "rk4": 4, "merson": 4, "rkf": 5, "cashkarp": 5, "dormandprince": 5}
    for m, p in order.items():
        errs, sig = [], []
        for n in (10, 20):
            out, s, _ = oracle.step_rk_method(g, pulse, psi, m, t0, span / n, n)
            errs.append(np.linalg.norm(out - ref)); sig.append(s[0])
        assert 0.8 * 2 ** p < errs[0] / errs[1] < 1.25 * 2 ** p, (m, errs)
        if m in ("euler", "rk4"):
            assert sig == [0.0, 0.0]
        else:
            lo = 3 if m == "merson" else 4      # order of the companion: Delta = O(dt^(lo+1)) per step, n = O(1/dt) steps
            assert sig[0] > 0 and 0.6 * 2 ** lo < sig[0] / sig[1] < 1.4 * 2 ** (lo + 1), (m, sig)   # (linear ODE: Merson gains one)
    e1 = oracle.step_rk_method(g, pulse, psi, "euler", t0, 1e-3, 7)[0]
    t1 = oracle.step_taylor(g, pulse, psi, 1, t0, 1e-3, 7, field_sample=1)[0]
    assert np.linalg.norm(e1 - t1) <= 1e-15 * np.linalg.norm(t1)
    # sigma of one Dormand-Prince step against the difference of the two solutions formed by hand from err of
    # oracle.step_rk_fixed (relative definition) -- same Delta, different normalisation
    out, s, _ = oracle.step_rk_method(g, pulse, psi, "dormandprince", t0, 2e-3, 1)
    _, rel, _ = oracle.step_rk_fixed(g, pulse, psi, 1, t0, 2e-3, 1)
    m_el = g.n_l * g.n_r
    assert abs(s[0] - rel[0] * np.linalg.norm(out) / math.sqrt(m_el)) <= 1e-12 * s[0]


# --------------------------------------------------------------- centrifugal inner cut-off (P15, NEXT f4: an extension)
def plain_held(n_r, dr, n_l, lam):
    """The definition written out: point (l, j) is held at zero iff l(l+1)/(2 r_j^2) > Lambda."""
    r = dr * np.arange(1, n_r + 1)
    l = np.arange(n_l)[:, None]
    return l * (l + 1) / (2.0 * r[None, :] ** 2) > lam


@pytest.mark.parametrize("fd", [3, 5])
def test_P15_cutoff_is_the_principal_submatrix(fd):
    """With a cut-off the dense H is the un-cut H on the points that are not held and zero elsewhere (a principal
    sub-matrix: still exactly symmetric); the matrix-free operator equals it column by column; its spectral radius obeys
    kappa_G/dr^2 + Lambda + E0 r_max (LAPACK) while the un-cut radius is dominated by the centrifugal term at r_1."""
    n_r, dr, n_l, lam, e = 60, 0.1, 7, 40.0, 0.07
    g0 = oracle.make_grid(n_r, dr, n_l, fd)
    gc = oracle.make_grid(n_r, dr, n_l, fd, cutoff_lambda=lam)
    held = plain_held(n_r, dr, n_l, lam)
    assert np.array_equal(oracle.held_mask(gc), held)
    assert held.sum() > 10 and not held[0].any() and held[-1, 0] and not held[-1, -1]
    h0, hc = oracle.dense_H(g0, e), oracle.dense_H(gc, e)
    act = ~held.ravel()
    expect = np.where(np.outer(act, act), h0, 0.0)
    assert np.array_equal(hc, expect)
    assert np.array_equal(hc, hc.T)
    x = rand_state((1, n_l, n_r), 77)
    y = oracle.apply_H(gc, x, e)
    assert np.max(np.abs(y.ravel() - hc @ x.ravel())) <= 1e-12 * np.max(np.abs(y))
    assert np.count_nonzero(y[0][held]) == 0
    kg = 2.0 if fd == 3 else 8.0 / 3.0
    rho_c = np.max(np.abs(np.linalg.eigvalsh(hc)))
    rho_0 = np.max(np.abs(np.linalg.eigvalsh(h0)))
    assert rho_c <= kg / dr ** 2 + lam + e * n_r * dr
    assert rho_0 > (n_l - 1) * n_l / (2 * dr ** 2) and rho_0 > 5 * rho_c
    # the same bound is what the step-size rule uses
    c = dict(n_r=n_r, dr=dr, n_l=n_l, fd_order=fd, batch=1, intensity=1e14, lam_nm=800.0, n_cycles=2, cutoff_lambda=lam)
    c["omega"] = wl.omega_of_nm(800.0)
    assert wl.rho_gershgorin(c, e0_max=e) >= rho_c


def test_P15_cutoff_stabilises_the_step_and_converges_with_lambda():
    """Purpose and harmlessness of the cut-off (the paper only says Taylor is "not always stable",
    P:454).  Hydrogen from the discrete 1s state through a whole 2-cycle pulse (omega = 0.6, E0 = 0.25), L = 10:
    (i) at 2.5/rho of the CUT operator the cut Taylor-4 run keeps the norm to 1e-10 and the held points exactly zero, in
    13 to 19 times fewer steps, while the un-cut operator overflows at that step; (ii) the 1s population, the dipole and
    the l <= 2 blocks converge to the un-cut run (at its own, much smaller stable step) as Lambda grows: 3e-2, 2e-3,
    1e-6 relative at Lambda = 10, 40, 160; (iii) a Lambda that holds no point is bit-identical to no cut-off."""
    n_r, dr, n_l = 200, 0.1, 10
    e0, om = 0.25, 0.6
    c = wl.config("cfg1", n_r=n_r, dr=dr, n_l=n_l, fd_order=3, intensity=e0 ** 2 * wl.AU_INTENSITY_W_CM2)
    pulses = [(e0, om, 2.0, 0.0)]
    t_run = 2 * math.pi * 2.0 / om
    g0 = oracle.make_grid(n_r, dr, n_l, 3)
    _, phi = oracle.bound_states(g0, 0, 1)
    st = (np.array([0], dtype=np.int32), phi)
    psi0 = wl.ground_state(c, phi[0])
    oracle.set_threads(4)
    res = {}
    for lam in (0.0, 10.0, 40.0, 160.0):
        dt = wl.dt_eff(dict(c, cutoff_lambda=lam), "taylor", 4, t_run=t_run)
        n = int(round(t_run / dt))
        g = oracle.make_grid(n_r, dr, n_l, 3, cutoff_lambda=lam)
        psi, rows = oracle.step_taylor(g, pulses, psi0, 4, 0.0, dt, n, states=st, obs_every=n)
        assert np.count_nonzero(psi[0][oracle.held_mask(g)]) == 0
        assert abs(rows[-1, 0, 0] - 1.0) <= 1e-10                        # (i) norm
        res[lam] = (n, rows[-1, 0], psi)
    oracle.set_threads(1)
    assert res[0.0][0] > 12 * res[160.0][0] and res[0.0][0] > 18 * res[10.0][0]
    dt = t_run / res[40.0][0]
    bad, _ = oracle.step_taylor(g0, pulses, psi0, 4, 0.0, dt, 400)       # the un-cut operator at the cut run's step
    assert not np.all(np.isfinite(bad.view(np.float64))) or np.max(np.abs(bad)) > 1e6
    ref = res[0.0]
    assert 0.2 < ref[1][3] < 0.5 and abs(ref[1][1]) > 0.1                # the pulse did something (p_1s = 0.313)
    low = [np.linalg.norm(res[lam][2][0, :3] - ref[2][0, :3]) / np.linalg.norm(ref[2][0, :3]) for lam in (10.0, 40.0, 160.0)]
    pop = [abs(res[lam][1][3] - ref[1][3]) for lam in (10.0, 40.0, 160.0)]
    dip = [abs(res[lam][1][1] - ref[1][1]) for lam in (10.0, 40.0, 160.0)]
    assert low[0] > 10 * low[1] > 100 * low[2] and low[2] <= 1e-5        # (ii)
    assert pop[0] > pop[1] > pop[2] and pop[2] <= 1e-6 and dip[0] > dip[1] > dip[2] and dip[2] <= 1e-5
    g_big = oracle.make_grid(n_r, dr, n_l, 3, cutoff_lambda=1e9)          # (iii)
    assert not oracle.held_mask(g_big).any()
    a, _ = oracle.step_taylor(g_big, pulses, psi0, 4, 0.0, 1e-4, 20)
    b, _ = oracle.step_taylor(g0, pulses, psi0, 4, 0.0, 1e-4, 20)
    assert np.array_equal(a, b)


def test_P15_cutoff_in_every_propagator_against_the_dense_exponential():
    """RK4, Dormand-Prince, Lanczos and imaginary time all go through the same P H P: each against scipy's expm of the
    cut dense matrix at a frozen field."""
    n_r, dr, n_l, lam, e = 50, 0.2, 5, 15.0, 0.05
    g = oracle.make_grid(n_r, dr, n_l, 5, cutoff_lambda=lam)
    hc = oracle.dense_H(g, e)
    psi0 = oracle.project(g, rand_state((1, n_l, n_r), 5))
    psi0 /= math.sqrt(dr * np.sum(np.abs(psi0) ** 2))
    dt, n = 2e-4, 10                                  # y = dt rho = 0.02: RK4's y^5/120 per step is far below 1e-9
    exact = (sla.expm(-1j * hc * dt * n) @ psi0.ravel()).reshape(psi0.shape)
    static = (e, 0.0, 1.0, 0.0)
    for name, got in (("rk4", oracle.step_rk4(g, static, psi0, 0.0, dt, n)[0]),
                      ("dp", oracle.step_rk_fixed(g, static, psi0, 1, 0.0, dt, n)[0]),
                      ("lanczos", oracle.step_lanczos(g, static, psi0, 12, 12, 0.0, dt, n)[0]),
                      ("taylor", oracle.step_taylor(g, static, psi0, 8, 0.0, dt, n)[0])):
        assert np.linalg.norm(got - exact) <= 1e-9, name
        assert np.count_nonzero(got[0][oracle.held_mask(g)]) == 0, name


# ---------------------------------------------------- vector potential by the running Gauss quadrature (P16, f1 widened)
def _closed_form_A_kind0(e0, om, nc, t):
    """A(t) = -int_0^t e0 sin^2(om t'/(2 nc)) cos(om t') dt' in closed form (cep = 0): sin^2 = (1 - cos 2 Om t)/2."""
    Om = om / (2.0 * nc)
    return -0.5 * e0 * (np.sin(om * t) / om - np.sin((om + 2 * Om) * t) / (2 * (om + 2 * Om))
                        - np.sin((om - 2 * Om) * t) / (2 * (om - 2 * Om)))


def test_P16_running_quadrature_against_the_analytic_vector_potential():
    """The paper's Fig. 8: the vector potential from the running 5-point Gauss quadrature of the field
     against the analytic one -- for the Hann-shaped A (kind 1, E = -dA/dt fed to the quadrature) and for the
    ordinary sin^2 pulse (kind 0, closed form above); from t = 0 and from a start inside the pulse (reading R-V4); the
    5-point rule is exact for polynomials of degree 9, so halving a coarse step cuts the error by about 2^10."""
    p1 = (0.1688, 0.3675, 10.0, 0.0, 1)                 # 1e15 W/cm^2, 10 eV, 10 cycles: the pulse of Fig. 8
    T = 2 * math.pi * p1[2] / p1[1]
    dt = 0.05
    n = int(T / dt)
    a = oracle.vecpot_running(p1, 0.0, dt, n)
    ref = np.array([oracle.pulse_A(p1, k * dt) for k in range(n + 1)])
    assert np.max(np.abs(ref)) > 0.4 and np.max(np.abs(a - ref)) <= 1e-13
    a = oracle.vecpot_running(p1, 33.37, dt, 500)       # starts inside the pulse, off the panel grid
    ref = np.array([oracle.pulse_A(p1, 33.37 + k * dt) for k in range(501)])
    assert np.max(np.abs(a - ref)) <= 1e-13
    e0, om, nc = 0.0534, 0.057, 4.0
    p0 = (e0, om, nc, 0.0, 0)
    T = 2 * math.pi * nc / om
    for t0 in (0.0, 101.3):
        a = oracle.vecpot_running(p0, t0, 0.5, 300)
        ts = t0 + 0.5 * np.arange(301)
        assert np.max(np.abs(a - _closed_form_A_kind0(e0, om, nc, ts))) <= 1e-13
    assert abs(oracle.vecpot_running(p0, 0.0, T / 400, 400)[-1]) <= 1e-13        # a whole pulse integrates to zero
    errs = []
    for h in (40.0, 20.0):                                                       # coarse panels: convergence order
        a = oracle.vecpot_running(p0, 0.0, h, int(200 / h))
        errs.append(abs(a[-1] - _closed_form_A_kind0(e0, om, nc, 200.0)))
    assert errs[1] < errs[0] / 300
    # one rule alone: exact on a constant field, antisymmetric in its limits
    assert abs(oracle.gl5_field_integral((0.3, 0.0, 1.0, 0.0, 0), 1.0, 3.5) - 0.75) <= 1e-15
    assert oracle.gl5_field_integral(p0, 10.0, 12.0) == -oracle.gl5_field_integral(p0, 12.0, 10.0)


def test_P16_velocity_gauge_propagators_with_a_field_pulse():
    """Velocity-gauge propagation under an ordinary (kind-0) pulse: Taylor and Lanczos freeze H at A(t_n + dt/2) =
    A(t_n) - int_{t_n}^{t_n+dt/2} E (P:480 with c_i = 1/2), RK4 takes A at its stage times; each against numpy on the
    independently built dense H (P13) with the CLOSED-FORM A(t) at those times."""
    n_r, dr, n_l, fd = 30, 0.2, 3, 5
    e0, om, nc = 0.4, 0.9, 2.0
    pulse = [(e0, om, nc, 0.0, 0)]
    g = oracle.make_grid(n_r, dr, n_l, fd, gauge=1)
    psi0 = rand_state((1, n_l, n_r), 9)
    psi0 /= math.sqrt(dr * np.sum(np.abs(psi0) ** 2))
    t0, dt, n = 2.31, 2e-3, 12
    A = lambda t: float(_closed_form_A_kind0(e0, om, nc, t))
    H = lambda t: _dense_velocity_H(n_r, dr, n_l, fd, A(t))
    # Taylor / Lanczos: product of frozen-midpoint exponentials
    ref = psi0.ravel().copy()
    for k in range(n):
        ref = sla.expm(-1j * dt * H(t0 + (k + 0.5) * dt)) @ ref
    got = oracle.step_taylor(g, pulse, psi0, 14, t0, dt, n)[0]
    assert np.linalg.norm(got.ravel() - ref) <= 1e-11
    got = oracle.step_lanczos(g, pulse, psi0, 30, 14, t0, dt, n)[0]
    assert np.linalg.norm(got.ravel() - ref) <= 1e-9
    # classic RK4 with H at the stage times, written out in numpy
    y = psi0.ravel().copy()
    f = lambda t, v: -1j * (H(t) @ v)
    for k in range(n):
        t = t0 + k * dt
        k1 = f(t, y); k2 = f(t + dt / 2, y + dt / 2 * k1); k3 = f(t + dt / 2, y + dt / 2 * k2); k4 = f(t + dt, y + dt * k3)
        y = y + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    got = oracle.step_rk4(g, pulse, psi0, t0, dt, n)[0]
    assert np.linalg.norm(got.ravel() - y) <= 1e-12
    # and the sign convention ties in with the analytic pulses: the SAME physical pulse given as kind 1 (A analytic) and
    # as its field integrated numerically must propagate identically -- here through apply_H at equal A
    p1 = (0.2, 0.6, 3.0, 0.0, 1)
    a_run = oracle.vecpot_running(p1, 0.0, 0.01, 500)[-1]
    assert abs(a_run - oracle.pulse_A(p1, 5.0)) <= 1e-14
