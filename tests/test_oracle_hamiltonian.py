"""Pins for oracle.hamiltonian / gradient / rhs (CPU only).

Each test ties the oracle to something other than itself: a closed form from the literature the
paper points to, a textbook limit, an exact algebraic identity, or a value the paper
prints (tests/golden/paper_coefficients.txt).  See DESIGN.md "Oracle pins".
"""
import os

import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.optimize import brentq

import oracle
from conftest import random_states

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_coefficients.txt")
ALL_MASKS = [0, 1, 3, 4, 8, 16, 7, 15, 31, 28]


def golden(name, beta=None):
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if len(line) == 3 and line[0] == name and (beta is None or abs(float(line[1]) - beta) < 1e-12):
            return float(line[2])
    raise KeyError(name)


def eta_of(beta):
    return beta / (1 + beta) ** 2


# ---- orbital part -----------------------------------------------------------------------------

def test_test_particle_limit_is_schwarzschild_in_isotropic_coordinates():
    """eta -> 0: H_N+1PN+2PN must be the 2PN expansion of the geodesic Hamiltonian of Schwarzschild in
    isotropic (= ADM) coordinates, H = (1-u/2)/(1+u/2) sqrt(1 + p^2/(1+u/2)^4) - 1, u = 1/r: the
    difference is 3PN, i.e. O(u^4) when p^2 ~ u.  Pins all eta^0 coefficients, off-circular too."""
    rng = np.random.default_rng(7)
    scaled = []
    for scale in (30.0, 300.0, 3000.0):
        for _ in range(4):
            r = rng.normal(size=3)
            r *= scale / np.linalg.norm(r)
            p = rng.normal(size=3)
            p *= rng.uniform(0.6, 1.2) / np.sqrt(scale) / np.linalg.norm(p)
            z = np.zeros(12)
            z[:3], z[3:6], z[6], z[9] = r, p, 1, 1
            u, P = 1 / scale, p @ p
            exact = (1 - u / 2) / (1 + u / 2) * np.sqrt(1 + P / (1 + u / 2) ** 4) - 1
            H = oracle.hamiltonian(z, beta=1e-13, terms=3)[0]
            scaled.append((H - exact) * scale ** 4)
    scaled = np.array(scaled)
    assert np.all(np.abs(scaled) < 12.0), scaled          # 3PN-sized residual at every scale
    # dropping or changing a 2PN coefficient would leave a residual ~ scale * O(1) here
    assert np.abs(scaled[-4:]).max() < 12.0 and np.abs(scaled[:4]).max() < 12.0


def _circular(beta, r0, terms=3):
    """p_y of the circular orbit through (r0,0,0) and its (E, Omega_phi)."""
    def radial_force(py):          # d(r.p)/dt = 0 with r.p = 0: the orbit stays at r = r0
        z = np.zeros(12)
        z[0], z[4], z[8], z[11] = r0, py, 1, 1
        f = oracle.rhs(z, beta=beta, terms=terms)[:, 0]
        return f[0:3] @ z[3:6] + z[0:3] @ f[3:6]
    py = brentq(radial_force, 0.5 / np.sqrt(r0), 2.0 / np.sqrt(r0), xtol=1e-18, rtol=1e-15)
    z = np.zeros(12)
    z[0], z[4], z[8], z[11] = r0, py, 1, 1
    return oracle.hamiltonian(z, beta=beta, terms=terms)[0], oracle.rhs(z, beta=beta, terms=terms)[1, 0] / r0


@pytest.mark.parametrize("beta", [1.0, 1.0 / 3.0, 0.127])
def test_circular_orbit_binding_energy_matches_2pn_closed_form(beta):
    """Gauge-invariant E(x), x = Omega^(2/3):  E = -(x/2)[1 - (3/4 + eta/12) x
    - (27/8 - 19 eta/8 + eta^2/24) x^2] + O(x^4)   (Blanchet, Living Rev. Relativ.; 2PN)."""
    eta = eta_of(beta)
    c1, c2 = 0.75 + eta / 12, 27 / 8 - 19 * eta / 8 + eta * eta / 24
    res3, res4 = [], []
    for r0 in (50.0, 200.0, 800.0):
        E, Om = _circular(beta, r0)
        x = Om ** (2.0 / 3.0)
        res3.append((E + 0.5 * x * (1 - c1 * x)) / x ** 3)
        res4.append((E + 0.5 * x * (1 - c1 * x - c2 * x * x)) / x ** 4)
    assert abs(res3[-1] / (0.5 * c2) - 1) < 0.02, res3     # 2PN coefficient resolved
    assert np.all(np.abs(res4) < 10.0), res4               # remainder is 3PN-sized
    assert abs(res4[-1] - res4[-2]) < 0.5, res4            # and converges to a constant


def _radial_period_and_advance(beta, r0, f, terms=3):
    """Start at apocentre (r0,0,0), p = (0, f/sqrt(r0), 0), f < 1; integrate the oracle's RHS with
    DOP853 to the next apocentre: returns k = Phi/2pi - 1, n = 2pi/T_r, E, h = |L|."""
    z0 = np.zeros(12)
    z0[0], z0[4], z0[8], z0[11] = r0, f / np.sqrt(r0), 1, 1
    E = oracle.hamiltonian(z0, beta=beta, terms=terms)[0]
    h = r0 * z0[4]

    def fun(t, y):
        z = np.zeros(12)
        z[:6], z[8], z[11] = y, 1, 1
        return oracle.rhs(z, beta=beta, terms=terms)[:6, 0]

    def apo(t, y):
        return y[0] * y[3] + y[1] * y[4]
    apo.direction = -1
    T0 = 2 * np.pi * (-1 / (2 * E)) ** 1.5
    sol = solve_ivp(fun, [0, 1.5 * T0], z0[:6], method="DOP853", rtol=1e-13, atol=1e-18, events=apo)
    sel = sol.t_events[0] > 0.1 * T0
    t_apo, y_apo = sol.t_events[0][sel][0], sol.y_events[0][sel][0]
    phi = np.arctan2(y_apo[1], y_apo[0]) % (2 * np.pi)
    return phi / (2 * np.pi), 2 * np.pi / t_apo, E, h


@pytest.mark.parametrize("beta,f", [(1.0, 0.8), (1.0, 0.45), (0.5, 0.5), (0.2, 0.85)])
def test_eccentric_orbit_periastron_advance_and_radial_period_match_2pn(beta, f):
    """Damour & Schaefer (1988) gauge-invariant 2PN functions of E (per mu) and h = |L|:
       k   = 3/h^2 + (3/2)(5-2 eta) E/h^2 + (15/4)(7-2 eta)/h^4
       n   = e^(3/2) {1 + (e/8)(-15+eta) + (e^2/128)[555 + 30 eta + 11 eta^2 - 192(5-2 eta)/sqrt(e h^2)]},
       e = -2E.  Eccentric orbits exercise every (n.p)-dependent coefficient of H_1PN and H_2PN."""
    eta = eta_of(beta)
    rk, rn = [], []
    for r0 in (1600.0, 6400.0):
        k, n, E, h = _radial_period_and_advance(beta, r0, f)
        e = -2 * E
        k_th = 3 / h ** 2 + 1.5 * (5 - 2 * eta) * E / h ** 2 + 3.75 * (7 - 2 * eta) / h ** 4
        n_th = e ** 1.5 * (1 + e / 8 * (-15 + eta) + e * e / 128 *
                           (555 + 30 * eta + 11 * eta ** 2 - 192 * (5 - 2 * eta) / np.sqrt(e * h * h)))
        rk.append((k - k_th) * h ** 6)
        rn.append((n / n_th - 1) / e ** 3)
        # the 2PN part itself is resolved to a few per cent (3PN remainder / 2PN term ~ 10/h^2)
        k_2pn = k_th - 3 / h ** 2
        assert abs((k - 3 / h ** 2) / k_2pn - 1) < 30.0 / h ** 2 + 1e-6
    assert np.all(np.abs(rk) < 400.0), rk
    assert np.all(np.abs(rn) < 200.0), rn
    assert abs(rn[1] - rn[0]) < 0.03 * abs(rn[0]) + 0.5, rn
    # the remainder is a pure 3PN term: a 2PN coefficient wrong by c would add c*h^2 to rk, i.e. change
    # it by ~c*3000 between the two radii (mutation-checked down to the eta^2 (n.p)^4 term)
    assert abs(rk[1] - rk[0]) < 2.5, rk


# ---- gradient and equations of motion ----------------------------------------------------------

@pytest.mark.parametrize("terms", ALL_MASKS)
def test_gradient_matches_finite_differences_of_H(terms):
    """4th-order central differences of the oracle's H in all 12 directions (north_star pin)."""
    z = random_states(6, seed=100 + terms)
    kw = dict(beta=np.linspace(0.3, 1.0, 6), chi1=0.9, chi2=0.7, kq1=2.5, kq2=4.0, terms=terms)
    g = oracle.gradient(z, **kw)
    s1 = kw["chi1"] * kw["beta"]
    s2 = kw["chi2"] / kw["beta"]
    blocks = [np.linalg.norm(z[0:3], axis=0), np.linalg.norm(z[3:6], axis=0), np.ones(6), np.ones(6)]
    for i in range(12):
        step = 5e-4 * blocks[i // 3]                      # per-orbit step, relative to |r|, |p|, 1
        d = np.zeros_like(z)
        d[i] = step
        H = lambda a: oracle.hamiltonian(z + a * d, **kw)
        fd = (8 * (H(1) - H(-1)) - (H(2) - H(-2))) / (12 * step)
        if i >= 9:
            fd = fd / s2      # dH/dS2 = (1/s2) dH/dS2hat
        elif i >= 6:
            fd = fd / s1
        b = 3 * (i // 3)
        scale = np.linalg.norm(g[b:b + 3], axis=0) + 1e-7
        assert np.all(np.abs(fd - g[i]) < 1e-9 * scale), (terms, i, np.abs(fd - g[i]).max())


@pytest.mark.parametrize("terms", ALL_MASKS)
def test_flow_conserves_the_six_integrals_identically(terms):
    """dH/dt = grad H . f, dJ/dt, d|S_i|^2/dt vanish algebraically."""
    z = random_states(16, seed=200 + terms)
    beta = np.linspace(0.25, 1.0, 16)
    kw = dict(beta=beta, chi1=0.8, chi2=0.95, kq1=3.0, kq2=1.5, terms=terms)
    f = oracle.rhs(z, **kw)
    g = oracle.gradient(z, **kw)
    s1, s2 = 0.8 * beta, 0.95 / beta
    dH = (g[0:6] * f[0:6]).sum(0) + s1 * (g[6:9] * f[6:9]).sum(0) + s2 * (g[9:12] * f[9:12]).sum(0)
    scale = (np.abs(g[0:6]) * np.abs(f[0:6])).sum(0)
    assert np.abs(dH / scale).max() < 5e-16
    dJ = np.cross(f[0:3].T, z[3:6].T).T + np.cross(z[0:3].T, f[3:6].T).T + s1 * f[6:9] + s2 * f[9:12]
    Ls = np.abs(np.cross(z[0:3].T, f[3:6].T)).sum() / 16
    assert np.abs(dJ).max() < 1e-15 * max(Ls, 1.0) * 30
    assert np.abs((z[6:9] * f[6:9]).sum(0)).max() < 1e-17
    assert np.abs((z[9:12] * f[9:12]).sum(0)).max() < 1e-17


def test_hamilton_equations_signs_on_a_newtonian_orbit():
    """terms = 0: dr/dt = p, dp/dt = -r/r^3 (Kepler), spins do not move."""
    z = random_states(5, seed=3)
    f = oracle.rhs(z, terms=0)
    r3 = np.linalg.norm(z[0:3], axis=0) ** 3
    assert np.allclose(f[0:3], z[3:6], rtol=0, atol=1e-17)
    assert np.allclose(f[3:6], -z[0:3] / r3, rtol=1e-15, atol=0)
    assert np.all(f[6:12] == 0)


# ---- spin couplings ------------------------------------------------------------------------------

@pytest.mark.parametrize("beta", [1.0 / 3.0, 1.0])
def test_spin_orbit_coefficients_are_the_papers(beta):
    """Omega_i(SO) is parallel to L with coefficient eta g_i / r^3; g_i are printed in eqs (8)-(9)."""
    z = random_states(4, seed=11)
    g = oracle.gradient(z, beta=beta, chi1=0.6, chi2=0.9, terms=oracle.TERM_SO)
    L = np.cross(z[0:3].T, z[3:6].T).T
    r3 = np.linalg.norm(z[0:3], axis=0) ** 3
    c1 = (g[6:9] * L).sum(0) / (L * L).sum(0) * r3 / eta_of(beta)
    c2 = (g[9:12] * L).sum(0) / (L * L).sum(0) * r3 / eta_of(beta)
    assert np.allclose(c1, golden("so_coeff_body1", beta), rtol=1e-14)
    assert np.allclose(c2, golden("so_coeff_body2", beta), rtol=1e-14)
    assert np.abs(np.cross(g[6:9].T, L.T)).max() < 1e-18


def test_geodetic_precession_rate_in_the_test_spin_limit():
    """beta -> 0, SO only: body 1 is a gyroscope orbiting mass M; its spin precesses about L at the
    de Sitter rate (3/2) |r x v| / r^3 (textbook).  Measured on an integrated circular orbit."""
    beta, r0 = 1e-6, 60.0
    z = np.zeros((12, 1))
    z[0], z[4] = r0, 1 / np.sqrt(r0)
    z[6], z[8] = np.sin(0.4), np.cos(0.4)      # tilted from L = z axis
    z[11] = 1.0
    n_steps, h = 4000, 0.5
    res = oracle.integrate(z, h, n_steps, mode=0, beta=beta, chi1=1e-3, chi2=0.0, terms=oracle.TERM_SO)
    s = res.states[6:9, 0]
    angle = np.arctan2(s[1], s[0])             # precession angle about z
    rate = 1.5 * (r0 * z[4, 0]) / r0 ** 3
    assert abs(angle / (rate * n_steps * h) - 1) < 2e-5
    assert abs(s[2] - np.cos(0.4)) < 1e-9      # tilt is preserved


@pytest.mark.parametrize("beta", [0.5, 1.0])
def test_quadrupole_monopole_relative_weights_are_the_papers(beta):
    """eqs (3)-(5): for equal spin vectors S1 = S2 the ratio (H_S1S1 + H_S2S2)/H_S1S2 is
    1/(2 beta) + beta/2."""
    z = random_states(3, seed=21)
    z[9:12] = z[6:9]
    chi1 = 0.4 / beta
    chi2 = 0.4 * beta           # s1 = chi1*beta = s2 = chi2/beta = 0.4
    orb = oracle.hamiltonian(z, beta=beta, chi1=chi1, chi2=chi2, terms=0)
    ss = oracle.hamiltonian(z, beta=beta, chi1=chi1, chi2=chi2, terms=oracle.TERM_S1S2) - orb
    qm = oracle.hamiltonian(z, beta=beta, chi1=chi1, chi2=chi2, terms=oracle.TERM_QM) - orb
    assert np.allclose(qm / ss, golden("qm_over_s1s2_equalS", beta), rtol=1e-12)


def test_quadrupole_spin_precession_ratio_is_the_papers():
    """Third terms of eqs (8), (9): coefficients (1+1/beta)^2 and (1+beta)^2, ratio 1/beta^2."""
    beta = 1.0 / 3.0
    z = random_states(3, seed=22)
    z[9:12] = z[6:9]
    chi1, chi2 = 0.3 / beta, 0.3 * beta          # equal spin vectors
    g = oracle.gradient(z, beta=beta, chi1=chi1, chi2=chi2, terms=oracle.TERM_QM)
    n = z[0:3] / np.linalg.norm(z[0:3], axis=0)
    w1 = (g[6:9] * n).sum(0) - 0   # component along n: (3 q/r^3)(2a) - 2 q a/r^3, same form both bodies
    w2 = (g[9:12] * n).sum(0)
    want = golden("qm_spin_coeff_body1", beta) / golden("qm_spin_coeff_body2", beta)
    assert np.allclose(w1 / w2, want, rtol=1e-12)


@pytest.mark.parametrize("beta", [0.4, 1.0])
def test_black_hole_spin_spin_sum_is_damours_S0_form(beta):
    """kq = 1: H_S1S2 + H_S1S1 + H_S2S2 = (eta^2/2) [3 (S0.n)^2 - S0.S0]/r^3 with
    S0 = (1+1/beta) S1 + (1+beta) S2  (Damour 2001, the source PAPER.md:101 cites for eqs 4-5)."""
    z = random_states(5, seed=31)
    chi1, chi2 = 0.7, 0.9
    eta = eta_of(beta)
    orb = oracle.hamiltonian(z, beta=beta, chi1=chi1, chi2=chi2, terms=0)
    ss = oracle.hamiltonian(z, beta=beta, chi1=chi1, chi2=chi2, terms=oracle.TERM_S1S2 | oracle.TERM_QM) - orb
    S0 = (1 + 1 / beta) * chi1 * beta * z[6:9] + (1 + beta) * chi2 / beta * z[9:12]
    r = np.linalg.norm(z[0:3], axis=0)
    n = z[0:3] / r
    want = 0.5 * eta ** 2 * (3 * (S0 * n).sum(0) ** 2 - (S0 * S0).sum(0)) / r ** 3
    assert np.allclose(ss, want, rtol=1e-12)
