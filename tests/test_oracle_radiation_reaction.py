"""Pins for the 2.5PN radiation-reaction term of the oracle (SURVEY 8f row 4; PAPER.md:103-107 eq 6, :219-223;
DESIGN.md R21).  PAPER.md does not print a_2.5PN, so the term is pinned by what physics fixes for ANY gauge of the
leading-order radiation reaction: the quadrupole-formula fluxes of Peters & Mathews (1963) / Peters (1964) for
circular and eccentric orbits, the adiabatic decay law of a circular orbit, and the integral invariant relation
(PAPER.md:221).  CPU only."""
import numpy as np
import pytest

import oracle
from paper_1802_00147_b200 import workloads

RR = oracle.TERM_RR


def kepler_z(a, e):
    """Newtonian orbit at apocentre on the x axis, moving along +y (mu = M = 1)."""
    z = np.zeros((12, 1))
    z[0], z[4] = a * (1 + e), np.sqrt((1 - e) / (a * (1 + e)))
    z[8], z[11] = 1, 1
    return z


@pytest.mark.parametrize("beta", [1.0, 1.0 / 3.0, 0.1])
def test_circular_orbit_radiates_the_quadrupole_power(beta):
    """dE/dt = -(32/5) eta^2 (M/r)^5 for a circular orbit (Peters & Mathews 1963); per unit mu: -(32/5) eta / r^5.
    Instantaneous, at any point of the circle and any orientation; angular momentum flux dL/dt = (dE/dt) / Omega."""
    eta = beta / (1 + beta) ** 2
    rng = np.random.default_rng(1)
    for r0 in (8.0, 30.0, 200.0):
        q, _ = np.linalg.qr(rng.normal(size=(3, 3)))          # random orientation of the orbital plane
        z = np.zeros((12, 1))
        z[0:3, 0] = r0 * q[:, 0]
        z[3:6, 0] = q[:, 1] / np.sqrt(r0)
        z[6:9, 0], z[9:12, 0] = q[:, 2], q[:, 2]
        f = oracle.evaluate("rhs16", z, beta=beta, terms=RR)[:, 0]
        power = -(32.0 / 5.0) * eta / r0 ** 5
        assert abs(f[12] / power - 1) < 1e-14                                     # dW/dt
        torque = power * r0 ** 1.5 * q[:, 2]                                      # dL/dt = P / Omega along L
        assert np.abs(f[13:16] / np.linalg.norm(torque) - torque / np.linalg.norm(torque)).max() < 1e-14
        plain = oracle.evaluate("rhs16", z, beta=beta, terms=0)[:, 0]
        assert np.all(plain[12:16] == 0) and np.array_equal(plain[0:3], f[0:3])   # the force enters dp/dt only (eq 6)
        assert np.abs((f[3:6] - plain[3:6]) @ q[:, 1] / np.sqrt(r0) / power - 1) < 1e-10   # F.v = power (difference of two rhs)


@pytest.mark.parametrize("e", [0.0, 0.3, 0.6])
def test_orbit_averaged_fluxes_of_an_eccentric_orbit_are_peters(e):
    """<dE/dt> = -(32/5) eta a^-5 (1 + 73/24 e^2 + 37/96 e^4) (1 - e^2)^-7/2 and
    <dL/dt> = -(32/5) eta a^-7/2 (1 + 7/8 e^2) (1 - e^2)^-2 (Peters 1964), per unit mu, whatever the gauge of the
    2.5PN force: one Newtonian radial period with the force on, W and G_z read off at the end.  A wrong coefficient
    in any of the six terms of the force changes these at O(1)."""
    a, beta = 60.0, 1e-4          # tiny eta: the orbit barely changes over the period, the averages are the closed forms
    eta = beta / (1 + beta) ** 2
    T = 2 * np.pi * a ** 1.5
    n_steps = 6000
    o = oracle.integrate(kepler_z(a, e), T / n_steps, n_steps, 0, beta=beta, terms=RR, r_merge=0.0)
    fE = (1 + 73 / 24 * e ** 2 + 37 / 96 * e ** 4) / (1 - e ** 2) ** 3.5
    fL = (1 + 7 / 8 * e ** 2) / (1 - e ** 2) ** 2
    dE = -(32 / 5) * eta * a ** -5 * fE * T
    dL = -(32 / 5) * eta * a ** -3.5 * fL * T
    # the orbit shrinks by ~1e-6 (times the flux contrast between peri- and apocentre) over the period
    assert abs(o.diss[0, 0] / dE - 1) < 2e-4, (o.diss[0, 0], dE)
    assert abs(o.diss[3, 0] / dL - 1) < 2e-4, (o.diss[3, 0], dL)
    assert np.abs(o.diss[1:3, 0]).max() < 1e-12 * abs(dL)                          # torque along L only


def test_circular_orbit_decays_as_peters_law():
    """Adiabatic inspiral of a circular orbit: a(t)^4 = a0^4 - (256/5) eta t (Peters 1964), Newtonian + 2.5PN."""
    beta, a0, t = 1.0, 40.0, 50_000
    eta = 0.25
    o = oracle.integrate(kepler_z(a0, 0.0), 2.0, t // 2, 0, beta=beta, terms=RR)
    r = np.linalg.norm(o.states[0:3, 0])
    want = (a0 ** 4 - 256 / 5 * eta * t) ** 0.25
    assert want < a0 - 0.7 and abs(r / want - 1) < 2e-3, (r, want)
    # and the energy lost is the energy radiated: E(t) - E0 = W(t) (integral invariant relation)
    E = oracle.integrals(o.states, beta=beta, terms=RR)[0, 0]
    assert abs((E - o.invariants[0, 0]) / o.diss[0, 0] - 1) < 1e-6


@pytest.mark.parametrize("mode", [0, 2, 3])
def test_integral_invariant_relation_with_the_full_hamiltonian(mode):
    """PAPER.md:221, orbit 3 (the paper's dissipative example): H(t) - W(t) and J(t) - G(t) are constants of the exact
    flow.  Uncorrected RK4 keeps them to truncation error; the correction (onto E0 + W, J0 + G) to round-off, while
    the energy itself really changes (the system is dissipative)."""
    w = workloads.paper_orbit(3)
    par = dict(w.params(), terms=31 - 16 | RR)
    o = oracle.integrate(w.states, 1.0, 20_000, mode, **par)
    assert o.status[0] == 0
    I0, I1, d = o.invariants[0:6, 0], oracle.integrals(o.states, **par)[:, 0], o.diss[:, 0]
    assert d[0] < 0 and abs(d[0]) > 1e-7 * abs(I0[0])                              # energy is radiated away
    resE = abs((I1[0] - d[0]) - I0[0]) / abs(I0[0])
    resJ = np.linalg.norm((I1[1:4] - d[1:4]) - I0[1:4]) / np.linalg.norm(I0[1:4])
    if mode == 0:
        assert 1e-16 < resE < 1e-8 and resJ < 1e-8
    elif mode == 2:
        assert resE < 1e-14 and abs(np.linalg.norm(I1[1:4]) / np.linalg.norm(I0[1:4] + d[1:4]) - 1) < 1e-14
    else:
        assert resE < 1e-14 and resJ < 1e-14
    off = oracle.integrate(w.states, 1.0, 2000, mode, **dict(par, terms=15))
    assert np.all(off.diss == 0)                                                    # no term, no dissipation integrals


def test_shadow_restarts_its_dissipation_integrals_with_its_references():
    """DESIGN.md R11 + R21: after a renormalisation the shadow is re-referenced (E0', J0' of its new state), so its W', G'
    restart from zero; between renormalisations it is corrected onto E0' + W', J0' + G'."""
    w = workloads.paper_orbit(3)
    par = dict(w.params(), terms=15 | RR)
    o = oracle.integrate(w.states, 1.0, 1000, 3, shadow_eps=1e-8, renorm_interval=500, want_shadow=True, **par)
    zs = o.shadow[0:12]
    Is = oracle.integrals(zs, **par)[:, 0]
    assert abs(o.shadow[12, 0] - Is[0]) < 1e-16 and np.abs(o.shadow[13:16, 0] - Is[1:4]).max() < 1e-15
    mid = oracle.integrate(w.states, 1.0, 900, 3, shadow_eps=1e-8, renorm_interval=500, want_shadow=True, **par)
    Im = oracle.integrals(mid.shadow[0:12], **par)[:, 0]
    assert abs(Im[0] - mid.shadow[12, 0]) > 1e-12                                   # 400 steps after: E' = E0' + W' != E0'
    assert 0.0 < o.fli[0] < 4.0                                                     # regular orbit
