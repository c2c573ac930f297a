"""Pins of four lines of the oracle's whole-orbit driver (oracle/pn_oracle.hpp, integrate_orbit) that the round-2
review found unpinned: a mutation of any of them passed every CPU test except the comparison with the oracle's own
stored output.  Each pin below compares the driver's pair (orbit + shadow) run with something the pair logic has no
part in: runs WITHOUT a shadow of the orbit alone and of the shadow's initial state alone, and the plain definition
FLI = log10 d(t)/d(0).

  (a) the final partial-interval term of the FLI, acc + log10(|z' - z| / d0)
  (b) merge / escape is decided by the MAIN trajectory's |r|                            (R13)
  (c) a non-finite component in the SHADOW alone also drops the orbit                    (R13)
  (d) the mode-2 "scaling skipped" flag reports the MAIN trajectory only                 (R7)
"""
import numpy as np
import pytest

import oracle
from paper_1802_00147_b200 import workloads

EPS = 1e-8


def _alone(z, n, **kw):
    return oracle.integrate(z, 1.0, n, **kw)


@pytest.mark.parametrize("which", [1, 4])
@pytest.mark.parametrize("n_steps", [150, 1250])
def test_fli_includes_the_separation_grown_since_the_last_renormalisation(which, n_steps):
    """(a) n_steps is not a multiple of renorm_interval, so the run ends 50 steps into an interval.  The definition,
    evaluated from two independent shadow-less runs started eps apart, is what the pair run must report -- with one
    renormalisation interval longer than the run (the FLI is then the final term alone) and with interval 100 (the
    accumulated part plus the final term; the tangent dynamics is linear, so the pull-backs change nothing to first
    order in eps).  Without the final term the first would be 0 and the second the FLI at the last multiple of 100,
    which differs by 0.02 ... 0.7 on these orbits."""
    w = workloads.paper_orbit(which)
    par = w.params()
    z = w.states
    zs = z.copy()
    zs[0] += EPS
    a, b = _alone(z, n_steps, mode=3, **par), _alone(zs, n_steps, mode=3, **par)
    direct = np.log10(np.linalg.norm(b.states - a.states) / EPS)
    assert 0.2 < direct < 3.0
    one_interval = oracle.integrate(z, 1.0, n_steps, mode=3, shadow_eps=EPS, renorm_interval=10 ** 6, **par).fli[0]
    every_100 = oracle.integrate(z, 1.0, n_steps, mode=3, shadow_eps=EPS, renorm_interval=100, **par).fli[0]
    assert abs(one_interval - direct) < 5e-6        # measured 4e-8 ... 2e-7 (states come back rounded to double)
    assert abs(every_100 - direct) < 5e-6           # measured 4e-8 ... 4e-7
    at_last_multiple = oracle.integrate(z, 1.0, (n_steps // 100) * 100, mode=3, shadow_eps=EPS, **par).fli[0]
    assert abs(at_last_multiple - direct) > 0.02    # the term under test is not a rounding-size quantity here


def _plunge():
    z = np.zeros((12, 1))
    z[0], z[4], z[8], z[11] = 6.0, 0.05, 1.0, 1.0
    return z


@pytest.mark.parametrize("offset", [-0.5, 0.5])
def test_merge_is_decided_by_the_main_trajectory_radius(offset):
    """(b) a wide pair (0.5 M apart, never pulled back): the shadow crosses r_merge three steps before (offset < 0) or
    after (offset > 0) the orbit does.  Status and freeze step of the pair are those of the orbit integrated alone."""
    z = _plunge()
    zs = z.copy()
    zs[0] += offset
    main, shadow = _alone(z, 3000, mode=3), _alone(zs, 3000, mode=3)
    assert main.status[0] == 1 and shadow.status[0] == 1
    assert abs(int(shadow.steps_done[0]) - int(main.steps_done[0])) >= 2
    pair = oracle.integrate(z, 1.0, 3000, mode=3, shadow_eps=offset, renorm_interval=10 ** 6)
    assert pair.status[0] == 1
    assert pair.steps_done[0] == main.steps_done[0]
    assert np.array_equal(pair.states, main.states)
    # escape: same rule.  A hyperbolic orbit whose shadow starts 30 M further out crosses r_escape later than its shadow
    y = np.zeros((12, 1))
    y[0], y[4], y[8], y[11] = 20.0, 0.5, 1.0, 1.0
    ys = y.copy()
    ys[0] += 30.0
    kw = dict(mode=3, r_escape=200.0)
    main, shadow = _alone(y, 3000, **kw), _alone(ys, 3000, **kw)
    assert main.status[0] == 2 and shadow.status[0] == 2 and shadow.steps_done[0] != main.steps_done[0]
    pair = oracle.integrate(y, 1.0, 3000, shadow_eps=30.0, renorm_interval=10 ** 6, **kw)
    assert pair.status[0] == 2 and pair.steps_done[0] == main.steps_done[0]


@pytest.mark.parametrize("mode", [0, 3])
def test_a_non_finite_shadow_alone_drops_the_orbit(mode):
    """(c) the shadow starts ON the singularity r = 0 (offset = -r0), so its first step is non-finite while the orbit
    itself is a harmless bound orbit.  The pair is dropped at once with MC_ST_NONFINITE, state frozen at the input;
    the run is shorter than the renormalisation interval, so nothing else could have noticed."""
    z = np.zeros((12, 1))
    z[0], z[4], z[8], z[11] = 20.0, 0.9 / np.sqrt(20.0), 1.0, 1.0
    main = _alone(z, 50, mode=mode)
    assert main.status[0] == 0 and main.steps_done[0] == 50
    pair = oracle.integrate(z, 1.0, 50, mode=mode, shadow_eps=-20.0)
    assert pair.status[0] == 3 and pair.steps_done[0] == 0
    assert np.array_equal(pair.states, z)


def test_mode2_flag_reports_the_main_trajectory_only():
    """(d) a wide pair in mode 2: the orbit is near-circular at r = 40, where the dual scaling never has a reason to be
    skipped; its shadow starts 35 M further in with the same momentum, dives to r = 2.4 within 60 steps and there RK4
    with h = 1 is so far off the energy surface that |v - 1| > 1e-3: its scaling IS skipped (shown by integrating the
    shadow's initial state alone: flag set, and that run is bit for bit the pair's shadow).  The pair reports no flag."""
    par = dict(beta=1.0, chi1=0.9, chi2=0.8, terms=15)
    kw = dict(mode=2, newton_iters=4, r_merge=0.0, r_escape=1e9, **par)
    z = np.zeros((12, 1))
    z[0], z[4], z[8], z[11] = 40.0, 0.95 / np.sqrt(40.0), 1.0, 1.0
    zs = z.copy()
    zs[0] += -35.0
    main, shadow = _alone(z, 60, **kw), _alone(zs, 60, **kw)
    assert main.status[0] == 0
    assert shadow.status[0] == 256 and shadow.steps_done[0] == 60
    pair = oracle.integrate(z, 1.0, 60, shadow_eps=-35.0, renorm_interval=10 ** 6, want_shadow=True, **kw)
    assert np.array_equal(pair.shadow[:12], shadow.states)      # the pair's shadow did skip
    assert pair.status[0] == 0 and pair.steps_done[0] == 60
    assert np.array_equal(pair.states, main.states)
    # and the flag is raised when the MAIN trajectory is the one that skips
    swapped = oracle.integrate(zs, 1.0, 60, shadow_eps=35.0, renorm_interval=10 ** 6, **kw)
    assert swapped.status[0] == 256
