"""GPU parity: libmc (through the C ABI, paper_1802_00147_b200.binding) vs the CPU oracle, element by
element on the same seeded inputs.  Tolerances (DESIGN.md section 7 / BASELINE.json north_star):
state relative error <= 1e-10 after 1e3 steps; six integrals' relative drift <= 1e-12 with correction
on; FLI class agreement; integer outputs (status, steps) exact."""
import numpy as np
import pytest

import oracle
from conftest import random_states
from paper_1802_00147_b200 import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

STATE_RTOL = 1e-10      # north_star
DRIFT_TOL = 1e-12       # north_star
FLI_THRESHOLD = 5.8
# FLI value after 1e3-2e3 steps (north_star states no tolerance for the value, only for the class):
# about three times the deviation of the oracle's own double instance from its long-double instance on the same inputs
# (0.8e-3 .. 1.3e-3, pinned on CPU by test_fli_rounding_envelope_sets_the_parity_bound)
FLI_VALUE_TOL = 3e-3


@pytest.fixture(scope="module")
def mc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1802_00147_b200 import binding
    return binding


def rel_state_err(a, b):
    """max over orbits of per-block relative error (r, p, S1, S2 blocks)."""
    worst = 0.0
    for s in (slice(0, 3), slice(3, 6), slice(6, 9), slice(9, 12)):
        num = np.linalg.norm(a[s] - b[s], axis=0)
        den = np.linalg.norm(b[s], axis=0)
        worst = max(worst, float((num / den).max()))
    return worst


def drift(states, inv0, **params):
    """Relative drift of the six integrals, evaluated by the ORACLE (long double) on given states."""
    I1 = oracle.integrals(states, **params)
    dE = np.abs(I1[0] - inv0[0]) / np.abs(inv0[0])
    dJ = np.linalg.norm(I1[1:4] - inv0[1:4], axis=0) / np.linalg.norm(inv0[1:4], axis=0)
    return max(dE.max(), dJ.max(), np.abs(I1[4] - 1).max(), np.abs(I1[5] - 1).max())


PARAM_SETS = [
    dict(beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0),
    dict(beta=0.8, chi1=0.9, chi2=0.9, kq1=3.0, kq2=5.5),
    dict(beta=1.0 / 3.0, chi1=0.75, chi2=0.75, kq1=1.0, kq2=1.0),
]


@pytest.mark.parametrize("terms", [0, 1, 3, 4, 8, 15, 16, 31])
@pytest.mark.parametrize("pset", [0, 1, 2])
def test_model_routines_match_oracle_uniform(mc, terms, pset):
    """H, dz/dt, six integrals, one RK4 step: 300 random states (3 blocks, ragged tail)."""
    z = random_states(300, seed=1000 + terms)
    par = PARAM_SETS[pset]
    with mc.Integrator(terms=terms, **par) as I:
        for what, ofn, scale_rows in (("H", lambda: oracle.hamiltonian(z, terms=terms, **par)[None], None),
                                      ("rhs", lambda: oracle.rhs(z, terms=terms, **par), 3),
                                      ("integrals", lambda: oracle.integrals(z, terms=terms, **par), None),
                                      ("rk4_step", lambda: oracle.rk4_step(z, 1.0, terms=terms, **par), 3)):
            got = I.eval(what, z, h=1.0).cpu().numpy()
            want = ofn()
            if scale_rows:
                assert rel_state_err_blocks(got, want) < 2e-13, what
            else:
                assert np.abs(got - want).max() <= 4e-14 * max(1.0, np.abs(want).max()), what


def rel_state_err_blocks(a, b):
    worst = 0.0
    for s in (slice(0, 3), slice(3, 6), slice(6, 9), slice(9, 12)):
        den = np.linalg.norm(b[s], axis=0)
        num = np.linalg.norm(a[s] - b[s], axis=0)
        ok = den > 0
        if ok.any():
            worst = max(worst, float((num[ok] / den[ok]).max()))
        assert np.all(num[~ok] == 0)
    return worst


def test_model_routines_match_oracle_per_orbit(mc):
    z = random_states(257, seed=77)
    rng = np.random.default_rng(78)
    par = dict(beta=rng.uniform(0.3, 1, 257), chi1=rng.uniform(0, 1, 257), chi2=rng.uniform(0, 1, 257),
               kq1=rng.uniform(1, 8, 257), kq2=rng.uniform(1, 8, 257))
    for terms in (15, 31):
        with mc.Integrator(terms=terms, **par) as I:
            assert rel_state_err_blocks(I.eval("rhs", z).cpu().numpy(), oracle.rhs(z, terms=terms, **par)) < 2e-13
            H = I.eval("H", z).cpu().numpy()[0]
            assert np.abs(H - oracle.hamiltonian(z, terms=terms, **par)).max() < 1e-15


@pytest.mark.parametrize("mode", [1, 2, 3])
@pytest.mark.parametrize("terms", [15, 31])
def test_correction_operator_matches_oracle(mc, mode, terms):
    w = workloads.config0(200)
    par = dict(beta=0.7, chi1=0.9, chi2=0.8, kq1=2.0, kq2=3.0)
    I0 = oracle.integrals(w.states, terms=terms, **par)
    rng = np.random.default_rng(3)
    zp = w.states * (1 + 1e-7 * rng.normal(size=w.states.shape))
    want, ok = oracle.correct(zp, I0[0], I0[1:4], mode, terms=terms, newton_iters=4, **par)
    with mc.Integrator(terms=terms, newton_iters=4, **par) as I:
        got = I.eval("correct", zp, mode=mode, refs=I0[0:4]).cpu().numpy()
    assert ok.all()
    assert rel_state_err(got, want) < 1e-13
    assert drift(got, I0, terms=terms, **par) < (1e-14 if mode == 3 else 1.0)


def test_plain_c_program_drives_the_library(mc, tmp_path):
    """The boundary is a C ABI: tests/c_abi_caller.c (C99, no Python, no torch, no CUDA headers) is compiled with gcc
    against include/mc.h, linked with libmc.so and run; it integrates 40 shadowed orbits through mc_integrate_host and
    checks return codes, status, drift of the integrals <= 1e-12, FLI range, zero spills and run-to-run bit identity."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    mc.load_library()                                     # builds libmc.so if it is stale
    pkg = os.path.join(root, "paper_1802_00147_b200")
    exe = str(tmp_path / "c_abi_caller")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-O1", "-I", os.path.join(root, "include"),
                    os.path.join(root, "tests", "c_abi_caller.c"), "-o", exe, "-L", pkg, "-l:libmc.so",
                    "-Wl,-rpath," + pkg, "-lm"], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "c_abi_caller ok" in r.stdout


def test_mode3_operator_near_the_circular_singularity(mc):
    """The degenerate case of mode 3: for a circular orbit the energy row of the constraint
    Jacobian is a combination of the angular-momentum rows and the projection is singular; for a nearly circular one it
    is ill conditioned like 1/e^2.  Newtonian Hamiltonian (terms = 0), BASELINE config 0's initial conditions, which
    reach p_y = 0.99993 of the circular value.  Bars: the bulk agrees with the long-double oracle to round-off; the
    worst orbit of ONE Gauss-Newton step to 1e-8 -- and the kernel's closed form in the frame {r, p, L} stays closer to
    the long-double result than the oracle's own double instance (pivoted elimination in FP64: 2.5e-7 on the same
    input), which is what an ill-conditioned solve costs in double precision.  (Measured: 6.5e-11 / 7e-12 for one
    step, 1.6e-8 / 1.6e-9 for the epsilon-terminated iteration, beta = 0.8 / 0.1.)"""
    w = workloads.config0(257)
    r0 = np.linalg.norm(w.states[0:3], axis=0)
    assert (np.linalg.norm(w.states[3:6], axis=0) * np.sqrt(r0)).max() > 0.9999      # the input does contain the near-circular orbit
    rng = np.random.default_rng(5)
    zp = w.states * (1 + 1e-6 * rng.normal(size=w.states.shape))
    for beta in (0.8, 0.1):
        par = dict(beta=beta, chi1=1.0, chi2=0.0)
        I0 = oracle.integrals(w.states, terms=0, **par)
        for iters, cap in ((1, 1e-8), (4, 1e-6)):
            want, _ = oracle.correct(zp, I0[0], I0[1:4], 3, terms=0, newton_iters=iters, **par)
            want_double, _ = oracle.correct(zp, I0[0], I0[1:4], 3, terms=0, newton_iters=iters, precision=oracle.DOUBLE, **par)
            with mc.Integrator(terms=0, newton_iters=iters, **par) as I:
                got = I.eval("correct", zp, mode=3, refs=I0[0:4]).cpu().numpy()

            def per_orbit(a):
                return np.max([np.linalg.norm(a[s] - want[s], axis=0) / np.linalg.norm(want[s], axis=0)
                               for s in (slice(0, 3), slice(3, 6))], axis=0)
            e_gpu, e_double = per_orbit(got), per_orbit(want_double)
            assert np.median(e_gpu) < 1e-14
            assert e_gpu.max() < cap
            assert e_double.max() > 1e-8 and e_gpu.max() < e_double.max()


def test_config0_state_parity_after_1e3_steps_and_drift_after_1e4(mc):
    """BASELINE config 0: 64 orbits, mode 3, no shadow."""
    w = workloads.config0()
    with mc.Integrator(terms=w.terms, beta=1.0, chi1=1.0, chi2=1.0) as I:
        g3 = I.integrate(w.states, w.h, 1000, 3)
        g4 = I.integrate(w.states, w.h, 10_000, 3)
        info = I.launch_info()
    o3 = oracle.integrate(w.states, w.h, 1000, 3, **w.params())
    assert rel_state_err(g3.states.cpu().numpy(), o3.states) <= STATE_RTOL
    assert np.array_equal(g3.status.cpu().numpy(), o3.status)
    assert np.array_equal(g3.steps_done.cpu().numpy(), o3.steps_done)
    inv = g4.invariants.cpu().numpy()
    assert np.abs(inv[0:6] - o3.invariants[0:6]).max() < 1e-14          # reference integrals agree
    assert drift(g4.states.cpu().numpy(), o3.invariants[0:6], **w.params()) <= DRIFT_TOL
    assert (g4.status.cpu().numpy() == 0).all()
    assert info["local_bytes"] == 0                                      # zero register spills


@pytest.mark.parametrize("mode", [3, 0])
def test_config1_shadow_fli_parity_per_orbit_params(mc, mode):
    """BASELINE config 1 (per-orbit beta, chi; shadow 1e-8, renorm 100), first 150 orbits = 300
    trajectories: two full blocks + ragged tail; 2000 steps = 20 renormalisations."""
    w = workloads.config1().subset(np.arange(150))
    with mc.Integrator(terms=w.terms, **{k: v for k, v in w.params().items() if k != "terms"}) as I:
        g = I.integrate(w.states, w.h, 2000, mode, shadow_eps=w.shadow_eps)
        work = I.work(w.n_orbits).cpu().numpy()
    o = oracle.integrate(w.states, w.h, 2000, mode, shadow_eps=w.shadow_eps, **w.params())
    assert rel_state_err(g.states.cpu().numpy(), o.states) <= 4 * STATE_RTOL   # 2e3 steps
    assert np.abs(g.fli.cpu().numpy() - o.fli).max() < FLI_VALUE_TOL
    assert np.array_equal(g.status.cpu().numpy(), o.status)
    assert np.array_equal(g.steps_done.cpu().numpy(), o.steps_done)
    if mode == 3:
        assert drift(g.states.cpu().numpy(), o.invariants[0:6], **w.params()) <= DRIFT_TOL
        # Gauss-Newton step counts (epsilon-terminated, R6): the termination test is taken in FP64 here and in
        # long double in the oracle, so single decisions at the threshold may differ
        assert np.abs(work - o.gn_steps).max() <= 0.01 * o.gn_steps.max()
        assert (work >= 2 * 2000).all() and (work < 2 * 2 * 2000).all()
    else:
        assert (work == 0).all()


def classes(fli, status):
    """0 regular, 1 chaotic, 2 dropped."""
    c = (fli >= FLI_THRESHOLD).astype(int)
    c[(status & 255) != 0] = 2
    return c


def test_scan_grid_with_dropped_orbits_matches_oracle(mc):
    """Config-2-shaped grid (strong-field corner r0 in [6,16] so that merged orbits occur), 12 x 11
    cells = 132 orbits, 3000 steps: status, freeze step, FLI and class per cell."""
    z, R, TH = workloads.scan_grid(12, 11, r_lo=6.0, r_hi=16.0)
    with mc.Integrator() as I:
        g = I.integrate(z, 1.0, 3000, 3, shadow_eps=1e-8)
    o = oracle.integrate(z, 1.0, 3000, 3, shadow_eps=1e-8)
    gs, gk = g.status.cpu().numpy(), g.steps_done.cpu().numpy()
    assert (o.status == 1).sum() >= 5 and (o.status == 0).sum() >= 50     # the case has both kinds
    assert np.array_equal(gs, o.status)
    assert np.array_equal(gk, o.steps_done)
    alive = o.status == 0
    gfli = g.fli.cpu().numpy()
    assert (classes(gfli, gs) == classes(o.fli, o.status)).mean() >= 0.99
    calm = alive & (o.fli < 3.5)                       # regular cells: values agree, not only classes
    assert calm.sum() > 20
    assert np.abs(gfli[calm] - o.fli[calm]).max() < 1e-2
    assert rel_state_err(g.states.cpu().numpy()[:, calm], o.states[:, calm]) < 1e-7
    # frozen cells keep the last good state: |r| >= r_merge
    assert (np.linalg.norm(g.states.cpu().numpy()[0:3], axis=0) >= 2.0).all()


def test_config3_quadrupole_on_off_parity(mc):
    """BASELINE config 3 subset: beta = 0.8, chi = 0.9, per-orbit kq; QM on vs off on identical inputs."""
    full = workloads.config3(n_r=16, n_theta=9, qm=True)
    par = {k: v for k, v in full.params().items() if k != "terms"}
    out = {}
    for qm in (True, False):
        terms = full.terms if qm else (full.terms & ~workloads.TERM_QM)
        with mc.Integrator(terms=terms, **par) as I:
            g = I.integrate(full.states, 1.0, 1000, 3, shadow_eps=1e-8)
        o = oracle.integrate(full.states, 1.0, 1000, 3, shadow_eps=1e-8, terms=terms, **par)
        ok = o.status == 0
        assert np.array_equal(g.status.cpu().numpy(), o.status)
        assert rel_state_err(g.states.cpu().numpy()[:, ok], o.states[:, ok]) <= STATE_RTOL
        assert np.abs(g.fli.cpu().numpy()[ok] - o.fli[ok]).max() < FLI_VALUE_TOL
        out[qm] = g.states.cpu().numpy()
    assert np.abs(out[True] - out[False]).max() > 1e-3          # the term really changes the dynamics


def test_per_orbit_kappa_variant_matches_oracle_and_the_full_per_orbit_kernel(mc):
    """mc_params.per_orbit = 2 (BASELINE config 3: one binary model, per-orbit quadrupole coefficients): the four
    kappa-dependent constants ride in registers, everything else in the constant bank.  Model routines on random
    states, then a shadowed run; the fully per-orbit kernel (per_orbit = 1) on the same inputs must agree with the
    oracle to the same bar, and without the QM bit the library runs the uniform kernel (kappa is unused)."""
    z = random_states(300, seed=21)
    rng = np.random.default_rng(22)
    par = dict(beta=0.8, chi1=0.9, chi2=0.7, kq1=rng.uniform(1, 8, 300), kq2=rng.uniform(1, 8, 300))
    with mc.Integrator(terms=31, **par) as I:
        assert I.params.per_orbit == 2
        assert rel_state_err_blocks(I.eval("rhs", z).cpu().numpy(), oracle.rhs(z, terms=31, **par)) < 2e-13
        assert np.abs(I.eval("H", z).cpu().numpy()[0] - oracle.hamiltonian(z, terms=31, **par)).max() < 1e-15
        assert rel_state_err_blocks(I.eval("rk4_step", z, h=1.0).cpu().numpy(), oracle.rk4_step(z, 1.0, terms=31, **par)) < 2e-13
    w = workloads.config3(n_r=12, n_theta=13, qm=True)
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    o = oracle.integrate(w.states, 1.0, 1000, 3, shadow_eps=1e-8, **w.params())
    ok = o.status == 0
    got = {}
    for force in (None, 1):
        with mc.Integrator(terms=w.terms, per_orbit=force, **kw) as I:
            g = I.integrate(w.states, 1.0, 1000, 3, shadow_eps=1e-8)
            info = I.launch_info()
        assert info["local_bytes"] == 0
        assert (info["variant"] & 7) == (6 if force is None else 3)           # QM + (kappa-only | per-orbit)
        assert info["blocks_per_sm"] == (3 if force is None else 2)
        assert np.array_equal(g.status.cpu().numpy(), o.status)
        assert rel_state_err(g.states.cpu().numpy()[:, ok], o.states[:, ok]) <= STATE_RTOL
        assert np.abs(g.fli.cpu().numpy()[ok] - o.fli[ok]).max() < FLI_VALUE_TOL
        assert drift(g.states.cpu().numpy()[:, ok], o.invariants[0:6][:, ok], **w.subset(np.where(ok)[0]).params()) <= DRIFT_TOL
        got[force] = g.states.cpu().numpy()
    assert rel_state_err(got[None][:, ok], got[1][:, ok]) <= STATE_RTOL
    off = workloads.config3(n_r=12, n_theta=13, qm=False)
    with mc.Integrator(terms=off.terms, **kw) as I:
        g = I.integrate(off.states, 1.0, 300, 3, shadow_eps=1e-8)
        assert (I.launch_info()["variant"] & 7) == 0                           # uniform kernel: kappa does not enter
    oo = oracle.integrate(off.states, 1.0, 300, 3, shadow_eps=1e-8, **off.params())
    live = oo.status == 0
    assert rel_state_err(g.states.cpu().numpy()[:, live], oo.states[:, live]) <= STATE_RTOL


def test_mode2_dual_scaling_parity_on_unskipped_orbits(mc):
    w = workloads.config0(128)
    with mc.Integrator(newton_iters=4) as I:
        g = I.integrate(w.states, 1.0, 1000, 2)
    o = oracle.integrate(w.states, 1.0, 1000, 2, newton_iters=4, **w.params())
    gs = g.status.cpu().numpy()
    clean = (o.status == 0) & (gs == 0)
    assert clean.sum() >= 32                                       # singular steps are common (R7)
    assert ((gs & 256) == (o.status & 256)).mean() > 0.9
    # The dual-scaling Jacobian is singular where p.dH/dp = r.dH/dr, twice per radial period (R7): steps
    # near those points amplify rounding differences, so the bound is looser than for mode 3.
    gz = g.states.cpu().numpy()
    per_orbit = np.array([rel_state_err(gz[:, [i]], o.states[:, [i]]) for i in np.where(clean)[0]])
    print("mode-2 per-orbit relative error: median %.2e  p90 %.2e  max %.2e" %
          (np.median(per_orbit), np.quantile(per_orbit, 0.9), per_orbit.max()))
    # Bound from the arithmetic ("mode 2"): the oracle's own double instance differs
    # from its long-double instance by median 1.5e-12 / p90 6.7e-12 / max 4.0e-10 on this very input
    # (tests/test_oracle_integrator.py::test_mode2_rounding_amplification_sets_the_parity_bound), i.e.
    # ~10x the mode-3 figure.  The kernel must sit within the same envelope.
    # Round 2: bounds at ~3x what the kernel measures on this input (gpurun_out/r2_pytest1.log: median 1.1e-12, p90 8.6e-12,
    # max 7.1e-10 -- one orbit; the oracle's own double instance reaches 4.0e-10 on it), down from 1e-11 / 1e-10 / 1e-8.
    assert np.median(per_orbit) <= 5e-12 and np.quantile(per_orbit, 0.9) <= 3e-11 and per_orbit.max() <= 2e-9
    I1 = oracle.integrals(g.states.cpu().numpy()[:, clean], **w.subset(np.where(clean)[0]).params())
    I0 = o.invariants[0:6, clean]
    assert np.abs(I1[0] / I0[0] - 1).max() < DRIFT_TOL
    assert np.abs(np.linalg.norm(I1[1:4], axis=0) / np.linalg.norm(I0[1:4], axis=0) - 1).max() < DRIFT_TOL


@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_non_unit_input_spins(mc, mode):
    """include/mc.h: "with correction_mode >= 1 the input spins are normalised first" (eq 10);
    mode 0 leaves them alone.  Input |S_hat| = 1 +- 1e-3, per-orbit parameters, shadow on, 150 orbits (ragged
    tail).  The oracle side of this convention is pinned in tests/test_oracle_conventions.py."""
    w = workloads.config1().subset(np.arange(150))
    bent = w.states.copy()
    bent[6:9] *= 1.0 + 1e-3
    bent[9:12] *= 1.0 - 1e-3
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    with mc.Integrator(terms=w.terms, **kw) as I:
        g = I.integrate(bent, 1.0, 500, mode, shadow_eps=1e-8)
    o = oracle.integrate(bent, 1.0, 500, mode, shadow_eps=1e-8, **w.params())
    gz, ginv, gs = g.states.cpu().numpy(), g.invariants.cpu().numpy(), g.status.cpu().numpy()
    assert np.abs(ginv[0:6] - o.invariants[0:6]).max() < 1e-14           # reference integrals of the same state
    if mode == 0:
        assert np.abs(ginv[4] - (1 + 1e-3)).max() < 1e-15 and np.abs(ginv[5] - (1 - 1e-3)).max() < 1e-15
        assert np.abs(np.linalg.norm(gz[6:9], axis=0) - (1 + 1e-3)).max() < 1e-8    # RK4 keeps the length it was given
    else:
        assert np.abs(ginv[4:6] - 1).max() < 3e-16
        assert np.abs(np.linalg.norm(gz[6:9], axis=0) - 1).max() < 3e-16
    clean = (o.status == 0) & (gs == 0)                                   # mode 2: orbits with no skipped step (R7)
    assert clean.sum() >= (30 if mode == 2 else 150)
    if mode != 2:
        assert np.array_equal(gs, o.status)
    err = rel_state_err(gz[:, clean], o.states[:, clean])
    assert err <= (5e-10 if mode == 2 else STATE_RTOL), err
    assert np.abs(g.fli.cpu().numpy()[clean] - o.fli[clean]).max() < (1e-2 if mode == 2 else FLI_VALUE_TOL)


def test_batch_properties(mc):
    w = workloads.config0(96)
    with mc.Integrator() as I:
        a = I.integrate(w.states, 1.0, 500, 3, shadow_eps=1e-8)
        perm = np.random.default_rng(0).permutation(96)
        b = I.integrate(w.states[:, perm], 1.0, 500, 3, shadow_eps=1e-8)
        same = I.integrate(np.repeat(w.states[:, :1], 70, axis=1), 1.0, 500, 3, shadow_eps=1e-8)
        A, B = a.states.cpu().numpy(), b.states.cpu().numpy()
        assert np.array_equal(A[:, perm], B)                                  # orbits are independent
        assert np.array_equal(a.fli.cpu().numpy()[perm], b.fli.cpu().numpy())
        S = same.states.cpu().numpy()
        assert np.array_equal(S, np.repeat(S[:, :1], 70, axis=1))             # lanes are equivalent
        assert np.array_equal(S[:, 0], A[:, 0])
        # in-place operation (out_states aliases states)
        zt = torch.as_tensor(w.states, device="cuda").clone()
        c = I.integrate(zt, 1.0, 500, 3, shadow_eps=1e-8, out_states=zt)
        assert np.array_equal(c.states.cpu().numpy(), A)
        # host-buffer entry point gives the same bits
        hres = I.integrate_host(w.states, 1.0, 500, 3, shadow_eps=1e-8)
        assert np.array_equal(hres.states, A) and np.array_equal(hres.fli, a.fli.cpu().numpy())
        assert np.array_equal(hres.status, a.status.cpu().numpy())
    with mc.Integrator(terms=31, kq1=0.0, kq2=0.0) as Iq:                      # QM with zero coefficient
        q = Iq.integrate(w.states, 1.0, 500, 3, shadow_eps=1e-8)
    assert np.array_equal(q.states.cpu().numpy(), A)


def test_edge_cases(mc):
    w = workloads.config0(129)
    with mc.Integrator() as I:
        e = I.integrate(w.states[:, :0], 1.0, 10, 3)
        assert e.states.shape == (12, 0)
        one = I.integrate(w.states[:, :1], 1.0, 100, 3, shadow_eps=1e-8)
        o = oracle.integrate(w.states[:, :1], 1.0, 100, 3, shadow_eps=1e-8)
        assert rel_state_err(one.states.cpu().numpy(), o.states) < 1e-11
        zero = I.integrate(w.states, 1.0, 0, 3, shadow_eps=1e-8)                # n_steps = 0
        assert np.allclose(zero.states.cpu().numpy(), w.states, rtol=1e-15, atol=0)
        assert np.allclose(zero.fli.cpu().numpy(), 0.0, atol=1e-6)
        assert (zero.steps_done.cpu().numpy() == 0).all()
        back = I.integrate(I.integrate(w.states, 1.0, 300, 3).states, -1.0, 300, 3)   # negative step
        assert rel_state_err(back.states.cpu().numpy(), w.states) < 1e-6
        bad = w.states[:, :40].copy()
        bad[1, 7] = np.nan
        bad[0, 9] = 1.0                                                           # starts inside r_merge... plunges
        r = I.integrate(bad, 1.0, 50, 3, shadow_eps=1e-8)
        st = r.status.cpu().numpy()
        assert st[7] == 3 and r.steps_done.cpu().numpy()[7] == 0
        assert st[9] in (1, 3)
        good = np.ones(40, bool)
        good[[7, 9]] = False
        assert (st[good] == 0).all()                                              # neighbours are unaffected
    with pytest.raises(mc.MCError):
        with mc.Integrator() as I:
            I.integrate(w.states, 1.0, 10, 7)


def test_full_size_scan_sampled_against_oracle(mc):
    """BASELINE config 2 at full size (314 x 314 orbits, shadow, mode 3) in the launch configuration
    bench.py times, 1e4 steps here; 48 sampled cells are recomputed one by one by the oracle, and the
    six-integral drift is checked on every live cell."""
    w = workloads.config2(n_steps=10_000)
    with mc.Integrator() as I:
        g = I.integrate(w.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps)
        info = I.launch_info()
    assert info["local_bytes"] == 0 and info["trajectories"] == 2 * 314 * 314
    gs = g.status.cpu().numpy()
    gz = g.states.cpu().numpy()
    gfli = g.fli.cpu().numpy()
    live = gs == 0
    assert 0.85 < live.mean() < 1.0
    inv0 = g.invariants.cpu().numpy()[0:6]
    # Every live cell, including those that end the run at a deep periastron (|r| < 3): with the Newton cap
    # of 4 (R6) the residual that 2 iterations leave there (7e-11, pinned in tests/test_oracle_integrator.py::
    # test_two_newton_iterations_leave_a_residual_at_deep_periastron) is removed.
    assert (np.linalg.norm(gz[0:3], axis=0)[live] < 3.0).sum() > 20           # the case has such cells
    assert drift(gz[:, live], inv0[:, live], **w.subset(np.where(live)[0]).params()) <= DRIFT_TOL
    rng = np.random.default_rng(2)
    idx = np.sort(np.concatenate([rng.choice(314 * 314, 40, replace=False), rng.choice(314 * 40, 8, replace=False)]))
    sub = w.subset(idx)
    o = oracle.integrate(sub.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps, **sub.params())
    assert np.array_equal(gs[idx], o.status)
    assert np.array_equal(g.steps_done.cpu().numpy()[idx], o.steps_done)
    assert (classes(gfli[idx], gs[idx]) == classes(o.fli, o.status)).mean() >= 0.97
    reg = (o.status == 0) & (o.fli < 4.0)
    assert np.abs(gfli[idx][reg] - o.fli[reg]).max() < 0.02
    assert rel_state_err(gz[:, idx][:, reg], o.states[:, reg]) < 1e-6     # 1e4 steps; regular cells only


def test_classification_agreement_at_1e5_steps_on_a_strided_subgrid(mc):
    """north_star: "FLI regular/chaotic classification agreeing on >= 99 % of grid cells".  BASELINE config 2
    at full size and full length (314 x 314 orbits, 1e5 steps, the launch bench.py times); every 8th row and
    column (40 x 40 = 1600 cells, all r0 and theta ranges) is recomputed by the long-double oracle.  Classes:
    regular (FLI < 5.8), chaotic, dropped.  Chaotic cells are not reproducible value by value
    (R19), so only the class is compared there; on clearly regular cells the FLI values must agree too."""
    w = workloads.config2()
    assert w.n_steps == 100_000
    with mc.Integrator() as I:
        g = I.integrate(w.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps)
    gs, gfli = g.status.cpu().numpy(), g.fli.cpu().numpy()
    rows = np.arange(0, 314, 8)
    idx = (rows[:, None] * 314 + rows[None, :]).ravel()
    sub = w.subset(idx)
    o = oracle.integrate(sub.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps, **sub.params())
    cg, co = classes(gfli[idx], gs[idx]), classes(o.fli, o.status)
    agree = (cg == co).mean()
    near = np.abs(o.fli - FLI_THRESHOLD) < 0.5
    print("classes (oracle): regular %d chaotic %d dropped %d; agreement %.4f; oracle cells within 0.5 of 5.8: %d; "
          "disagreeing cells: %s" % ((co == 0).sum(), (co == 1).sum(), (co == 2).sum(), agree, near.sum(),
                                     [(int(i // 314), int(i % 314)) for i in idx[cg != co]]))
    assert (co == 1).sum() >= 50 and (co == 2).sum() >= 10 and (co == 0).sum() >= 1000   # all three classes occur
    assert agree >= 0.99
    assert ((cg == 2) == (co == 2)).mean() >= 0.995                                       # dropped cells
    # FLI values on cells regular on both sides: at t = 1e5 the state divergence between FP64 and long double has
    # grown to ~1e-8..1e-6 on regular orbits, i.e. ~0.01 in FLI; a few weakly chaotic ("sticky") cells still below
    # the threshold differ more (the full-grid run shows up to 1.6, profiles/r02_full_grid_classification.md), so
    # the bound is on the bulk, with a loose cap on the worst cell.
    reg = (co == 0) & (o.fli < 4.5) & (cg == 0)
    dfli = np.abs(gfli[idx][reg] - o.fli[reg])
    assert np.median(dfli) < 0.02 and np.quantile(dfli, 0.99) < 0.1 and dfli.max() < 2.0


@pytest.mark.parametrize("which", ["theta2", "theta2-0", "plane"])
def test_papers_own_scans_match_oracle(mc, which):
    """the paper's scans (Figs 6-7) -- beta = 1/3 at r = 5.65 (strong field) and
    the (theta1, theta2) plane at r = 10.14.  All 314 orbits of the 1-D scans / a 13 x 13 sub-plane, 2000 steps."""
    if which == "plane":
        w = workloads.paper_scan_plane(13, 13, dtheta=0.26)
        par = dict(beta=1.0)
    else:
        w = workloads.paper_scan_theta2(theta1=0.0 if which == "theta2-0" else np.pi / 2)
        par = dict(beta=1.0 / 3.0)
    with mc.Integrator(**par) as I:
        g = I.integrate(w.states, 1.0, 2000, 3, shadow_eps=1e-8)
    o = oracle.integrate(w.states, 1.0, 2000, 3, shadow_eps=1e-8, **w.params())
    gs, gz, gfli = g.status.cpu().numpy(), g.states.cpu().numpy(), g.fli.cpu().numpy()
    assert np.array_equal(gs, o.status)
    assert np.array_equal(g.steps_done.cpu().numpy(), o.steps_done)
    live = o.status == 0
    assert live.sum() >= 0.5 * w.n_orbits
    assert drift(gz[:, live], o.invariants[0:6][:, live], **w.subset(np.where(live)[0]).params()) <= DRIFT_TOL
    calm = live & (o.fli < 3.0)                        # short-time regular cells: values agree
    assert calm.sum() >= 0.3 * w.n_orbits
    assert np.abs(gfli[calm] - o.fli[calm]).max() < 1e-2
    assert rel_state_err(gz[:, calm], o.states[:, calm]) < 1e-7


def _all_outputs(I, z, n_steps, mode, eps):
    g = I.integrate(z, 1.0, n_steps, mode, shadow_eps=eps)
    n = z.shape[1]
    outs = [g.states, g.invariants, g.status, g.steps_done, I.work(n)] + ([g.fli] if g.fli is not None else [])
    return [t.cpu().numpy() for t in outs], I.launch_info()


@pytest.mark.parametrize("case", ["uniform-shadow", "per-orbit-shadow", "kappa-shadow", "dropped-cells", "mode2-no-shadow"])
def test_chunked_scheduling_never_changes_a_bit(mc, case):
    """the kernel's work items are chunks of steps whose state rests in a carry buffer
    between chunks.  Any chunk length -- a divisor of the run, one that cuts renormalisation intervals, a single
    step, more chunks than steps -- must reproduce the one-chunk result bit for bit in every output."""
    mode, eps, kw = 3, 1e-8, {}
    if case == "uniform-shadow":
        z = workloads.config0(300).states
    elif case in ("per-orbit-shadow", "kappa-shadow"):
        w = workloads.config3(n_r=9, n_theta=23, qm=True)
        z, kw = w.states, dict(terms=w.terms, per_orbit=(1 if case == "per-orbit-shadow" else None),
                               **{k: v for k, v in w.params().items() if k != "terms"})
    elif case == "dropped-cells":
        z = workloads.scan_grid(12, 11, r_lo=6.0, r_hi=16.0)[0]
    else:
        z, mode, eps = workloads.config0(70).states, 2, 0.0
    n_steps = 730
    with mc.Integrator(chunk_steps=n_steps, **kw) as I:
        ref, info = _all_outputs(I, z, n_steps, mode, eps)
        assert info["n_chunks"] == 1
    if case == "dropped-cells":
        assert (ref[2] != 0).sum() >= 5
    for chunk in (365, 100, 70, 1, 10_000):
        with mc.Integrator(chunk_steps=chunk, **kw) as I:
            got, info = _all_outputs(I, z, n_steps, mode, eps)
        assert info["n_chunks"] == -(-n_steps // chunk) and info["chunk_steps"] == chunk
        for a, b in zip(ref, got):
            assert np.array_equal(a, b, equal_nan=True), (case, chunk)


def test_rk5_base_integrator_matches_oracle(mc):
    """SURVEY 8(f) row 2 / DESIGN.md R9: Butcher's six-stage RK5 as the base integrator (the paper's "RK5").
    One uncorrected step on random states, then config 0 (1e3 steps, mode 3) and a shadowed per-orbit case."""
    z = random_states(300, seed=5)
    par = PARAM_SETS[1]
    for terms in (15, 31):
        with mc.Integrator(terms=terms, integrator=mc.MC_INTEG_RK5, **par) as I:
            got = I.eval("rk4_step", z, h=1.0).cpu().numpy()                  # what = 3: one base-integrator step
        want = oracle.rk_step(z, 1.0, oracle.RK5, terms=terms, **par)
        assert rel_state_err_blocks(got, want) < 2e-13
        assert rel_state_err_blocks(got, oracle.rk4_step(z, 1.0, terms=terms, **par)) > 1e-9      # really another method
    w = workloads.config0()
    with mc.Integrator(integrator=mc.MC_INTEG_RK5) as I:
        g = I.integrate(w.states, 1.0, 1000, 3)
        info = I.launch_info()
    o = oracle.integrate(w.states, 1.0, 1000, 3, integrator=oracle.RK5, **w.params())
    assert info["local_bytes"] == 0 and (info["variant"] >> 8) & 1 == 1
    assert rel_state_err(g.states.cpu().numpy(), o.states) <= STATE_RTOL
    assert drift(g.states.cpu().numpy(), o.invariants[0:6], **w.params()) <= DRIFT_TOL
    assert np.array_equal(g.steps_done.cpu().numpy(), o.steps_done)
    w = workloads.config1().subset(np.arange(150))
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    with mc.Integrator(terms=w.terms, integrator=mc.MC_INTEG_RK5, **kw) as I:
        g = I.integrate(w.states, 1.0, 1500, 3, shadow_eps=1e-8)
    with mc.Integrator(terms=w.terms, integrator=mc.MC_INTEG_RK5, chunk_steps=170, **kw) as I:
        gc = I.integrate(w.states, 1.0, 1500, 3, shadow_eps=1e-8)
    o = oracle.integrate(w.states, 1.0, 1500, 3, shadow_eps=1e-8, integrator=oracle.RK5, **w.params())
    assert rel_state_err(g.states.cpu().numpy(), o.states) <= 4 * STATE_RTOL
    assert np.abs(g.fli.cpu().numpy() - o.fli).max() < FLI_VALUE_TOL
    assert np.array_equal(g.status.cpu().numpy(), o.status)
    assert np.array_equal(g.states.cpu().numpy(), gc.states.cpu().numpy())       # chunking: bit-identical
    assert np.array_equal(g.fli.cpu().numpy(), gc.fli.cpu().numpy())


def test_step_size_and_tolerance_studies(mc):
    """convergence in h for both base integrators and the Newton-tolerance study of
    PAPER.md:195-197 (epsilon = 1e-6, 1e-8, 1e-10) for the mode-3 correction.  Prints the tables recorded in
    profiles/r01_rk5_and_studies.md (run with -s)."""
    w = workloads.paper_orbit(1)                                     # PAPER.md:193 orbit 1 (regular), beta = 1/3, chi = 0.75
    par = dict(beta=float(w.beta[0]), chi1=float(w.chi1[0]), chi2=float(w.chi2[0]))
    t_end = 2048
    ref = oracle.integrate(w.states, 0.0625, t_end * 16, 0, integrator=oracle.RK5, **w.params()).states[:, 0]
    print("\\nh-study, paper orbit 1, uncorrected, t = %d: max |r - r_ref|" % t_end)
    errs = {}
    for integ, name in ((mc.MC_INTEG_RK4, "RK4"), (mc.MC_INTEG_RK5, "RK5")):
        with mc.Integrator(integrator=integ, **par) as I:
            for h in (4.0, 2.0, 1.0, 0.5):
                g = I.integrate(w.states, h, int(t_end / h), 0).states.cpu().numpy()[:, 0]
                errs[name, h] = np.abs(g[0:3] - ref[0:3]).max()
        print("  %s: " % name + "  ".join("h=%g: %.3e" % (h, errs[name, h]) for h in (4.0, 2.0, 1.0, 0.5)))
    assert 12 < errs["RK4", 2.0] / errs["RK4", 1.0] < 20 and 12 < errs["RK4", 4.0] / errs["RK4", 2.0] < 20     # 2^4
    assert 25 < errs["RK5", 4.0] / errs["RK5", 2.0] < 40 and 25 < errs["RK5", 2.0] / errs["RK5", 1.0] < 40     # 2^5
    assert errs["RK5", 1.0] < 0.1 * errs["RK4", 1.0]

    w0 = workloads.config0()
    print("epsilon-study, config 0 (64 orbits), RK4 h = 1, 1e4 steps, mode 3, cap 4: max relative drift of E, J; "
          "Gauss-Newton steps per step")
    res = {}
    for eps in (1e-4, 1e-6, 1e-8, 1e-10, 0.0):
        with mc.Integrator(newton_tol=eps) as I:
            g = I.integrate(w0.states, 1.0, 10_000, 3)
            gn = I.work(64).cpu().numpy().mean() / 10_000
        inv0 = g.invariants.cpu().numpy()[0:6]
        I1 = oracle.integrals(g.states.cpu().numpy(), **w0.params())
        dE = (np.abs(I1[0] - inv0[0]) / np.abs(inv0[0])).max()
        dJ = (np.linalg.norm(I1[1:4] - inv0[1:4], axis=0) / np.linalg.norm(inv0[1:4], axis=0)).max()
        res[eps] = (dE, dJ, gn)
        print("  eps=%-6g dE=%.2e dJ=%.2e steps=%.3f" % (eps, dE, dJ, gn))
    with mc.Integrator() as I:
        g0 = I.integrate(w0.states, 1.0, 10_000, 0)
    E0 = oracle.integrals(w0.states, **w0.params())[0]
    dE0 = (np.abs(oracle.integrals(g0.states.cpu().numpy(), **w0.params())[0] - E0) / np.abs(E0)).max()
    print("  uncorrected RK4: dE=%.2e" % dE0)
    assert dE0 > 1e-9                                                  # the correction has work to do
    assert max(res[1e-10][0:2]) <= DRIFT_TOL and max(res[1e-8][0:2]) <= DRIFT_TOL
    assert res[1e-4][2] <= res[1e-8][2] <= res[0.0][2] and res[0.0][2] > 2.5    # eps = 0: runs to the cap
    assert res[1e-4][2] < 1.05                                          # loose tolerance: one step per step


def test_sampled_trajectory_output_matches_oracle(mc):
    """SURVEY 8(f) row 3 (mc_integrate_sampled): states after every 50th step, 1234 steps (a trailing partial
    interval), strong-field grid with dropped cells (whole warps and single lanes) + regular orbits."""
    z = np.concatenate([workloads.scan_grid(6, 20, r_lo=6.0, r_hi=9.0)[0], workloads.config0(100).states], axis=1)
    n = z.shape[1]
    with mc.Integrator() as I:
        g = I.integrate(z, 1.0, 1234, 3, shadow_eps=1e-8, sample_interval=50)
        plain = I.integrate(z, 1.0, 1234, 3, shadow_eps=1e-8)
    with mc.Integrator(chunk_steps=170) as I:
        gc = I.integrate(z, 1.0, 1234, 3, shadow_eps=1e-8, sample_interval=50)
    o = oracle.integrate(z, 1.0, 1234, 3, shadow_eps=1e-8, sample_interval=50)
    S, So = g.samples.cpu().numpy(), o.samples
    assert S.shape == So.shape == (24, 12, n)
    assert np.array_equal(g.status.cpu().numpy(), o.status) and (o.status != 0).sum() >= 20
    assert np.array_equal(g.states.cpu().numpy(), plain.states.cpu().numpy())        # sampling changes nothing else
    assert np.array_equal(S, gc.samples.cpu().numpy())                                # nor does chunking
    live = o.status == 0
    for s in range(24):
        assert rel_state_err(S[s][:, live], So[s][:, live]) < 2e-9                    # 1234 steps, some cells chaotic
    calm = live & (o.fli < 3.0)
    assert calm.sum() > 80 and rel_state_err(S[23][:, calm], So[23][:, calm]) <= 2 * STATE_RTOL
    dead = np.where(~live)[0]                                                          # frozen state is reported on
    last = S[23][:, dead]
    assert np.array_equal(last, g.states.cpu().numpy()[:, dead])
    assert np.abs(last - So[23][:, dead]).max() < 1e-6


def test_full_grid_classification_against_the_oracle(mc):
    """north_star, literally: "FLI regular/chaotic classification agreeing on >= 99 % of grid cells".  The whole
    314 x 314 scan at 1e5 steps in the launch configuration bench.py times, every one of the 98 596 cells compared
    with the long-double oracle's result stored in tests/golden/config2_1e5_oracle.npz (written by
    tests/golden/make_config2_golden.py, which calls only oracle/; about an hour of 16 cores).  Classes: regular
    (FLI < 5.8), chaotic, dropped."""
    import os
    gold = np.load(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config2_1e5_oracle.npz"))
    w = workloads.config2()
    assert w.n_orbits == gold["fli"].size == 98596 and w.n_steps == 100_000
    with mc.Integrator() as I:
        g = I.integrate(w.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps)
        work = I.work(w.n_orbits).cpu().numpy()
    gs, gfli, gk = g.status.cpu().numpy(), g.fli.cpu().numpy(), g.steps_done.cpu().numpy()
    ofli, ost, ok_ = gold["fli"], gold["status"].astype(np.int32), gold["steps"].astype(np.int64)
    cg, co = classes(gfli, gs), classes(ofli, ost)
    agree = (cg == co).mean()
    conf = np.array([[((co == a) & (cg == b)).sum() for b in range(3)] for a in range(3)])
    near = np.abs(ofli - FLI_THRESHOLD) < 0.5
    reg = (co == 0) & (cg == 0) & (ofli < 4.5)
    dfli = np.abs(gfli[reg] - ofli[reg])
    print("\nfull grid vs stored oracle: agreement %.5f (%d of %d cells differ); confusion matrix rows = oracle (regular, chaotic, "
          "dropped), columns = GPU:\n%s\ncells with |FLI_oracle - 5.8| < 0.5: %d, of which differing: %d; status equal on %.5f; "
          "steps_done equal on %.5f; |dFLI| on regular cells (FLI < 4.5): median %.2e, q99 %.2e, max %.2e"
          % (agree, (cg != co).sum(), cg.size, conf, near.sum(), (near & (cg != co)).sum(), (gs == ost).mean(), (gk == ok_).mean(),
             np.median(dfli), np.quantile(dfli, 0.99), dfli.max()))
    assert (co == 0).sum() > 80_000 and (co == 1).sum() > 5000 and (co == 2).sum() > 1000      # all three classes occur
    assert agree >= 0.99
    assert ((cg == 2) == (co == 2)).mean() >= 0.995
    assert np.median(dfli) < 0.02 and np.quantile(dfli, 0.99) < 0.1
    # regular cells: same number of completed steps, Gauss-Newton work within 1 % (decisions at the eps threshold, R6)
    both = (co == 0) & (cg == 0)
    assert (gk[both] == ok_[both]).all()
    assert abs(work[both].sum() / gold["gn_steps"][both].sum() - 1) < 0.01


def test_config3_quadrupole_scan_at_full_length_sampled_against_oracle(mc):
    """BASELINE config 3 at full size and full length (314 x 314, beta = 0.8, chi = 0.9, per-orbit kappa in [1, 8], 1e5
    steps), QM on and QM off on identical seeds through the scan front end.  400 cells drawn uniformly from the grid
    are recomputed by the long-double oracle both ways: regular / not-regular agrees on >= 99 % (north_star's bar is on
    grid cells, so the sample is uniform).  100 more cells come from the strong-field rows (r0 < 18, where every chaotic
    and dropped cell lives and single cells flip between "chaotic" and "dropped" with the last bits, R19).  The three-way
    agreement is held against the flips of the oracle's own double instance on the same cells (derived bar, below).  The
    class-change matrix QM off -> QM on of the sampled cells is the oracle's up to the cells whose class differs."""
    from paper_1802_00147_b200 import scan
    w_on, w_off = workloads.config3(qm=True), workloads.config3(qm=False)
    assert w_on.n_steps == 100_000 and np.array_equal(w_on.states, w_off.states)
    on, off = scan.run_scan(w_on), scan.run_scan(w_off)
    from conftest import config3_sample
    idx, is_uni = config3_sample()
    uni, strong = idx[is_uni], idx[~is_uni]
    res = {}
    for name, w, g in (("on", w_on, on), ("off", w_off, off)):
        sub = w.subset(idx)
        o = oracle.integrate(sub.states, 1.0, w.n_steps, 3, shadow_eps=1e-8, **sub.params())
        cg = scan.classes(g["fli"].ravel()[idx], g["status"].ravel()[idx])
        co = scan.classes(o.fli, o.status)
        res[name] = (cg, co)
        bad = np.where(cg != co)[0]
        print("config 3 QM %s: uniform sample %d cells, oracle classes regular/chaotic/dropped %s, agreement %.4f; strong-field "
              "sample %d cells %s, agreement %.4f; differing cells (row, col, oracle, gpu): %s"
              % (name, uni.size, [int((co[is_uni] == k).sum()) for k in range(3)], (cg == co)[is_uni].mean(), strong.size,
                 [int((co[~is_uni] == k).sum()) for k in range(3)], (cg == co)[~is_uni].mean(),
                 [(int(idx[i] // 314), int(idx[i] % 314), int(co[i]), int(cg[i])) for i in bad]))
        # north_star's classification is regular vs chaotic.  Every disagreement measured here (5 of 400 uniform cells with
        # QM on, gpurun_out/r2_pytest3.log) is a strongly chaotic cell that one side still counts as "chaotic" while on the
        # other its plunge below r_merge = 2 came before t = 1e5 ("dropped"): the last bits decide that (R19), and with
        # kappa up to 8 one cell in six of this grid is chaotic or dropped (one in eleven for config 2).  So the 99 % bar
        # is asserted on regular vs not-regular, and the three-way agreement is asserted at the level the flips allow.
        assert ((cg == 0) == (co == 0))[is_uni].mean() >= 0.99
        assert ((cg == 0) == (co == 0))[~is_uni].mean() >= 0.97
        # Three classes: the bar is DERIVED, not a literal.  The oracle's own double instance on the same cells flips
        # k_dbl of them against its long-double instance (tests/test_oracle_conventions.py pins on CPU that those flips
        # exist and are chaotic <-> dropped only); the GPU is another double-precision realisation, so its count k_gpu is
        # a second draw from the same distribution: the two may differ by two standard deviations of a Poisson
        # difference, 2 sqrt(k_gpu + k_dbl).  Flips that involve "regular" are bounded by the 99 % / 97 % above.
        od = oracle.integrate(sub.states, 1.0, w.n_steps, 3, shadow_eps=1e-8, precision=oracle.DOUBLE, **sub.params())
        cd = scan.classes(od.fli, od.status)
        for part, label in ((is_uni, "uniform"), (~is_uni, "strong-field")):
            k_gpu, k_dbl = int((cg != co)[part].sum()), int((cd != co)[part].sum())
            print("config 3 QM %s, %s sample: three-way flips vs long double: GPU %d, oracle double instance %d of %d cells"
                  % (name, label, k_gpu, k_dbl, int(part.sum())))
            assert k_gpu - k_dbl <= 2.0 * np.sqrt(k_gpu + k_dbl), (name, label, k_gpu, k_dbl)
        print("  of the GPU's flips, chaotic <-> dropped: %d of %d" % (sum({int(cg[i]), int(co[i])} == {1, 2} for i in bad), bad.size))
        reg = (co == 0) & (cg == 0) & (o.fli < 4.5)
        d = np.abs(g["fli"].ravel()[idx][reg] - o.fli[reg])
        assert reg.sum() > 300 and np.median(d) < 0.02 and np.quantile(d, 0.99) < 0.2
    changed_gpu = res["on"][0] != res["off"][0]
    changed_or = res["on"][1] != res["off"][1]
    assert (changed_gpu != changed_or).sum() <= 0.03 * idx.size
    cmp = scan.compare_runs(off, on)
    assert cmp["matrix"].sum() == 314 * 314 and cmp["live_both"] > 80_000
    assert cmp["mean_abs_dfli_regular"] > 1e-3                       # the term really changes the dynamics


@pytest.mark.parametrize("case", ["uniform-shadow", "per-orbit-qm-rk5", "dropped-cells", "no-shadow-mode2"])
def test_checkpoint_resume_is_bitwise_identical_to_one_run(mc, case):
    """SURVEY section 5 (checkpoint / resume), mc_integrate_ex: 3 calls of 310 + 457 + 233 steps, resumed from the
    caller-owned carry buffer, reproduce one 1000-step call bit for bit in every output (states, final invariants,
    FLI, status, cumulative step and work counters), with and without internal chunking."""
    mode, eps, kw = 3, 1e-8, {}
    if case == "uniform-shadow":
        z = workloads.config0(300).states
    elif case == "per-orbit-qm-rk5":
        w = workloads.config3(n_r=7, n_theta=19, qm=True)
        z, kw = w.states, dict(terms=w.terms, integrator=mc.MC_INTEG_RK5, per_orbit=1, **{k: v for k, v in w.params().items() if k != "terms"})
    elif case == "dropped-cells":
        z = workloads.scan_grid(12, 11, r_lo=6.0, r_hi=16.0)[0]
    else:
        z, mode, eps = workloads.config0(70).states, 2, 0.0
    n = z.shape[1]
    with mc.Integrator(**kw) as I:
        one = I.integrate(z, 1.0, 1000, mode, shadow_eps=eps)
        one_work = I.work(n).cpu().numpy()
    for chunk in (0, 90):
        with mc.Integrator(chunk_steps=chunk, **kw) as I:
            a = I.integrate_ex(z, 1.0, 310, mode, shadow_eps=eps)
            b = I.integrate_ex(None, 1.0, 457, mode, shadow_eps=eps, carry=a.carry, resume=True, n_orbits=n, invariants=a.invariants)
            c = I.integrate_ex(None, 1.0, 233, mode, shadow_eps=eps, carry=a.carry, resume=True, n_orbits=n, invariants=a.invariants)
            work = I.work(n).cpu().numpy()
        for x, y in ((one.states, c.states), (one.invariants, c.invariants), (one.status, c.status), (one.steps_done, c.steps_done)):
            assert np.array_equal(x.cpu().numpy(), y.cpu().numpy(), equal_nan=True), (case, chunk)
        if eps != 0.0:
            assert np.array_equal(one.fli.cpu().numpy(), c.fli.cpu().numpy(), equal_nan=True)
        assert np.array_equal(one_work, work)


def test_scan_command_line_tool(mc, tmp_path):
    """paper_1802_00147_b200.scan: the scan front end writes FLI / status / image files from a GPU run."""
    from paper_1802_00147_b200 import scan
    out = scan.main(["--scan", "paper-theta2", "--steps", "600", "--out", str(tmp_path / "s.npz"), "--pgm", str(tmp_path / "s.pgm")])
    z = np.load(tmp_path / "s.npz")
    assert z["fli"].shape == (314,) and z["states"].shape == (12, 314) and np.array_equal(z["fli"], out["fli"])
    head = (tmp_path / "s.pgm").read_bytes()[:15]
    assert head.startswith(b"P5\n314 1\n255\n")
    w = workloads.paper_scan_theta2(n_steps=600)
    o = oracle.integrate(w.states, 1.0, 600, 3, shadow_eps=1e-8, **w.params())
    assert np.array_equal(z["status"], o.status & 255) and np.abs(z["fli"] - o.fli).max() < FLI_VALUE_TOL


def test_config1_full_size_correction_on_and_off_in_the_same_run(mc):
    """BASELINE config 1 at full size and length: 1024 orbits, per-orbit beta and chi, 1e5 steps, shadow + FLI,
    the same inputs once with the correction (mode 3) and once without (mode 0).  Drift of the six integrals on
    every orbit both ways (oracle-evaluated, R18); 48 sampled orbits recomputed by the oracle both ways."""
    w = workloads.config1()
    assert w.n_orbits == 1024 and w.n_steps == 100_000
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    out = {}
    with mc.Integrator(terms=w.terms, **kw) as I:
        for mode in (3, 0):
            out[mode] = I.integrate(w.states, w.h, w.n_steps, mode, shadow_eps=w.shadow_eps)
    inv0 = out[3].invariants.cpu().numpy()[0:6]
    live3 = out[3].status.cpu().numpy() == 0
    assert live3.mean() > 0.95
    d3 = drift(out[3].states.cpu().numpy()[:, live3], inv0[:, live3], **w.subset(np.where(live3)[0]).params())
    live0 = out[0].status.cpu().numpy() == 0
    I1 = oracle.integrals(out[0].states.cpu().numpy()[:, live0], **w.subset(np.where(live0)[0]).params())
    dE0 = np.abs(I1[0] / inv0[0][live0] - 1)
    assert d3 <= DRIFT_TOL and np.median(dE0) > 1e-9 and dE0.max() > 1e-6        # the correction has work to do
    idx = np.sort(np.random.default_rng(11).choice(1024, 48, replace=False))
    sub = w.subset(idx)
    for mode in (3, 0):
        o = oracle.integrate(sub.states, w.h, w.n_steps, mode, shadow_eps=w.shadow_eps, **sub.params())
        gs, gfli = out[mode].status.cpu().numpy()[idx], out[mode].fli.cpu().numpy()[idx]
        assert (gs == o.status).mean() >= 0.95
        assert (classes(gfli, gs) == classes(o.fli, o.status)).mean() >= 0.95
        reg = (o.status == 0) & (gs == 0) & (o.fli < 4.5)                 # bulk bound, loose cap: see the config-2 test
        dfli = np.abs(gfli[reg] - o.fli[reg])
        # corrected runs stay closer to the oracle (both sides are pulled onto the same manifold every step):
        # measured median / max 0.002 / 0.017 with the correction, 0.03 / 0.10 without
        med, q90 = (0.02, 0.1) if mode == 3 else (0.1, 0.3)
        assert reg.sum() >= 30 and np.median(dfli) < med and np.quantile(dfli, 0.9) < q90 and dfli.max() < 2.0


def test_config3_full_size_quadrupole_sampled_against_oracle(mc):
    """BASELINE config 3 at full size (314 x 314, beta = 0.8, chi = 0.9, per-orbit kappa in [1, 8], QM on), 1e4
    steps: drift on every live cell, 40 sampled cells recomputed by the oracle."""
    w = workloads.config3(n_steps=10_000, qm=True)
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    with mc.Integrator(terms=w.terms, **kw) as I:
        g = I.integrate(w.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps)
        info = I.launch_info()
    assert info["local_bytes"] == 0 and info["variant"] & 7 == 6          # QM on, per-orbit kappa only (per_orbit = 2)
    gs, gz, gfli = g.status.cpu().numpy(), g.states.cpu().numpy(), g.fli.cpu().numpy()
    live = gs == 0
    assert 0.7 < live.mean() < 1.0
    inv0 = g.invariants.cpu().numpy()[0:6]
    assert drift(gz[:, live], inv0[:, live], **w.subset(np.where(live)[0]).params()) <= DRIFT_TOL
    idx = np.sort(np.random.default_rng(5).choice(314 * 314, 40, replace=False))
    sub = w.subset(idx)
    o = oracle.integrate(sub.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps, **sub.params())
    assert (gs[idx] == o.status).mean() >= 0.95
    same = gs[idx] == o.status
    assert np.array_equal(g.steps_done.cpu().numpy()[idx][same & (o.status == 0)], o.steps_done[same & (o.status == 0)])
    reg = (o.status == 0) & (gs[idx] == 0) & (o.fli < 4.0)
    assert reg.sum() >= 20 and np.abs(gfli[idx][reg] - o.fli[reg]).max() < 0.02
    assert rel_state_err(gz[:, idx][:, reg], o.states[:, reg]) < 1e-6


def test_config4_maximum_size_properties(mc):
    """BASELINE config 4 at its largest size, 2^20 orbits + shadows (2 M trajectories, 65 536 work units), 300
    steps: the second half of the batch repeats the first half and must reproduce it bit for bit; the six
    integrals hold on every orbit (oracle-evaluated)."""
    half = workloads.config4(19, n_steps=300)
    z = np.concatenate([half.states, half.states], axis=1)
    n = z.shape[1]
    assert n == 1 << 20
    with mc.Integrator() as I:
        g = I.integrate(z, 1.0, 300, 3, shadow_eps=1e-8)
        info = I.launch_info()
    assert info["trajectories"] == 2 * n and info["local_bytes"] == 0
    gz, gf = g.states.cpu().numpy(), g.fli.cpu().numpy()
    assert np.array_equal(gz[:, : n // 2], gz[:, n // 2:]) and np.array_equal(gf[: n // 2], gf[n // 2:])
    assert (g.status.cpu().numpy() == 0).all() and (g.steps_done.cpu().numpy() == 300).all()
    inv = g.invariants.cpu().numpy()
    I1 = oracle.integrals(gz[:, : n // 2], **half.params())
    assert np.abs(I1[0] / inv[0, : n // 2] - 1).max() <= DRIFT_TOL
    assert (np.linalg.norm(I1[1:4] - inv[1:4, : n // 2], axis=0) / np.linalg.norm(inv[1:4, : n // 2], axis=0)).max() <= DRIFT_TOL
    assert np.abs(inv[6:12, : n // 2] - I1).max() < 1e-13                    # the kernel's own final invariants agree


RR = workloads.TERM_RR


@pytest.mark.parametrize("terms", [RR, 15 | RR, 31 | RR])
def test_radiation_reaction_model_routines_match_oracle(mc, terms):
    """SURVEY 8(f) row 4 (MC_TERM_RR; eq 6; R21): dz/dt with the 2.5PN force and the rates
    of the work and torque integrals (16 rows), one RK4 / RK5 step of all 16 components."""
    z = random_states(300, seed=31)
    par = PARAM_SETS[1]
    for integ, ointeg in ((mc.MC_INTEG_RK4, oracle.RK4), (mc.MC_INTEG_RK5, oracle.RK5)):
        with mc.Integrator(terms=terms, integrator=integ, **par) as I:
            got = I.eval("rhs", z).cpu().numpy()
            step = I.eval("rk4_step", z, h=1.0).cpu().numpy()
        want = oracle.evaluate("rhs16", z, terms=terms, **par)
        assert got.shape == (16, 300)
        assert rel_state_err_blocks(got[0:12], want[0:12]) < 2e-13
        assert np.abs(got[12] / want[12] - 1).max() < 1e-12                           # dW/dt
        assert (np.linalg.norm(got[13:16] - want[13:16], axis=0) / np.linalg.norm(want[13:16], axis=0)).max() < 1e-12
        plain = oracle.rhs(z, terms=terms & ~RR, **par)
        assert rel_state_err_blocks(got[3:6], plain[3:6]) > 1e-9                      # the force really is in dp/dt
        o = oracle.integrate(z, 1.0, 1, 0, terms=terms, integrator=ointeg, r_merge=0.0, r_escape=1e9, **par)
        assert rel_state_err_blocks(step[0:12], o.states) < 2e-13
        assert np.abs(step[12] / o.diss[0] - 1).max() < 1e-11 and np.abs(step[13:16] - o.diss[1:4]).max() < 1e-13 * np.abs(o.diss[1:4]).max()


@pytest.mark.parametrize("mode", [0, 2, 3])
def test_radiation_reaction_runs_match_oracle(mc, mode):
    """Dissipative runs: config-0 orbits and the paper's orbit 3 with the 2.5PN term, shadow on.  State
    parity, status, FLI, and the moving references E0 + W, J0 + G (mc_get_dissipation) against the oracle's W, G;
    with the correction the integral invariant relation holds to round-off on the GPU's output (oracle-evaluated)."""
    w = workloads.config0(149)
    wide = w.states.copy()                     # config-0 orbits moved out to a in [45, 90]: the leading-order force is a
    wide[0:3] *= 3.0                           # perturbation there (at the 3.7 M periastra of the originals it is not, and
    wide[3:6] /= np.sqrt(3.0)                  # those orbits merge within a few hundred steps -- on both sides alike)
    z = np.concatenate([wide, workloads.paper_orbit(3).states], axis=1)
    par = dict(beta=1.0, chi1=1.0, chi2=0.85)
    terms = 15 | RR
    n = z.shape[1]
    EPS = 3e-8      # the same RELATIVE offset as 1e-8 at r ~ 20 (configs 0-2): the FLI is the log of a separation that small,
                    # so it magnifies the 1e-16 |r| rounding of the state by |r| / EPS
    with mc.Integrator(terms=terms, **par) as I:
        g = I.integrate(z, 1.0, 1000, mode, shadow_eps=EPS)
        ref = I.dissipation(n).cpu().numpy()
        info = I.launch_info()
    with mc.Integrator(terms=terms, chunk_steps=170, **par) as I:
        gc = I.integrate(z, 1.0, 1000, mode, shadow_eps=EPS)
        refc = I.dissipation(n).cpu().numpy()
    o = oracle.integrate(z, 1.0, 1000, mode, shadow_eps=EPS, terms=terms, **par)
    assert info["local_bytes"] == 0 and info["variant"] & 8
    gz, ginv = g.states.cpu().numpy(), g.invariants.cpu().numpy()
    assert np.array_equal(g.status.cpu().numpy() & 255, o.status & 255) and ((o.status & 255) == 0).all()
    clean = o.status == 0                                                              # mode 2: no skipped step (R7)
    assert clean.sum() >= (30 if mode == 2 else n)
    assert rel_state_err(gz[:, clean], o.states[:, clean]) <= (2e-9 if mode == 2 else STATE_RTOL)
    dfli = np.abs(g.fli.cpu().numpy()[clean] - o.fli[clean])
    if mode == 2:      # the dual scaling is singular twice per radial period (R7): bound on the bulk, loose cap on the worst orbit
        assert np.median(dfli) < 5e-3 and np.quantile(dfli, 0.9) < 5e-2 and dfli.max() < 0.5
    else:
        assert dfli.max() < FLI_VALUE_TOL
    W = ref[0] - ginv[0]
    G = ref[1:4] - ginv[1:4]
    assert (W < 0).all()                                                               # energy is radiated
    assert np.abs(W[clean] / o.diss[0][clean] - 1).max() < 1e-6                        # E0 + W carries 1e-16 E0 of rounding, W ~ 1e-7 E0
    assert (np.linalg.norm(G - o.diss[1:4], axis=0) / np.linalg.norm(o.diss[1:4], axis=0))[clean].max() < 1e-6
    I1 = oracle.integrals(gz, terms=terms, **par)
    resE = np.abs(I1[0] - ref[0]) / np.abs(ginv[0])
    resJ = np.linalg.norm(I1[1:4] - ref[1:4], axis=0) / np.linalg.norm(ginv[1:4], axis=0)
    if mode == 3:
        assert resE.max() <= DRIFT_TOL and resJ.max() <= DRIFT_TOL                     # integral invariant relation
    elif mode == 2:
        assert resE[clean].max() <= DRIFT_TOL
    else:
        assert 1e-14 < resE.max() < 1e-6                                               # uncorrected: truncation error only
    assert np.array_equal(gz, gc.states.cpu().numpy()) and np.array_equal(ref, refc)   # chunking never changes a bit
    assert np.array_equal(g.fli.cpu().numpy(), gc.fli.cpu().numpy())


def test_radiation_reaction_variants_and_resume(mc):
    """The other instantiations of the dissipative kernel: per-orbit parameters, per-orbit kappa + QM, RK5; checkpoint /
    resume carries the moving references; the one combination that is not built is refused."""
    w = workloads.config3(n_r=6, n_theta=11, qm=True)
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    terms = w.terms | RR
    o = oracle.integrate(w.states, 1.0, 600, 3, shadow_eps=1e-8, **dict(w.params(), terms=terms))
    ok = o.status == 0
    assert ok.sum() > 30
    for force in (None, 1):
        with mc.Integrator(terms=terms, per_orbit=force, **kw) as I:
            g = I.integrate(w.states, 1.0, 600, 3, shadow_eps=1e-8)
            ref = I.dissipation(w.n_orbits).cpu().numpy()
            assert I.launch_info()["local_bytes"] == 0
        assert np.array_equal(g.status.cpu().numpy(), o.status)
        assert rel_state_err(g.states.cpu().numpy()[:, ok], o.states[:, ok]) <= STATE_RTOL
        W = ref[0] - g.invariants.cpu().numpy()[0]
        assert np.abs(W[ok] / o.diss[0][ok] - 1).max() < 1e-6
    o5 = oracle.integrate(w.states, 1.0, 600, 3, shadow_eps=1e-8, integrator=oracle.RK5, **dict(w.params(), terms=terms))
    with mc.Integrator(terms=terms, integrator=mc.MC_INTEG_RK5, **kw) as I:
        one = I.integrate(w.states, 1.0, 600, 3, shadow_eps=1e-8)
        one_ref = I.dissipation(w.n_orbits).cpu().numpy()
        a = I.integrate_ex(w.states, 1.0, 250, 3, shadow_eps=1e-8)
        b = I.integrate_ex(None, 1.0, 350, 3, shadow_eps=1e-8, carry=a.carry, resume=True, n_orbits=w.n_orbits, invariants=a.invariants)
        b_ref = I.dissipation(w.n_orbits).cpu().numpy()
    ok5 = o5.status == 0
    assert rel_state_err(one.states.cpu().numpy()[:, ok5], o5.states[:, ok5]) <= STATE_RTOL
    assert np.array_equal(one.states.cpu().numpy(), b.states.cpu().numpy()) and np.array_equal(one_ref, b_ref)
    assert np.array_equal(one.fli.cpu().numpy(), b.fli.cpu().numpy(), equal_nan=True)
    with mc.Integrator(terms=terms, integrator=mc.MC_INTEG_RK5, per_orbit=1, **kw) as I:   # not built: register budget (mc.h)
        with pytest.raises(mc.MCError) as e:
            I.integrate(w.states, 1.0, 10, 3, shadow_eps=1e-8)
        assert e.value.code == mc.MC_EINVAL
    with mc.Integrator(terms=w.terms, **kw) as I:                                       # without the bit: no dissipation output
        I.integrate(w.states, 1.0, 10, 3, shadow_eps=1e-8)
        with pytest.raises(mc.MCError):
            I.dissipation(w.n_orbits)


def test_mc_eval_rejects_null_references(mc):
    """mc_eval(what = 4) reads refs for every mode; a NULL must be MC_EINVAL, not a device fault."""
    z = random_states(40, seed=2)
    with mc.Integrator() as I:
        for mode in (0, 1, 2, 3):
            with pytest.raises(mc.MCError) as e:
                I.eval("correct", z, mode=mode, refs=None)
            assert e.value.code == mc.MC_EINVAL
        assert I.eval("H", z).shape == (1, 40)                                           # the handle is still usable


@pytest.mark.parametrize("integ", ["rk4", "rk5"])
def test_papers_dissipative_orbit3_at_full_length(mc, integ):
    """PAPER.md:219-223, Fig 5: orbit 3 (beta = 1, r = 50, p_y = 0.140, chi = 1 / 0.85) with the 2.5PN term, corrected,
    t = 1e5 -- the paper's RK5 and BASELINE's RK4 -- and 39 neighbours (r0 = 45 ... 55) to fill the warps.  The orbit
    loses 11 % of its binding energy; the relative error of the energy against the integral-invariant reference shows
    "no secular growth" (Fig 5a): round-off at the end of the run, on the GPU's output evaluated by the oracle."""
    w3 = workloads.paper_orbit(3)
    z = np.repeat(w3.states, 40, axis=1)
    z[0] = np.concatenate([[50.0], np.linspace(45.0, 55.0, 39)])
    z[4] = 0.140 * np.sqrt(50.0 / z[0])
    par = dict(beta=1.0, chi1=1.0, chi2=0.85)
    terms = 15 | RR
    with mc.Integrator(terms=terms, integrator=mc.MC_INTEG_RK5 if integ == "rk5" else mc.MC_INTEG_RK4, **par) as I:
        g = I.integrate(z, 1.0, 100_000, 3, shadow_eps=1e-8)
        ref = I.dissipation(40).cpu().numpy()
    o = oracle.integrate(z, 1.0, 100_000, 3, shadow_eps=1e-8, terms=terms,
                         integrator=oracle.RK5 if integ == "rk5" else oracle.RK4, **par)
    gz, ginv, gfli = g.states.cpu().numpy(), g.invariants.cpu().numpy(), g.fli.cpu().numpy()
    assert (o.status == 0).all() and np.array_equal(g.status.cpu().numpy(), o.status)
    assert np.array_equal(g.steps_done.cpu().numpy(), o.steps_done)
    W = ref[0] - ginv[0]
    assert 0.05 < W[0] / ginv[0, 0] < 0.2                                  # a tenth of the binding energy is radiated
    assert np.abs(W / o.diss[0] - 1).max() < 1e-8
    # the oracle's own double instance departs from its long-double one by 7e-10 on this run (regular orbit, 1e5 steps)
    assert rel_state_err(gz, o.states) < 2e-9
    I1 = oracle.integrals(gz, terms=terms, **par)
    assert (np.abs(I1[0] - ref[0]) / np.abs(ginv[0])).max() <= DRIFT_TOL
    assert (np.linalg.norm(I1[1:4] - ref[1:4], axis=0) / np.linalg.norm(ginv[1:4], axis=0)).max() <= DRIFT_TOL
    assert (gfli < FLI_THRESHOLD).all() and (o.fli < FLI_THRESHOLD).all() and np.abs(gfli - o.fli).max() < 0.1


@pytest.mark.parametrize("variant", ["kappa-qm", "rr", "rr-kappa-qm-rk5"])
def test_edge_cases_of_the_round2_kernel_variants(mc, variant):
    """Empty and ragged batches, n_steps = 0, in-place output and orbit permutation for the kernel variants added in round 2
    (per-orbit kappa, 2.5PN): the same properties test_edge_cases / test_batch_properties check for the base kernel."""
    w = workloads.config3(n_r=7, n_theta=19, qm=True)                       # 133 orbits: ragged (4 blocks + 10 lanes)
    kw = {k: v for k, v in w.params().items() if k != "terms"}
    terms = {"kappa-qm": w.terms, "rr": 15 | RR, "rr-kappa-qm-rk5": w.terms | RR}[variant]
    if variant == "rr":
        kw = dict(beta=0.8, chi1=0.9, chi2=0.9)
    integ = mc.MC_INTEG_RK5 if variant.endswith("rk5") else mc.MC_INTEG_RK4
    n = w.n_orbits

    def sub(idx):
        return {k: (v[idx] if hasattr(v, "__len__") else v) for k, v in kw.items()}
    with mc.Integrator(terms=terms, integrator=integ, **kw) as I:
        e = I.integrate(w.states[:, :0], 1.0, 10, 3, shadow_eps=1e-8)
        assert e.states.shape == (12, 0)
        zero = I.integrate(w.states, 1.0, 0, 3, shadow_eps=1e-8)
        assert np.allclose(zero.states.cpu().numpy(), w.states, rtol=1e-15, atol=0) and (zero.steps_done.cpu().numpy() == 0).all()
        a = I.integrate(w.states, 1.0, 400, 3, shadow_eps=1e-8)
        A, Af = a.states.cpu().numpy(), a.fli.cpu().numpy()
        zt = torch.as_tensor(w.states, device="cuda").clone()
        c = I.integrate(zt, 1.0, 400, 3, shadow_eps=1e-8, out_states=zt)             # in place
        assert np.array_equal(c.states.cpu().numpy(), A)
        if terms & RR:
            ref = I.dissipation(n).cpu().numpy()
            assert (ref[0] < a.invariants.cpu().numpy()[0])[a.status.cpu().numpy() == 0].all()      # energy only goes down
    perm = np.random.default_rng(4).permutation(n)
    with mc.Integrator(terms=terms, integrator=integ, **sub(perm)) as I:
        b = I.integrate(w.states[:, perm], 1.0, 400, 3, shadow_eps=1e-8)
    assert np.array_equal(A[:, perm], b.states.cpu().numpy(), equal_nan=True)         # orbits are independent
    assert np.array_equal(Af[perm], b.fli.cpu().numpy(), equal_nan=True)
    with mc.Integrator(terms=terms, integrator=integ, **sub(np.arange(1))) as I:     # a single orbit
        one = I.integrate(w.states[:, :1], 1.0, 400, 3, shadow_eps=1e-8)
    assert np.array_equal(one.states.cpu().numpy()[:, 0], A[:, 0], equal_nan=True)


def test_checked_build_runs_clean(mc):
    """SURVEY section 5 (sanitizers): compute-sanitizer is closed on this GPU pool, so the library has a checked build
    (-DMC_CHECKED, built by __graft_entry__.build()): every index and pointer is tested before the global access that
    uses it (mc_debug_check).  tests/checked_cases.py drives 40-odd representative launches through it in a process of
    its own; the product library must say it has no checks (-1)."""
    import os
    import subprocess
    import sys
    from paper_1802_00147_b200 import build
    with mc.Integrator() as I:
        I.integrate(workloads.config0(8).states, 1.0, 10, 3)
        assert I.debug_check() == -1
    lib = build.build_checked()
    env = dict(os.environ, MC_LIBMC_PATH=lib)
    script = os.path.join(os.path.dirname(os.path.abspath(__file__)), "checked_cases.py")
    r = subprocess.run([sys.executable, script], env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "launches clean" in r.stdout


@pytest.mark.parametrize("case", ["random-shadow", "random-no-shadow-in-place", "per-orbit", "kappa-qm-dropped", "rr", "nan-input"])
def test_regroup_never_changes_a_bit(mc, case):
    """mc_params.regroup: slot s of the launch integrates the s-th orbit in energy order.  An
    index mapping only: every output, in the caller's order, equals the unmapped run bit for bit -- ragged sizes, in
    place, per-orbit parameters (the mapping carries them along), dropped cells, 2.5PN, a NaN among the inputs."""
    kw, mode, eps, terms, steps = {}, 3, 1e-8, 15, 700
    if case == "random-shadow":
        z = workloads.config4(12).states[:, :1237]
    elif case == "random-no-shadow-in-place":
        z, eps = workloads.config4(12).states[:, :333], 0.0
    elif case == "per-orbit":
        w = workloads.config1().subset(np.arange(301))
        z, kw = w.states, {k: v for k, v in w.params().items() if k != "terms"}
    elif case == "kappa-qm-dropped":
        w = workloads.config3(n_r=10, n_theta=23, qm=True)
        z, terms, kw = w.states, w.terms, {k: v for k, v in w.params().items() if k != "terms"}
        steps = 3000
    elif case == "rr":
        z, terms = workloads.config4(12).states[:, :200] * np.array([3.0] * 3 + [3 ** -0.5] * 3 + [1.0] * 6)[:, None], 15 | RR
    else:
        z = workloads.config4(12).states[:, :130].copy()
        z[2, 77] = np.nan
    n = z.shape[1]
    outs = {}
    for rg in (0, 1):
        with mc.Integrator(terms=terms, regroup=rg, chunk_steps=(90 if rg else 0), **kw) as I:
            if case == "random-no-shadow-in-place":
                zt = torch.as_tensor(z, device="cuda").clone()
                g = I.integrate(zt, 1.0, steps, mode, shadow_eps=eps, out_states=zt)
            else:
                g = I.integrate(z, 1.0, steps, mode, shadow_eps=eps)
            info = I.launch_info()
            extra = [I.work(n).cpu().numpy()] + ([I.dissipation(n).cpu().numpy()] if terms & RR else [])
        assert bool(info["variant"] & 1024) == bool(rg)
        outs[rg] = [t.cpu().numpy() for t in (g.states, g.invariants, g.status, g.steps_done)] + extra + ([g.fli.cpu().numpy()] if eps else [])
    if case == "kappa-qm-dropped":
        assert (outs[0][2] != 0).sum() >= 10
    if case == "nan-input":
        assert outs[0][2][77] == 3 and (np.delete(outs[0][2], 77) == 0).all()
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b, equal_nan=True), case
    with mc.Integrator(regroup=1) as I:                       # below 64 orbits the mapping is not worth a sort: ignored
        I.integrate(z[:, :40], 1.0, 10, 3, shadow_eps=1e-8)
        assert not (I.launch_info()["variant"] & 1024)


def test_dual_scaling_skip_policy_and_root_selection_match_the_oracle(mc):
    """DESIGN.md R7 on the kernel's side: the constructed cases of tests/test_oracle_conventions.py
    (test_dual_scaling_skip_policy_and_root_selection) through mc_eval -- scaling applied for |v - 1| <= 1e-3, skipped
    with (r, p) untouched beyond, and the root continuous with gamma = 1 when L.L + L.S < 0."""
    par = dict(beta=1.0, chi1=0.9, chi2=0.8)
    z = workloads.paper_orbit(4).states
    J0 = oracle.total_J(z, terms=15, **par)
    states, refs = [], []
    for v in (1 + 5e-4, 1 - 8e-4, 1 + 1.5e-3, 1 - 1.5e-3):
        zs = z.copy()
        zs[0:3] /= v
        zs[3:6] *= v
        states.append(z)
        refs.append(np.concatenate([oracle.hamiltonian(zs, terms=15, **par)[None], J0], axis=0))
    y = np.zeros((12, 1))
    y[0], y[4], y[8], y[11] = 3.0, 0.05, -1.0, -1.0
    Ry = np.concatenate([oracle.hamiltonian(y, terms=15, **par)[None], oracle.total_J(y, terms=15, **par)], axis=0)
    yp = y.copy()
    yp[0:3] *= 1 + 2e-4
    yp[3:6] *= 1 - 1e-4
    states += [y, yp]
    refs += [Ry, Ry]
    Z, R = np.concatenate(states, axis=1), np.concatenate(refs, axis=1)
    want, ok = oracle.correct(Z, R[0], R[1:4], 2, newton_iters=6, terms=15, **par)
    assert list(ok) == [1, 1, 0, 0, 1, 1]
    with mc.Integrator(newton_iters=6, **par) as I:
        got = I.eval("correct", Z, mode=2, refs=R).cpu().numpy()
    assert rel_state_err(got, want) < 1e-12
    assert np.array_equal(got[0:6, 2:4], Z[0:6, 2:4])                    # skipped: (r, p) untouched, bit for bit
