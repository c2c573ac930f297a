"""The roofline's flop figures are derived, not hand-counted: mc_flop_model runs
the kernels' own math templates with a counting scalar on the host.  These checks tie the model to the structure of
the method (stage counts, what each correction mode adds), to bench.py (which must use it) and to the oracle's
independent count (the factored kernel formulation may not need more work than the unfactored oracle).  CPU only."""
import numpy as np
import pytest

import oracle
import benchlib
from paper_1802_00147_b200 import binding, workloads

RK4, RK5 = binding.MC_INTEG_RK4, binding.MC_INTEG_RK5


def test_base_step_is_stages_times_rhs_plus_the_stage_sums():
    for terms in (0, 15, 31):
        m4 = benchlib.flop_model(terms, 3, RK4)
        m5 = benchlib.flop_model(terms, 3, RK5)
        assert m4["rhs"] == m5["rhs"]
        # classical RK4, low storage: 3 stage inputs + 4 accumulations of 12 components = 84 FMAs
        assert m4["base_step"]["flop"] == 4 * m4["rhs"]["flop"] + 2 * 84
        assert m4["base_step"]["fma"] == 4 * m4["rhs"]["fma"] + 84 and m4["base_step"]["special"] == 4
        # Butcher RK5: 6 stages; inputs 1 + 2 + 1 + 2 + 1, carried sums A4, S6 (1 + 2 + 1 + 1), output 2 + 1 + 1 + 1: 17 x 12 FMAs
        assert m5["base_step"]["flop"] == 6 * m5["rhs"]["flop"] + 2 * 204
        assert m4["rhs"]["special"] == 1                      # one rsqrt per RHS, no division


def test_terms_and_modes_add_what_they_should():
    base = benchlib.flop_model(15, 3, RK4)
    qm = benchlib.flop_model(31, 3, RK4)
    newt = benchlib.flop_model(0, 3, RK4)
    assert newt["rhs"]["flop"] == base["rhs"]["flop"]        # disabled terms are zero coefficients, not less work
    assert 30 <= qm["rhs"]["flop"] - base["rhs"]["flop"] <= 60 and qm["gn_step"]["flop"] > base["gn_step"]["flop"]
    m0, m1, m2 = (benchlib.flop_model(15, k, RK4) for k in (0, 1, 2))
    assert m0["correct_fixed"]["flop"] == 0 and m0["gn_step"]["flop"] == 0
    assert m1["correct_fixed"] == dict(fma=4, mul=8, add=0, special=2, flop=18)       # eq (10) twice: dot, rsqrt, 3 mul
    assert base["correct_fixed"]["flop"] == 18 + 12                                   # + L_t = J0 - s1 S1 - s2 S2
    assert m2["gn_step"]["flop"] == 0 and 200 < m2["correct_fixed"]["flop"] < 400      # polynomial dual scaling (SURVEY: ~0.3 k)
    assert 280 < base["gn_step"]["flop"] < 350 and base["gn_step"]["special"] == 2     # one rsqrt (eval) + one reciprocal (solve); 395 before the step was written in the {r, p, L} frame
    assert base["status"]["flop"] == 5
    it2, it6 = benchlib.flop_model(15, 2, RK4, 2), benchlib.flop_model(15, 2, RK4, 6)
    per_iter = (it6["correct_fixed"]["flop"] - it2["correct_fixed"]["flop"]) / 4
    assert 20 <= per_iter <= 40                                                        # one Horner pair + division per iteration


def test_radiation_reaction_adds_the_force_and_four_accumulations():
    """MC_TERM_RR: the force costs two coefficients (F = fr r + fp p) plus the rates dW/dt, dG/dt, and the RK step
    accumulates four more components (no stage inputs for them: they never enter the right-hand side)."""
    a, b = benchlib.flop_model(15, 3, RK4), benchlib.flop_model(15 | 32, 3, RK4)
    extra = b["rhs"]["flop"] - a["rhs"]["flop"]
    assert 20 <= extra <= 40 and b["rhs"]["special"] == 1
    assert b["base_step"]["flop"] == 4 * b["rhs"]["flop"] + 2 * (84 + 4 * 4)
    b5 = benchlib.flop_model(15 | 32, 3, RK5)
    assert b5["base_step"]["flop"] == 6 * b["rhs"]["flop"] + 2 * (204 + 5 * 4)          # b2 = 0: five accumulations
    assert b["gn_step"] == a["gn_step"]                                                # the projection uses grad H only
    assert b["correct_fixed"]["flop"] == a["correct_fixed"]["flop"]                    # the references are carried, not added


def test_kernel_formulation_needs_less_work_than_the_oracles():
    """the oracle's unfactored formulation costs about twice as much; using the kernel's own count for
    `roofline.achieved` is the conservative choice."""
    z = workloads.paper_orbit(2).states[:, 0]
    for terms in (15, 31):
        o = oracle.count_flops(z, terms=terms, mode=3, newton_iters=2)
        m = benchlib.flop_model(terms, 3, RK4)
        assert m["rhs"]["flop"] < o["rhs"] < 3.5 * m["rhs"]["flop"]
        assert m["base_step"]["flop"] < o["rk4_step"]
        assert m["correct_fixed"]["flop"] + 2 * m["gn_step"]["flop"] < o["correct"]


def test_bench_uses_the_model():
    import bench
    w = workloads.config2(n_r=2, n_theta=2, n_steps=1000)
    steps_done = np.array([1000, 1000, 400, 1000])
    gn = np.array([2400, 2300, 900, 2500])
    m = benchlib.flop_model(w.terms, 3, RK4)
    per_traj_step = m["base_step"]["flop"] + m["correct_fixed"]["flop"] + m["status"]["flop"]
    want = 2 * steps_done.sum() * per_traj_step + gn.sum() * m["gn_step"]["flop"] + (steps_done // 100).sum() * m["renorm"]["flop"]
    got = bench.algorithmic_flop(w, 3, RK4, steps_done, gn)
    assert got["flop_per_launch"] == want
    assert got["model"]["rhs"] == m["rhs"]["flop"]
    # no shadow: one trajectory per orbit, no renormalisation (config 0 was overstated 2x)
    w0 = workloads.config0(4, n_steps=1000)
    got0 = bench.algorithmic_flop(w0, 3, RK4, steps_done, gn)
    assert got0["flop_per_launch"] == steps_done.sum() * per_traj_step + gn.sum() * m["gn_step"]["flop"]


def test_model_rejects_bad_arguments():
    lib = benchlib.load_library()
    out = benchlib.mc_flop_model_t()
    import ctypes
    assert lib.mc_flop_model(64, 3, 0, 4, ctypes.byref(out)) == binding.MC_EINVAL
    assert lib.mc_flop_model(15, 4, 0, 4, ctypes.byref(out)) == binding.MC_EINVAL
    assert lib.mc_flop_model(15, 3, 2, 4, ctypes.byref(out)) == binding.MC_EINVAL
    assert lib.mc_flop_model(15, 3, 0, 0, ctypes.byref(out)) == binding.MC_EINVAL
    assert lib.mc_flop_model(15, 3, 0, 4, None) == binding.MC_EINVAL
