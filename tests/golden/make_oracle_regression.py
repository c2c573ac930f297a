#!/usr/bin/env python
"""Writes tests/golden/oracle_conservative_regression.txt: final states (hex floats) of a few small runs of the
CPU oracle on the conservative Hamiltonian, every correction mode, with and without shadow / QM / RK5.

Purpose: the oracle gains opt-in terms over time (e.g. the 2.5PN radiation reaction).  A run WITHOUT
the new term bit must stay bit-identical to what the oracle computed before the term existed; this file is that
"before" (written at the commit that precedes the 2.5PN term).  Calls only oracle/ and the seeded input generator.

    python tests/golden/make_oracle_regression.py            # rewrite the fixture
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1802_00147_b200 import workloads  # noqa: E402

CASES = [  # name, terms, mode, shadow_eps, integrator, n_steps
    ("mode0", 15, 0, 0.0, oracle.RK4, 400),
    ("mode1-shadow", 15, 1, 1e-8, oracle.RK4, 400),
    ("mode2", 15, 2, 0.0, oracle.RK4, 400),
    ("mode3-shadow", 15, 3, 1e-8, oracle.RK4, 400),
    ("mode3-qm-shadow", 31, 3, 1e-8, oracle.RK4, 400),
    ("mode3-rk5", 15, 3, 0.0, oracle.RK5, 300),
    ("newtonian", 0, 0, 1e-8, oracle.RK4, 300),
]


def run_case(name, terms, mode, eps, integ, n_steps):
    w = workloads.config1().subset(np.arange(6))
    par = {k: v for k, v in w.params().items() if k != "terms"}
    par["kq1"], par["kq2"] = np.linspace(1, 6, 6), np.linspace(8, 2, 6)
    return oracle.integrate(w.states, 1.0, n_steps, mode, shadow_eps=eps, terms=terms, integrator=integ, **par)


def lines():
    for case in CASES:
        o = run_case(*case)
        for i in range(o.states.shape[1]):
            vals = list(o.states[:, i]) + [o.fli[i]] + list(o.invariants[:, i])
            yield "%s %d %d %d %d %s" % (case[0], i, o.status[i], o.steps_done[i], o.gn_steps[i],
                                         " ".join(float(v).hex() for v in vals))


if __name__ == "__main__":
    out = os.path.join(HERE, "oracle_conservative_regression.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_oracle_regression.py (oracle only); case orbit status steps gn_steps "
                "12 state + FLI + 12 invariants as hex floats\n")
        for l in lines():
            f.write(l + "\n")
    print("wrote", out)
