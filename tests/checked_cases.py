"""Representative launches through the CHECKED build of the library (libmc_checked.so, -DMC_CHECKED): ragged sizes,
chunked scheduling with a carry buffer, sampled output, per-orbit / per-orbit-kappa / 2.5PN variants, checkpoint and
resume, dropped cells.  After each launch mc_debug_check must report 0 (no index or pointer test failed).  Run as a
script by tests/test_parity_gpu.py::test_checked_build_runs_clean with MC_LIBMC_PATH pointing at the checked library
(compute-sanitizer is closed on the GPU pool)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1802_00147_b200 import binding, workloads  # noqa: E402


def main():
    import torch
    cases = 0

    def clean(I, what):
        nonlocal cases
        torch.cuda.synchronize()
        line = I.debug_check()
        assert line == 0, f"{what}: check at mc_kernel.cuh:{line} failed" if line > 0 else f"{what}: not the checked library ({line})"
        cases += 1

    w0 = workloads.config0(300)
    for n in (1, 31, 33, 129, 300):
        for eps in (0.0, 1e-8):
            for chunk in (0, 37):
                with binding.Integrator(chunk_steps=chunk) as I:
                    I.integrate(w0.states[:, :n], 1.0, 150, 3, shadow_eps=eps, sample_interval=40)
                    clean(I, f"uniform n={n} eps={eps} chunk={chunk}")
    w1 = workloads.config1().subset(np.arange(150))
    kw1 = {k: v for k, v in w1.params().items() if k != "terms"}
    for mode in (0, 1, 2, 3):
        with binding.Integrator(terms=w1.terms, chunk_steps=64, **kw1) as I:
            I.integrate(w1.states, 1.0, 200, mode, shadow_eps=1e-8)
            clean(I, f"per-orbit mode {mode}")
    w3 = workloads.config3(n_r=7, n_theta=19, qm=True)
    kw3 = {k: v for k, v in w3.params().items() if k != "terms"}
    for terms, integ in ((w3.terms, 0), (w3.terms | 32, 0), (w3.terms | 32, 1), (15 | 32, 0)):
        with binding.Integrator(terms=terms, integrator=integ, chunk_steps=50, **kw3) as I:
            a = I.integrate_ex(w3.states, 1.0, 120, 3, shadow_eps=1e-8)
            clean(I, f"kappa terms={terms} integ={integ} first")
            I.integrate_ex(None, 1.0, 130, 3, shadow_eps=1e-8, carry=a.carry, resume=True, n_orbits=w3.n_orbits, invariants=a.invariants)
            clean(I, f"kappa terms={terms} integ={integ} resumed")
    z = workloads.scan_grid(12, 11, r_lo=6.0, r_hi=16.0)[0]                      # dropped cells, whole warps and single lanes
    with binding.Integrator(chunk_steps=100) as I:
        I.integrate(z, 1.0, 1500, 3, shadow_eps=1e-8, sample_interval=100)
        clean(I, "dropped cells")
    w4 = workloads.config4(12)
    for n in (64, 1237, 4096):
        with binding.Integrator(regroup=1, chunk_steps=70) as I:
            I.integrate(w4.states[:, :n], 1.0, 200, 3, shadow_eps=1e-8)
            assert I.launch_info()["variant"] & 1024
            clean(I, f"regroup n={n}")
    wl = workloads.config2(n_r=120, n_theta=314, n_steps=600)                    # 37 680 orbits: more units than resident warps
    with binding.Integrator() as I:
        I.integrate(wl.states, 1.0, 600, 3, shadow_eps=1e-8)
        info = I.launch_info()
        clean(I, "automatic chunking")
        assert info["n_chunks"] > 1
    print(f"checked build: {cases} launches clean")


if __name__ == "__main__":
    main()
