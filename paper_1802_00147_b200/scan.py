"""Command-line phase-space scan: the use the paper makes of the method (Figs 6-7, Table 3).

    python -m paper_1802_00147_b200.scan --scan config2 --out fli.npz
    python -m paper_1802_00147_b200.scan --scan paper-plane --steps 100000 --pgm fig7.pgm

Integrates every orbit of a 2-D grid of initial conditions with its shadow (RK4 or RK5 + manifold correction), and
writes the fast Lyapunov indicator, the per-orbit status and the chaos mask (FLI >= 5.8).  Everything
is computed by libmc on the GPU (binding.Integrator); this module only generates inputs and writes files.
"""
import argparse
import time

import numpy as np

from . import binding, workloads

FLI_THRESHOLD = 5.8


def build_workload(name, n_steps):
    kw = {} if n_steps is None else {"n_steps": n_steps}
    if name == "config2":
        return workloads.config2(**kw)
    if name == "config3":
        return workloads.config3(qm=True, **kw)
    if name == "config3-qmoff":
        return workloads.config3(qm=False, **kw)
    if name == "paper-plane":
        return workloads.paper_scan_plane(**kw)
    if name == "paper-theta2":
        return workloads.paper_scan_theta2(**kw)
    raise SystemExit(f"unknown scan {name}")


def run_scan(w, integrator="rk4", mode=3, device=0):
    """-> dict(fli, status, steps, states, seconds): numpy arrays shaped like the grid (flat for 1-D scans)."""
    import torch
    par = (dict(beta=float(w.beta[0]), chi1=float(w.chi1[0]), chi2=float(w.chi2[0]), kq1=float(w.kq1[0]), kq2=float(w.kq2[0]))
           if w.uniform else {k: v for k, v in w.params().items() if k != "terms"})
    with binding.Integrator(terms=w.terms, device=device, integrator=int(integrator == "rk5"),
                            renorm_interval=w.renorm_interval, **par) as I:
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        res = I.integrate(w.states, w.h, w.n_steps, mode, shadow_eps=w.shadow_eps)
        torch.cuda.synchronize(device)
        dt = time.perf_counter() - t0
    shape = w.meta.get("shape", (w.n_orbits,))
    return dict(fli=res.fli.cpu().numpy().reshape(shape), status=(res.status.cpu().numpy() & 255).reshape(shape),
                steps=res.steps_done.cpu().numpy().reshape(shape), states=res.states.cpu().numpy(), seconds=dt)


def write_pgm(path, out):
    """8-bit grey map in the style of the paper's Fig 7: black = chaotic (FLI >= 5.8), light grey = regular,
    white = dropped (merged / unbound / non-finite)."""
    fli, status = np.atleast_2d(out["fli"]), np.atleast_2d(out["status"])
    img = np.where(status != 0, 255, np.where(fli >= FLI_THRESHOLD, 0, 170)).astype(np.uint8)
    with open(path, "wb") as f:
        f.write(b"P5\n%d %d\n255\n" % (img.shape[1], img.shape[0]))
        f.write(img.tobytes())


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--scan", default="config2", help="config2 | config3 | config3-qmoff | paper-plane | paper-theta2")
    ap.add_argument("--steps", type=int, default=None, help="steps of h = 1 (default 1e5)")
    ap.add_argument("--integrator", default="rk4", choices=["rk4", "rk5"])
    ap.add_argument("--mode", type=int, default=3, choices=[0, 1, 2, 3], help="correction mode (include/mc.h)")
    ap.add_argument("--out", default=None, help=".npz file: fli, status, steps, states")
    ap.add_argument("--pgm", default=None, help="grey-map image of the classes")
    args = ap.parse_args(argv)
    w = build_workload(args.scan, args.steps)
    out = run_scan(w, args.integrator, args.mode)
    ok = out["status"] == 0
    print(f"{w.name}: {w.n_orbits} orbits x {w.n_steps} steps in {out['seconds']:.2f} s; regular "
          f"{int((ok & (out['fli'] < FLI_THRESHOLD)).sum())}, chaotic {int((ok & (out['fli'] >= FLI_THRESHOLD)).sum())}, "
          f"dropped {int((~ok).sum())}")
    if args.out:
        np.savez_compressed(args.out, fli=out["fli"], status=out["status"], steps=out["steps"], states=out["states"])
    if args.pgm:
        write_pgm(args.pgm, out)
    return out


if __name__ == "__main__":
    main()
