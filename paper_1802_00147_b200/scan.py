"""Command-line phase-space scan: the use the paper makes of the method (Figs 6-7, Table 3).

    python -m paper_1802_00147_b200.scan --scan config2 --out fli.npz
    python -m paper_1802_00147_b200.scan --scan paper-plane --steps 100000 --pgm fig7.pgm
    python -m paper_1802_00147_b200.scan --scan config3 --compare-qm --report qm.md     # QM on vs off, identical seeds

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
    par = {k: v for k, v in w.params().items() if k != "terms"}      # the binding picks uniform / per-orbit kernels from the data
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


CLASS_NAMES = ("regular", "chaotic", "dropped")


def classes(fli, status):
    """0 regular (FLI < 5.8), 1 chaotic, 2 dropped (merged / unbound / non-finite): the three outcomes of a scan cell."""
    c = (np.asarray(fli) >= FLI_THRESHOLD).astype(int)
    c[(np.asarray(status) & 255) != 0] = 2
    return c


DFLI_EDGES = np.array([-np.inf, -3, -1, -0.3, -0.1, -0.03, -0.01, 0.01, 0.03, 0.1, 0.3, 1, 3, np.inf])


def compare_runs(a, b):
    """Cell-by-cell comparison of two scans of the same grid (e.g. the quadrupole-monopole term off / on, the study of
    PAPER.md:246-256 widened to a grid, BASELINE config 3): 3 x 3 class-change matrix (rows = a, columns = b),
    histogram and quantiles of dFLI = FLI_b - FLI_a over the cells that finish the run in both."""
    ca, cb = classes(a["fli"], a["status"]).ravel(), classes(b["fli"], b["status"]).ravel()
    matrix = np.array([[int(((ca == i) & (cb == j)).sum()) for j in range(3)] for i in range(3)])
    live = (ca != 2) & (cb != 2)
    d = (np.asarray(b["fli"]).ravel() - np.asarray(a["fli"]).ravel())[live]
    hist, _ = np.histogram(d, bins=DFLI_EDGES)
    both_regular = ((ca == 0) & (cb == 0))[live]
    q = lambda x: [float(v) for v in np.quantile(x, [0.01, 0.25, 0.5, 0.75, 0.99])] if x.size else [float("nan")] * 5
    return dict(matrix=matrix, changed=int((ca != cb).sum()), cells=int(ca.size), live_both=int(live.sum()),
                dfli_hist=hist, dfli_quantiles=q(d), dfli_quantiles_regular=q(d[both_regular]),
                mean_abs_dfli_regular=float(np.abs(d[both_regular]).mean()) if both_regular.any() else float("nan"))


def report_markdown(cmp, name_a, name_b, header=""):
    lines = [header, "", f"Class changes, rows = {name_a}, columns = {name_b} ({cmp['cells']} cells, {cmp['changed']} change class):", "",
             "| | " + " | ".join(CLASS_NAMES) + " |", "|---|---|---|---|"]
    for i, nm in enumerate(CLASS_NAMES):
        lines.append(f"| {nm} | " + " | ".join(str(int(v)) for v in cmp["matrix"][i]) + " |")
    lines += ["", f"dFLI = FLI({name_b}) - FLI({name_a}) over the {cmp['live_both']} cells alive in both runs:", "",
              "| dFLI bin | cells |", "|---|---|"]
    for k, cnt in enumerate(cmp["dfli_hist"]):
        lo, hi = DFLI_EDGES[k], DFLI_EDGES[k + 1]
        lines.append(f"| [{lo:g}, {hi:g}) | {int(cnt)} |")
    lines += ["", "quantiles 1 / 25 / 50 / 75 / 99 %: all live cells " + " / ".join(f"{v:+.4f}" for v in cmp["dfli_quantiles"]) +
              "; cells regular in both " + " / ".join(f"{v:+.4f}" for v in cmp["dfli_quantiles_regular"]) +
              f"; mean |dFLI| on cells regular in both {cmp['mean_abs_dfli_regular']:.4f}", ""]
    return "\n".join(lines)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--scan", default="config2", help="config2 | config3 | config3-qmoff | paper-plane | paper-theta2")
    ap.add_argument("--steps", type=int, default=None, help="steps of h = 1 (default 1e5)")
    ap.add_argument("--integrator", default="rk4", choices=["rk4", "rk5"])
    ap.add_argument("--mode", type=int, default=3, choices=[0, 1, 2, 3], help="correction mode (include/mc.h)")
    ap.add_argument("--out", default=None, help=".npz file: fli, status, steps, states")
    ap.add_argument("--pgm", default=None, help="grey-map image of the classes")
    ap.add_argument("--compare-qm", action="store_true",
                    help="run the scan twice on identical initial conditions, quadrupole-monopole term off and on, and report "
                         "the class-change matrix and the dFLI histogram (BASELINE config 3; PAPER.md:246-256)")
    ap.add_argument("--report", default=None, help="markdown file for the --compare-qm report")
    args = ap.parse_args(argv)
    if args.compare_qm:
        base = args.scan.replace("-qmoff", "")
        w_on, w_off = build_workload(base, args.steps), build_workload(base + "-qmoff", args.steps)
        assert np.array_equal(w_on.states, w_off.states) and np.array_equal(w_on.kq1, w_off.kq1)     # identical seeds
        on, off = run_scan(w_on, args.integrator, args.mode), run_scan(w_off, args.integrator, args.mode)
        cmp = compare_runs(off, on)
        head = (f"{base}: {w_on.n_orbits} orbits x {w_on.n_steps} steps, QM off {off['seconds']:.2f} s "
                f"({w_off.n_orbits * w_off.n_steps / off['seconds']:.3e} scheduled orbit-steps/s), QM on {on['seconds']:.2f} s "
                f"({w_on.n_orbits * w_on.n_steps / on['seconds']:.3e})")
        text = report_markdown(cmp, "QM off", "QM on", head)
        print(text)
        if args.report:
            with open(args.report, "w") as f:
                f.write(text)
        if args.out:
            np.savez_compressed(args.out, fli_on=on["fli"], status_on=on["status"], steps_on=on["steps"],
                                fli_off=off["fli"], status_off=off["status"], steps_off=off["steps"])
        if args.pgm:
            write_pgm(args.pgm, on)
        return dict(on=on, off=off, compare=cmp)
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
