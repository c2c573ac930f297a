#!/usr/bin/env python
"""Writes tests/golden/config2_1e5_oracle.npz: BASELINE config 2 (the 314 x 314 scan, RK4 h = 1, 1e5 steps,
shadow 1e-8 renormalised every 100 steps, correction mode 3) integrated cell by cell by the LONG-DOUBLE CPU
oracle (oracle/pn_oracle.hpp).  The GPU test test_full_grid_classification_against_the_oracle compares all
98 596 cells of the kernel's scan with this file (north_star: FLI classes agree on >= 99 % of grid cells;
threshold 5.8).

Calls only oracle/ and the seeded input generator (paper_1802_00147_b200/workloads.py holds no arithmetic of
the method); never the CUDA path.  About 1 hour on 16 cores, 2 hours on 8.  Restartable: progress is kept in
<out>.partial.npz.

    python tests/golden/make_config2_golden.py [--threads N] [--out PATH] [--rows-per-block 8]

Stored arrays: fli float64[98596], status int16[98596] (mc_status), steps int32[98596] (completed steps),
gn_steps int64[98596] (Gauss-Newton steps, orbit + shadow), oracle_sha256 (of the oracle's two source files at
the time of writing), wall_s, threads.
"""
import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1802_00147_b200 import workloads  # noqa: E402


def oracle_hash():
    h = hashlib.sha256()
    for f in ("pn_oracle.hpp", "pn_oracle_capi.cpp"):
        h.update(open(os.path.join(ROOT, "oracle", f), "rb").read())
    return h.hexdigest()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--out", default=os.path.join(HERE, "config2_1e5_oracle.npz"))
    ap.add_argument("--rows-per-block", type=int, default=8)
    a = ap.parse_args()
    w = workloads.config2()
    assert w.n_orbits == 314 * 314 and w.n_steps == 100_000 and w.shadow_eps == 1e-8 and w.correction_mode == 3
    n = w.n_orbits
    sha = oracle_hash()
    part = a.out + ".partial.npz"
    fli, status = np.full(n, np.nan), np.zeros(n, np.int16)
    steps, gn = np.zeros(n, np.int32), np.zeros(n, np.int64)
    done, wall = 0, 0.0
    if os.path.exists(part):
        p = np.load(part)
        if str(p["oracle_sha256"]) == sha:
            fli, status, steps, gn, done, wall = p["fli"], p["status"], p["steps"], p["gn_steps"], int(p["done"]), float(p["wall_s"])
            print(f"resuming at orbit {done}", flush=True)
    blk = a.rows_per_block * 314
    threads = a.threads or oracle.max_threads()
    while done < n:
        hi = min(n, done + blk)
        sub = w.subset(np.arange(done, hi))
        t0 = time.time()
        o = oracle.integrate(sub.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps, n_threads=threads,
                             precision=oracle.LONG_DOUBLE, **sub.params())
        wall += time.time() - t0
        fli[done:hi], status[done:hi], steps[done:hi], gn[done:hi] = o.fli, o.status, o.steps_done, o.gn_steps
        done = hi
        np.savez(part[:-4], fli=fli, status=status, steps=steps, gn_steps=gn, done=done, wall_s=wall, oracle_sha256=sha)
        print(f"{done}/{n} orbits, {wall:.0f} s", flush=True)
    np.savez_compressed(a.out[:-4] if a.out.endswith(".npz") else a.out, fli=fli, status=status, steps=steps,
                        gn_steps=gn, oracle_sha256=sha, wall_s=wall, threads=threads)
    os.remove(part)
    print("wrote", a.out, f"({wall:.0f} s on {threads} threads)")


if __name__ == "__main__":
    main()
