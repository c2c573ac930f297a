#!/usr/bin/env python
"""Writes tests/golden/config2_1e5_oracle.npz: BASELINE config 2 (the 314 x 314 scan, RK4 h = 1, 1e5 steps,
shadow 1e-8 renormalised every 100 steps, correction mode 3) integrated cell by cell by the LONG-DOUBLE CPU
oracle (oracle/pn_oracle.hpp).  The GPU test test_full_grid_classification_against_the_oracle compares all
98 596 cells of the kernel's scan with this file (north_star: FLI classes agree on >= 99 % of grid cells;
threshold 5.8).

Calls only oracle/ and the seeded input generator (paper_1802_00147_b200/workloads.py holds no arithmetic of
the method); never the CUDA path.  About 1 hour on 16 cores.  Restartable, and the orbit range can be split over
machines: each run keeps its progress in <out>.part_<lo>_<hi>.npz; --merge assembles the final file once the parts
cover all 98 596 orbits (orbits are independent and the long-double arithmetic is deterministic).

    python tests/golden/make_config2_golden.py [--threads N] [--lo A --hi B] [--out PATH] [--rows-per-block 8]
    python tests/golden/make_config2_golden.py --merge

Stored arrays: fli float64[98596], status int16[98596] (mc_status), steps int32[98596] (completed steps),
gn_steps int64[98596] (Gauss-Newton steps, orbit + shadow), oracle_sha256 (of the oracle's two source files at
the time each part was written), wall_s, how (ranges, seconds, threads).
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
    ap.add_argument("--lo", type=int, default=0)
    ap.add_argument("--hi", type=int, default=314 * 314)
    ap.add_argument("--merge", action="store_true")
    a = ap.parse_args()
    w = workloads.config2()
    assert w.n_orbits == 314 * 314 and w.n_steps == 100_000 and w.shadow_eps == 1e-8 and w.correction_mode == 3
    n = w.n_orbits
    sha = oracle_hash()
    if a.merge:
        return merge(a.out, n)
    lo, hi = max(0, a.lo), min(n, a.hi)
    part = f"{a.out}.part_{lo}_{hi}.npz"
    m = hi - lo
    fli, status = np.full(m, np.nan), np.zeros(m, np.int16)
    steps, gn = np.zeros(m, np.int32), np.zeros(m, np.int64)
    done, wall = 0, 0.0
    if os.path.exists(part):
        p = np.load(part)
        fli, status, steps, gn, done, wall = p["fli"], p["status"], p["steps"], p["gn_steps"], int(p["done"]), float(p["wall_s"])
        sha = str(p["oracle_sha256"])
        print(f"resuming {part} at {done} of {m}", flush=True)
    blk = a.rows_per_block * 314
    threads = a.threads or oracle.max_threads()
    while done < m:
        nxt = min(m, done + blk)
        sub = w.subset(np.arange(lo + done, lo + nxt))
        t0 = time.time()
        o = oracle.integrate(sub.states, w.h, w.n_steps, 3, shadow_eps=w.shadow_eps, n_threads=threads,
                             precision=oracle.LONG_DOUBLE, **sub.params())
        wall += time.time() - t0
        fli[done:nxt], status[done:nxt], steps[done:nxt], gn[done:nxt] = o.fli, o.status, o.steps_done, o.gn_steps
        done = nxt
        np.savez(part[:-4], fli=fli, status=status, steps=steps, gn_steps=gn, done=done, wall_s=wall, oracle_sha256=sha,
                 lo=lo, hi=hi, threads=threads)
        print(f"[{lo},{hi}): {done}/{m} orbits, {wall:.0f} s", flush=True)
    print("range complete:", part)
    if lo == 0 and hi == n:
        merge(a.out, n)


def merge(out, n):
    import glob
    parts = sorted(glob.glob(out + ".part_*.npz"), key=lambda f: int(f.split(".part_")[1].split("_")[0]))
    fli, status = np.full(n, np.nan), np.zeros(n, np.int16)
    steps, gn = np.zeros(n, np.int32), np.zeros(n, np.int64)
    covered = np.zeros(n, bool)
    wall, shas, how = 0.0, set(), []
    for f in parts:
        p = np.load(f)
        lo, d = int(p["lo"]), int(p["done"])
        sl = slice(lo, lo + d)
        fli[sl], status[sl], steps[sl], gn[sl] = p["fli"][:d], p["status"][:d], p["steps"][:d], p["gn_steps"][:d]
        covered[sl] = True
        wall += float(p["wall_s"])
        shas.add(str(p["oracle_sha256"]))
        how.append(f"[{lo},{lo + d}) {float(p['wall_s']):.0f} s on {int(p['threads'])} threads")
    if not covered.all():
        raise SystemExit(f"parts cover {covered.sum()} of {n} orbits; first missing orbit {int(np.argmin(covered))}")
    np.savez_compressed(out[:-4] if out.endswith(".npz") else out, fli=fli, status=status, steps=steps, gn_steps=gn,
                        oracle_sha256=" ".join(sorted(shas)), wall_s=wall, how="; ".join(how))
    print("wrote", out, "from", how)


if __name__ == "__main__":
    main()
