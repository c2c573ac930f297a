#!/usr/bin/env python
"""bench.py -- orbit-RK4-steps/s (with correction + FLI) on BASELINE config 2, and the FP64 roofline.

One "step" = one pass of the whole hot path (mc_integrate: load, 1e5 x [RK4 + six-integral correction]
on orbit and shadow, FLI renormalisation every 100 steps, status, store) over the 314 x 314 grid.
`value` counts accepted orbit-steps (dropped cells stop counting when they freeze).
N > 1 (torchrun): the global grid has 314*N rows of r0, dealt to the ranks round-robin (row i -> rank i mod N, so
every rank sees the same mix of strong- and weak-field cells), no collective on the data path (weak scaling).  `--impl reference` times the CPU oracle instead.
Prints ONE JSON line on rank 0.  See DESIGN.md section 8 for every number's definition.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1802_00147_b200 import sharding, workloads  # noqa: E402

METRIC = "orbit-RK4-steps/sec (with correction+FLI)"
UNIT = "orbit-steps/s"
# Algorithmic FP64 flops: NOT constants of this file.  They come from mc_flop_model (include/mc_bench.h, benchlib/), which runs the
# kernels' own math templates with a counting scalar on the host (FMA = 2, add/mul = 1, rsqrt/reciprocal/division/
# sqrt = 1; the Newton refinements around the hardware seeds are not algorithmic work) -- see algorithmic_flop()
# below and tests/test_flop_model.py.  The number of Gauss-Newton steps of mode 3 is data dependent (epsilon-
# terminated, R6): the kernel counts them (mc_get_work).
# DRAM traffic of ONE FULL-LENGTH launch (314 x 314 orbits + shadows, 1e5 steps) of the hot kernel:
# dram__bytes_read.sum + dram__bytes_write.sum from the ncu capture of that very launch configuration
# (profiles/r03_ncu_other_kernels.md, section "DRAM traffic of the full-length launch"; profiles/r03_traffic_full_length_launch.csv).  Outputs (31 MB) and the carry buffer (31 MB) live in the 126 MB L2;
# algorithmic: 340 B per orbit.
NCU_DRAM_BYTES_PER_LAUNCH_314 = 9861888 + 7502080   # read + write, bytes (round 3: profiles/r03_ncu_other_kernels.md, last section)
FP64_LANES_PER_SM = 64


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mc", choices=["mc", "reference"])
    ap.add_argument("--grid", type=int, default=314, help="grid edge (314 = BASELINE config 2)")
    ap.add_argument("--n-steps", type=int, default=None, help="RK4 steps per orbit (default: the workload's own; 1e5 for config 2)")
    ap.add_argument("--workload", default="config2",
                    help="config2 (default, the bench line) | config2:rr | config0 | config1 | config1:mode0 | config3 | config3:qmoff | "
                         "config4:<log2 n> | paper-theta2 | paper-theta2:0 | paper-plane  -- the other BASELINE configs and the "
                         "paper's own scans (PAPER.md:227), for profiles/ tables only")
    ap.add_argument("--integrator", default="rk4", choices=["rk4", "rk5"],
                    help="rk4 (BASELINE, default) | rk5 (Butcher six-stage, the paper's 'RK5'; profiles/ tables only)")
    ap.add_argument("--mode", type=int, default=None, choices=[0, 1, 2, 3],
                    help="correction mode override (default: the workload's own, 3 = six-integral projection; profiles/ tables only)")
    ap.add_argument("--sample-interval", type=int, default=0,
                    help="mc_integrate_sampled: record every orbit every K steps (profiles/ tables only; 0 = off)")
    ap.add_argument("--regroup", action="store_true",
                    help="mc_params.regroup: integrate the orbits in energy order (index mapping only; profiles/ tables only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1, config2 only: weak (default, the driver's contract) = 314 N rows, 314 per GPU; strong = the SAME "
                         "314 x 314 scan dealt row by row over the N GPUs (SURVEY 8e: n/G orbits per GPU)")
    ap.add_argument("--tabulate", default=None, metavar="FILE.jsonl",
                    help="no GPU work: print a markdown table of the bench lines in FILE.jsonl (profiles/ tables are made this way)")
    return ap.parse_args()


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU every 100 ms (NVML) while the timed region runs."""
    REASONS = {0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x10: "sync_boost",
               0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
               0x100: "display_clock_setting"}

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.mask, self.max_mhz, self.power = index, [], 0, None, []
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        while self.ok and not self._stop_evt.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                self.power.append(self.nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.1)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        reasons = [n for b, n in self.REASONS.items() if self.mask & b]
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "power_w_max": max(self.power) if self.power else None,
                "samples": len(self.samples)}


def algorithmic_flop(w, mode, integrator, steps_done, gn_steps):
    """Algorithmic FP64 flop of one launch from mc_flop_model (the kernels' own formulation, counted by a counting
    scalar) and the work the launch really did: accepted steps per orbit (`steps_done`), Gauss-Newton steps per
    orbit summed over orbit and shadow (`gn_steps`, mc_get_work).  A trajectory-step = base integrator step +
    the per-step part of the correction + status test; with a shadow every accepted orbit-step is two
    trajectory-steps and every renorm_interval-th step one renormalisation."""
    import benchlib
    m = benchlib.flop_model(w.terms, mode, integrator)
    traj = 2 if w.shadow_eps != 0.0 else 1
    steps_done = np.asarray(steps_done, dtype=np.int64)
    per_traj_step = m["base_step"]["flop"] + m["correct_fixed"]["flop"] + m["status"]["flop"]
    renorms = int((steps_done // w.renorm_interval).sum()) if traj == 2 else 0
    total = int(traj * steps_done.sum()) * per_traj_step + int(np.asarray(gn_steps).sum()) * m["gn_step"]["flop"] \
        + renorms * m["renorm"]["flop"]
    return {"flop_per_launch": int(total), "trajectories_per_orbit": traj,
            "model": {k: v["flop"] for k, v in m.items()},
            "model_ops": {k: {kk: v[kk] for kk in ("fma", "mul", "add", "special")} for k, v in m.items()},
            "per_trajectory_step_without_gn": per_traj_step}


def executed_from_sass(w, rk5, warp_work, per_launch_s, num_sms, sm_mhz, value, probe=None):
    """What the device executed in one launch, from the SASS instruction mix of the step loop (sass_mix.py, read from
    the library's own object file) times the warp-level work counters of the launch (mc_get_warp_work), and the time
    the FP64 pipe needs for it under the measured operand-bandwidth rule (3 cycles for an FMA with three distinct
    register operands, 2 otherwise; mc_fp64_probe).  None for kernels the SASS reader does not handle."""
    from benchlib import sass_mix
    if rk5 or w.correction_mode != 3 or (w.terms & 32) or not warp_work["warp_steps"]:
        return None
    params = 0 if w.uniform else (2 if (w.terms & 16 and len(set(w.beta)) == 1 and len(set(w.chi1)) == 1 and len(set(w.chi2)) == 1) else
                                  (0 if not (w.terms & 16) and len(set(w.beta)) == 1 and len(set(w.chi1)) == 1 and len(set(w.chi2)) == 1 else 1))
    mix = sass_mix.analyse(params=params, qm=bool(w.terms & 16))
    if mix is None:
        return None
    g = warp_work["gn_warp_passes"] / warp_work["warp_steps"]
    rule, rule_text = None, "3.03 cycles per FMA reading 3 distinct registers, 2.19 with an operand-reuse hit, 2.03 otherwise (frozen B200 figures)"
    if probe:                                   # the cycle rule as mc_fp64_probe measured it in THIS run
        kinds = benchlib_probe_kinds()
        rule = (probe[kinds[0]][0], probe[kinds[1]][0], max(probe[kinds[2]][0], probe[kinds[3]][0]))
        rule_text = ("%.2f cycles per FMA reading 3 distinct registers, %.2f with an operand-reuse hit, %.2f otherwise "
                     "(mc_fp64_probe, measured in this run)" % rule)
    per = sass_mix.per_warp_step(mix, g, rule)
    flop = per["flop"] * 32.0 * warp_work["warp_steps"]              # every lane slot of every executed warp instruction
    cycles = per["cycles"] * warp_work["warp_steps"] / (4.0 * num_sms)   # per sub-partition, perfectly balanced
    model_s = cycles / (sm_mhz * 1e6)
    return {"source": "SASS mix of the built library (benchlib/sass_mix.py) x mc_get_warp_work",
            "gn_passes_per_warp_step": g, "fp64_instr_per_warp_step": per["fp64"], "dfma_3_register_per_warp_step": per["dfma_3reg"],
            "dfma_share_of_fp64_instr": per["DFMA"] / per["fp64"], "executed_flop_per_launch": flop,
            "executed_tflops": flop / per_launch_s / 1e12,
            "operand_bandwidth_model": {"cycles_per_warp_step": per["cycles"], "kernel_ms": model_s * 1e3,
                                        "measured_over_model": per_launch_s / model_s,
                                        "rule": rule_text}}


def benchlib_probe_kinds():
    import benchlib
    return benchlib.FP64_PROBE_KINDS


def global_workload(args, world):
    """Config 2 widened to 314*world rows of r0 (same r0 range, same theta axis); the other configs are
    replicated per rank as they are."""
    name, _, opt = args.workload.partition(":")
    kw = {} if args.n_steps is None else {"n_steps": args.n_steps}
    if name == "config2":
        strong = getattr(args, "scaling", "weak") == "strong"
        w = workloads.config2(n_r=args.grid * (1 if strong else world), n_theta=args.grid, **kw)
        if opt == "rr":                             # the same scan with the 2.5PN radiation reaction (MC_TERM_RR)
            w.terms |= 32
        return w
    if name == "config0":
        return workloads.config0(**kw)
    if name == "config1":
        w = workloads.config1(**kw)
        if opt == "mode0":
            w.correction_mode = 0
        return w
    if name == "config3":
        return workloads.config3(qm=(opt != "qmoff"), **kw)
    if name == "config4":
        return workloads.config4(int(opt or 12), **kw)
    if name == "paper-theta2":                      # PAPER.md:227, Fig 6a (theta1 = pi/2) / 6b (paper-theta2:0)
        return workloads.paper_scan_theta2(theta1=(0.0 if opt == "0" else np.pi / 2), **kw)
    if name == "paper-plane":                       # PAPER.md:227, Fig 7
        return workloads.paper_scan_plane(**kw)
    raise SystemExit(f"unknown workload {args.workload}")


def rank_shard(w, args, rank, world):
    if args.workload.partition(":")[0] != "config2":
        return w
    if getattr(args, "scaling", "weak") == "strong":
        return sharding.strong_shard(w, args.grid, args.grid, rank, world)
    return sharding.rank_shard(w, args.grid, args.grid, rank, world)


def describe(w, args):
    integ = "RK5 (Butcher six-stage)" if args.integrator == "rk5" else "RK4"
    if w.name.startswith("config2"):
        per = "in total, rows dealt over the GPUs" if getattr(args, "scaling", "weak") == "strong" else "per GPU"
        return (f"config2: {args.grid}x{args.grid} orbit scan {per} (r0 in [10,60] x theta in [0,pi]), equal mass, chi=1, "
                f"N+1PN+2PN+SO+SS{'+2.5PN radiation reaction' if w.terms & 32 else ''}, {integ} h=1, {w.n_steps} steps, shadow 1e-8 renormalised every 100 steps + FLI, "
                + ("six-integral correction (mode 3, Gauss-Newton terminated at eps=1e-10, cap 4)" if w.correction_mode == 3
                   else f"correction mode {w.correction_mode}"))
    return (f"{args.workload} ({w.name}): {w.n_orbits} orbits per GPU, terms mask {w.terms}, "
            f"{'uniform' if w.uniform else 'per-orbit'} parameters, {integ} h={w.h}, {w.n_steps} steps, shadow {w.shadow_eps}, "
            f"correction mode {w.correction_mode}")


def cpu_baseline_sample(w, target_seconds=15.0):
    """Time the oracle (double instance, all host cores) on a strided sample of the workload."""
    import oracle
    cores = oracle.max_threads()
    n_probe = max(2 * cores, 16)
    idx = np.linspace(0, w.n_orbits - 1, n_probe).astype(int)
    sub = w.subset(idx)
    t0 = time.perf_counter()
    oracle.integrate(sub.states, w.h, 200, w.correction_mode, shadow_eps=w.shadow_eps, precision=oracle.DOUBLE,
                     **sub.params())
    rate = n_probe * 200 / (time.perf_counter() - t0)
    steps = int(min(w.n_steps, 20_000))
    n = int(max(cores, min(w.n_orbits, rate * target_seconds / steps)))
    n = max(cores, (n // cores) * cores)
    idx = np.linspace(0, w.n_orbits - 1, n).astype(int)
    sub = w.subset(idx)
    t0 = time.perf_counter()
    oracle.integrate(sub.states, w.h, steps, w.correction_mode, shadow_eps=w.shadow_eps, precision=oracle.DOUBLE,
                     **sub.params())
    dt = time.perf_counter() - t0
    return {"value": n * steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n} orbits strided over the grid x {steps} steps, double-precision instance of "
                      f"oracle/pn_oracle.hpp, OpenMP static, {dt:.1f} s"}, (n, steps)


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = global_workload(args, 1)
    base, (n, steps) = cpu_baseline_sample(w, target_seconds=8.0)
    import oracle
    idx = np.linspace(0, w.n_orbits - 1, n).astype(int)
    sub = w.subset(idx)
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.integrate(sub.states, w.h, steps, w.correction_mode, shadow_eps=w.shadow_eps,
                         precision=oracle.DOUBLE, **sub.params())
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = sum(times)
    value = n * steps * args.steps / total
    base["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config2: {args.grid}x{args.grid} orbit scan, RK4 h=1, shadow 1e-8 + FLI, "
                                   f"six-integral correction; each step = bounded sample ({n} orbits x {steps} steps)"},
            "cpu_baseline": base,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_mc(args):
    import torch
    import torch.distributed as dist
    from paper_1802_00147_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = rank_shard(global_workload(args, world), args, rank, world)
    if args.mode is not None:
        w.correction_mode = args.mode
    n = w.n_orbits
    orbit_steps_rank = float(n) * w.n_steps
    z_dev = torch.as_tensor(w.states, device=dev)
    z_pin = torch.as_tensor(w.states).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    import benchlib
    peak_tf, peak_clock = benchlib.fp64_peak(local, 200.0) if rank == 0 else (None, None)
    probe = benchlib.fp64_probe(local, 50.0) if rank == 0 else None      # operand-bandwidth rule of the FP64 pipe, measured here
    if w.uniform:
        par = dict(beta=float(w.beta[0]), chi1=float(w.chi1[0]), chi2=float(w.chi2[0]), kq1=float(w.kq1[0]), kq2=float(w.kq2[0]))
    else:
        par = {k: v for k, v in w.params().items() if k != "terms"}
    rk5 = args.integrator == "rk5"
    I = binding.Integrator(terms=w.terms, device=local, integrator=int(rk5), regroup=int(args.regroup), **par)
    out = torch.empty_like(z_dev)
    stream = torch.cuda.current_stream(dev)
    launches = 0

    def one_step():
        nonlocal launches
        res = I.integrate(z_dev, w.h, w.n_steps, w.correction_mode, shadow_eps=w.shadow_eps, out_states=out,
                          sample_interval=args.sample_interval)
        launches += 1
        return res

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches = 0
    barrier()
    t_wall0 = time.perf_counter()
    res = None
    for k in range(args.steps):
        flush.zero_()                                   # flush L2 between timed iterations
        ev[k][0].record(stream)
        res = one_step()
        ev[k][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    kernel_ms = [a.elapsed_time(b) for a, b in ev]
    dev_ms = float(sum(kernel_ms))
    dev_ms_max = sharding.max_over_ranks(dev_ms, dev)

    # end to end through the C ABI with HOST buffers (pinned): H2D + kernel + D2H inside the timed call
    z_host = z_pin.numpy()
    I.integrate_host(z_host, w.h, min(w.n_steps, 100), w.correction_mode, shadow_eps=w.shadow_eps)   # warm scratch
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        hres = I.integrate_host(z_host, w.h, w.n_steps, w.correction_mode, shadow_eps=w.shadow_eps)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s_max = sharding.max_over_ranks(e2e_s, dev)
    h2d = 12 * 8 * n
    d2h = (12 + 12 + 1) * 8 * n + 4 * n + 8 * n

    info = I.launch_info()
    status = res.status.cpu().numpy()
    fli = res.fli.cpu().numpy() if res.fli is not None else np.zeros(n)
    warp_work = I.warp_work()                                 # what the warps executed in the last timed launch
    steps_done_per_orbit = res.steps_done.cpu().numpy()
    gn_per_orbit = I.work(n).cpu().numpy()
    steps_done = float(steps_done_per_orbit.sum())            # accepted orbit-steps of one launch (this rank)
    gn_steps = float(gn_per_orbit.sum())                      # Gauss-Newton steps of one launch, orbit + shadow
    steps_done_job = sharding.sum_over_ranks(steps_done, dev)
    scheduled_job = sharding.sum_over_ranks(orbit_steps_rank, dev)
    # orbit-steps actually integrated (dropped cells stop counting when they freeze), whole job
    value = steps_done_job * args.steps / (dev_ms_max * 1e-3)
    e2e_value = steps_done_job * args.steps / e2e_s_max
    I.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    st = status & 255                                     # bit 8 = mode-2 skip flag, not a drop
    mp = measured_peaks()
    sm_max = float(mp.get("sm_max_mhz", clocks.get("sm_max_mhz") or 1965.0))
    nominal_tf = info["num_sms"] * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    per_launch_s = (dev_ms / args.steps) * 1e-3
    alg = algorithmic_flop(w, w.correction_mode, int(rk5), steps_done_per_orbit, gn_per_orbit)
    flop_per_launch = float(alg["flop_per_launch"])
    traj = alg["trajectories_per_orbit"]
    achieved_tf = flop_per_launch / per_launch_s / 1e12
    executed = executed_from_sass(w, rk5, warp_work, per_launch_s, info["num_sms"], sm_max, value, probe)
    roofline = {"bound": "alu", "achieved": achieved_tf, "peak": nominal_tf, "unit": "TFLOP/s",
                "frac": achieved_tf / nominal_tf,
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH_314 if (w.name.startswith("config2") and args.grid == 314 and world == 1) else None,
                "traffic_unit": "bytes per launch: dram__bytes_read.sum + dram__bytes_write.sum of one full-length (1e5-step) launch of "
                                "this kernel and grid under ncu (profiles/r03_ncu_other_kernels.md, r03_traffic_full_length_launch.csv); not re-measured in this run",
                "algorithmic_bytes_per_launch": 340.0 * n,
                "peak_source": f"derived: {info['num_sms']} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 x {sm_max:.0f} MHz "
                               "(MEASURED_PEAKS.json has no FP64 entry)",
                "peak_measured_dfma": peak_tf, "frac_of_measured_dfma": achieved_tf / peak_tf if peak_tf else None,
                "dfma_probe_implied_sm_mhz": peak_clock,
                "fp64_operand_probe": {k: {"cycles_per_warp_instr": v[0], "tflops": v[1]} for k, v in probe.items()} if probe else None,
                "flop_per_launch": flop_per_launch, "flop_per_orbit_step": flop_per_launch / max(steps_done, 1.0),
                "flop_model": alg["model"], "flop_model_ops": alg["model_ops"],
                "flop_source": "mc_flop_model: the kernels' math templates run with a counting scalar (tests/test_flop_model.py)",
                # continuity with BENCH_r01 (config 2, RK4, mode 3, QM off only): round 1's frozen hand count, 2270 per orbit-step +
                # 390 per Gauss-Newton step, counted the rsqrt / reciprocal refinements as algorithmic work
                "frac_with_round1_hand_count": ((2270.0 * steps_done + 390.0 * gn_steps) / per_launch_s / 1e12 / nominal_tf
                                                if (traj == 2 and w.correction_mode == 3 and not rk5 and not (w.terms & 48)) else None),
                "gn_steps_per_trajectory_step": gn_steps / max(traj * steps_done, 1.0),
                "executed": executed,
                "accepted_orbit_steps_per_launch": steps_done, "kernel": "mc::integrate_kernel<%s,QM %s,mode %d,%s%s>" % (
                    "per-orbit" if info["variant"] & 1 else ("per-orbit kappa" if info["variant"] & 4 else "uniform"),
                    "on" if info["variant"] & 2 else "off", (info["variant"] >> 4) & 3, "RK5" if info["variant"] & 256 else "RK4",
                    ",2.5PN" if info["variant"] & 8 else ""),
                "kernel_ms_per_launch": dev_ms / args.steps,
                "regs_per_thread": info["regs_per_thread"], "spill_bytes": info["local_bytes"],
                "blocks_per_sm": info["blocks_per_sm"], "grid": info["grid"], "block": info["block"]}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True,
            "scaling": args.scaling if w.name.startswith("config2") else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": describe(w, args),
                       "orbits_per_gpu": n, "rk4_steps": w.n_steps, "sample_interval": args.sample_interval,
                       "sample_bytes_per_launch": (w.n_steps // args.sample_interval) * 96 * n if args.sample_interval else 0,
                       "orbit_steps_counted": "accepted steps (sum of steps_done); scheduled = orbits x rk4_steps = %d" % int(orbit_steps_rank * world), "l2": "flushed (256 MiB write) between timed iterations",
                       "regroup": bool(args.regroup),
                       "parallelism": f"orbit-sharded x{world} (grid rows round-robin over ranks; {args.scaling} scaling), no collective"},
            "clocks": clocks, "wall_s_timed_region": t_wall,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": launches, "roofline": roofline,
            "outcome": {"regular": int(((st == 0) & (fli < 5.8)).sum()), "chaotic": int(((st == 0) & (fli >= 5.8)).sum()),
                        "dropped": int((st != 0).sum()), "near_threshold": int(((st == 0) & (np.abs(fli - 5.8) < 0.5)).sum()),
                        "mode2_skip_flagged": int(((status & 256) != 0).sum())}}
    if not args.no_cpu_baseline and world == 1:           # rank 0 at N = 1 only (contract)
        line["cpu_baseline"], _ = cpu_baseline_sample(w)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


TABLE_COLUMNS = [("workload", lambda l: l["config"]["workload"].split(": ")[0] + (" regroup" if l["config"].get("regroup") else "")),
                 ("kernel", lambda l: l["roofline"]["kernel"].replace("mc::integrate_kernel", "")),
                 ("orbits per GPU", lambda l: l["config"]["orbits_per_gpu"]),
                 ("steps", lambda l: l["config"]["rk4_steps"]),
                 ("orbit-steps/s", lambda l: "%.3e" % l["value"]),
                 ("ms per launch", lambda l: "%.1f" % l["ms_per_step"]),
                 ("TFLOP/s", lambda l: "%.2f" % l["roofline"]["achieved"]),
                 ("frac", lambda l: "%.3f" % l["roofline"]["frac"]),
                 ("regs", lambda l: l["roofline"]["regs_per_thread"]),
                 ("spill B", lambda l: l["roofline"]["spill_bytes"]),
                 ("blocks/SM", lambda l: l["roofline"]["blocks_per_sm"]),
                 ("grid", lambda l: l["roofline"]["grid"]),
                 ("GN steps per lane-step", lambda l: "%.3f" % l["roofline"]["gn_steps_per_trajectory_step"]),
                 ("regular / chaotic / dropped", lambda l: "%d / %d / %d" % (l["outcome"]["regular"], l["outcome"]["chaotic"], l["outcome"]["dropped"])),
                 ("SM MHz (median / max)", lambda l: "%s / %s" % (l["clocks"]["sm_mhz"], l["clocks"]["sm_max_mhz"])),
                 ("throttle reasons", lambda l: ", ".join(l["clocks"]["reasons"]) or "none"),
                 ("power W max", lambda l: l["clocks"]["power_w_max"])]


def tabulate(path):
    """Markdown table of the bench lines in a .jsonl file: one row per line, the clock record of the run beside its number."""
    lines = [json.loads(t) for t in open(path) if t.strip().startswith("{")]
    print("| " + " | ".join(name for name, _ in TABLE_COLUMNS) + " |")
    print("|" + "---|" * len(TABLE_COLUMNS))
    for l in lines:
        print("| " + " | ".join(str(fn(l)) for _, fn in TABLE_COLUMNS) + " |")


def main():
    args = parse_args()
    if args.tabulate:
        return tabulate(args.tabulate)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mc(args)


if __name__ == "__main__":
    main()
