"""Executed instruction mix of the hot kernel's step loop, read from the SASS of the library that was just built.

    python -m benchlib.sass_mix            # table for integrate_kernel<uniform, QM off, mode 3, RK4>

Why: bench.py reports ALGORITHMIC flop (mc_flop_model).  The flop the device really executes are a little higher
(Newton refinements around the MUFU seeds, lanes idling through a neighbour's second Gauss-Newton step), and the
time the FP64 pipe needs for them follows an operand-bandwidth rule measured on B200 (mc_fp64_probe, DESIGN.md
section 10): a warp-wide FP64 instruction occupies the sub-partition's pipe 2 cycles, but an FMA whose three source
operands are three distinct vector registers, none of them served by the operand-reuse cache, takes 3.  This module
counts both from `cuobjdump -sass` of csrc/build/mc_kernel_mode3.o and predicts the kernel time from the rule; bench.py
prints the prediction beside the measurement (`roofline.executed`).  Sections are found by landmarks of the loop
(VOTE.ALL at its top, VOTE.ANY at the top of the Gauss-Newton loop, the two back edges); if a future kernel no longer
has them, analyse() returns None and bench.py says so.

Host-side text processing only: nothing here is on the product path.
"""
import json
import os
import re
import subprocess

from paper_1802_00147_b200 import build as _build

CYC_3RF, CYC_REUSE, CYC_PLAIN = 3.03, 2.19, 2.03      # cycles per warp instruction per sub-partition (mc_fp64_probe, B200)
_PAT = re.compile(r"/\*([0-9a-f]{4,})\*/\s+(@!?U?P\w+\s+)?([A-Z0-9_.]+)\s*([^;]*);")
_REG = re.compile(r"[-|~]*R(\d+)(\.reuse)?")
FP64_OPS = ("DFMA", "DMUL", "DADD", "DSETP")


def kernel_symbol(params=0, qm=False, mode=3, integ=0, rr=False, minb=None):
    if minb is None:
        minb = 2 if (params == 1 or integ == 1 or rr) else 3
    return "_ZN2mc16integrate_kernelILi%dELb%dELi%dELi%dELb%dELi%dEEEv8McConstsNS_13IntegrateArgsE" % (
        params, int(qm), mode, integ, int(rr), minb)


def disassemble(obj, symbol):
    """[(address, opcode, operand string)] of one function."""
    txt = subprocess.run(["cuobjdump", "-sass", obj], capture_output=True, text=True, check=True).stdout
    start = txt.find("Function : " + symbol)
    if start < 0:
        return []
    end = txt.find("Function : ", start + 10)
    ins = []
    for line in txt[start:end if end > 0 else None].splitlines():
        m = _PAT.search(line)
        if m:
            ins.append((int(m.group(1), 16), m.group(3), m.group(4)))
    return ins


def _sections(ins):
    tops = [a for a, op, _ in ins if op.startswith("VOTE.ALL")]
    gns = [a for a, op, _ in ins if op.startswith("VOTE.ANY")]
    if not tops or not gns:
        return None
    loop0, gn0 = tops[0], gns[0]
    gn1 = None
    for a, op, ar in ins:
        if a > gn0 and op.startswith("BRA"):
            m = re.search(r"0x([0-9a-f]+)", ar)
            if m and loop0 < int(m.group(1), 16) <= gn0:
                gn1 = a + 16
                break
    if gn1 is None:
        return None
    return loop0, gn0, gn1


def _count(ins, lo, hi):
    c = dict(DFMA=0, DMUL=0, DADD=0, DSETP=0, MUFU=0, all=0, dfma_3reg=0, dfma_reuse_hit=0, cycles=0.0)
    prev_reuse = set()
    for a, op, ar in ins:
        if not lo <= a < hi:
            continue
        o = op.split(".")[0]
        c["all"] += 1
        cur_reuse = set()
        if o == "MUFU":
            c["MUFU"] += 1
        if o in FP64_OPS:
            c[o] += 1
            srcs = [s.strip() for s in ar.split(",")]
            srcs = srcs[2:] if o == "DSETP" else srcs[1:]
            regs, hit = set(), False
            for slot, s in enumerate(srcs):
                m = _REG.match(s)
                if m and not re.match(r"[-|~]*RZ", s):
                    if (slot, m.group(1)) in prev_reuse:
                        hit = True
                    else:
                        regs.add(m.group(1))
                    if m.group(2):
                        cur_reuse.add((slot, m.group(1)))
            if len(regs) >= 3:
                c["dfma_3reg"] += 1
                c["cycles"] += CYC_3RF
            elif hit and o == "DFMA":
                c["dfma_reuse_hit"] += 1
                c["cycles"] += CYC_REUSE
            else:
                c["cycles"] += CYC_PLAIN
        prev_reuse = cur_reuse
    c["fp64"] = c["DFMA"] + c["DMUL"] + c["DADD"] + c["DSETP"]
    c["flop"] = 2 * c["DFMA"] + c["DMUL"] + c["DADD"]
    return c


def analyse(params=0, qm=False, mode=3, integ=0, rr=False, obj=None):
    """Per-section counts of the step loop, or None if the object / symbol / landmarks are missing."""
    obj = obj or os.path.join(_build.OBJ, "mc_kernel_mode%d.o" % mode)
    if not os.path.exists(obj):
        return None
    try:
        ins = disassemble(obj, kernel_symbol(params, qm, mode, integ, rr))
    except (OSError, subprocess.CalledProcessError):
        return None
    sec = _sections(ins) if ins else None
    if sec is None:
        return None
    loop0, gn0, gn1 = sec
    return {"kernel": kernel_symbol(params, qm, mode, integ, rr),
            "step_fixed": _count(ins, loop0, gn0),           # base integrator step + eq (10) + L_t
            "gn_iteration": _count(ins, gn0, gn1),           # one pass of the Gauss-Newton loop (executed per WARP)
            "tail": _count(ins, gn1, gn1 + 0x5a0),           # status test, accept, counters (common path)
            "cycle_rule": {"dfma_3_registers": CYC_3RF, "dfma_reuse_hit": CYC_REUSE, "other_fp64": CYC_PLAIN}}


def per_warp_step(mix, gn_iterations_per_warp_step, rule=None):
    """Executed FP64 instructions, flop (per lane) and model cycles of one warp-step.  `rule` = (cycles of a 3-register
    FMA, of an FMA with an operand-reuse hit, of any other FP64 instruction) as measured in the same run by mc_fp64_probe;
    without it the B200 figures frozen in this file (CYC_*) apply."""
    g = gn_iterations_per_warp_step
    out = {}
    for k in ("fp64", "flop", "cycles", "all", "DFMA", "DMUL", "DADD", "dfma_3reg", "dfma_reuse_hit"):
        out[k] = mix["step_fixed"][k] + g * mix["gn_iteration"][k] + mix["tail"][k]
    if rule is not None:
        c3, cr, cp = rule
        out["cycles"] = c3 * out["dfma_3reg"] + cr * out["dfma_reuse_hit"] + cp * (out["fp64"] - out["dfma_3reg"] - out["dfma_reuse_hit"])
    return out


def write_json(path=None):
    path = path or os.path.join(_build.OBJ, "sass_mix.json")
    mix = analyse()
    with open(path, "w") as f:
        json.dump(mix, f, indent=1)
    return path, mix


def main():
    mix = analyse()
    if mix is None:
        raise SystemExit("no SASS to analyse (build the library first)")
    print("| section | DFMA | DMUL | DADD | DSETP | FP64 instr | all instr | 3-register DFMA | reuse hits | flop | model cycles |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for name in ("step_fixed", "gn_iteration", "tail"):
        c = mix[name]
        print("| %s | %d | %d | %d | %d | %d | %d | %d | %d | %d | %.0f |" % (name, c["DFMA"], c["DMUL"], c["DADD"], c["DSETP"], c["fp64"],
                                                                           c["all"], c["dfma_3reg"], c["dfma_reuse_hit"], c["flop"], c["cycles"]))
    for g in (1.0, 1.18, 1.34):
        w = per_warp_step(mix, g)
        print("Gauss-Newton iterations per warp-step %.2f: %.0f FP64 instructions, %.0f flop per lane, %.0f model cycles "
              "(%.3f per FP64 instruction)" % (g, w["fp64"], w["flop"], w["cycles"], w["cycles"] / w["fp64"]))


if __name__ == "__main__":
    main()
