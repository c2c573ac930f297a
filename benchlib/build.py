"""Build benchlib/libmc_bench.so (include/mc_bench.h): the bench's instruments -- the DFMA peak probe, the operand-bandwidth
probe and the flop model.  Separate from libmc.so on purpose: none of this is part of the product boundary."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(ROOT, "paper_1802_00147_b200", "csrc")      # mc_flop_model.cpp instantiates the kernels' own math templates
LIB = os.path.join(HERE, "libmc_bench.so")
SOURCES = ["mc_bench.cu", "mc_flop_model.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo", "-Xcompiler", "-fPIC", "-I", CSRC]


def _deps():
    out = [os.path.join(HERE, s) for s in SOURCES] + [os.path.join(ROOT, "include", f) for f in ("mc.h", "mc_bench.h")]
    out += [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    return out


def is_stale() -> bool:
    return not os.path.exists(LIB) or any(os.path.getmtime(f) > os.path.getmtime(LIB) for f in _deps())


def build(force: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:      # under torchrun every rank may get here at once
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not is_stale():
            return LIB
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + ["-shared", "-Wno-deprecated-gpu-targets", "-o", LIB + ".tmp"] + \
              [os.path.join(HERE, s) for s in SOURCES] + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on benchlib:\n{r.stdout}\n{r.stderr}")
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
