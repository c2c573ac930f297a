"""Build libmc.so (the C-ABI CUDA library of include/mc.h) in-tree with nvcc for sm_100a."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libmc.so")
LIB_CHECKED = os.path.join(HERE, "libmc_checked.so")     # -DMC_CHECKED: index / pointer tests before every global access
SOURCES = ["mc_api.cu", "mc_kernel_mode0.cu", "mc_kernel_mode1.cu", "mc_kernel_mode2.cu", "mc_kernel_mode3.cu",
           "mc_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _deps():
    out = [os.path.join(HERE, "..", "include", "mc.h")]
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def sources_newer_than_library() -> bool:
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _deps())


def is_stale() -> bool:
    return not os.path.exists(LIB) or sources_newer_than_library()


def spill_report(log: str):
    """(kernel, line) for every integrate_kernel / eval_kernel instantiation that ptxas -v reports with a stack frame
    or spill traffic.  north_star: zero register spills -- build() refuses to ship a library that has any."""
    bad, current = [], None
    for line in log.splitlines():
        if "Function properties for" in line:
            current = line.split("Function properties for")[1].strip()
        elif "bytes stack frame" in line and current is not None:
            nums = [int(x) for x in line.replace(",", " ").split() if x.isdigit()]
            if any(nums[:3]) and ("integrate_kernel" in current or "eval_kernel" in current):
                bad.append((current, line.strip()))
            current = None
    return bad


def build_checked(force: bool = False) -> str:
    """libmc_checked.so: the same sources with -DMC_CHECKED (mc_debug_check).  Used by the GPU tests only."""
    if not force and os.path.exists(LIB_CHECKED) and not any(os.path.getmtime(f) > os.path.getmtime(LIB_CHECKED) for f in _deps()):
        return LIB_CHECKED
    return build(force=True, checked=True)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    if not checked and not force and not is_stale():
        return LIB
    obj_dir = OBJ + ("_checked" if checked else "")
    os.makedirs(obj_dir, exist_ok=True)
    # one builder at a time: under torchrun every rank imports the binding, and if the library is stale they would
    # all compile into the same object files.  The others wait here and then find a fresh library.
    import fcntl
    with open(os.path.join(obj_dir, ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not checked and not force and not is_stale():
            return LIB
        return _build_locked(obj_dir, verbose, checked)


def _build_locked(obj_dir: str, verbose: bool, checked: bool) -> str:
    lib = LIB_CHECKED if checked else LIB
    flags = NVCC_FLAGS + (["-DMC_CHECKED"] if checked else [])
    nvcc = os.environ.get("NVCC", "nvcc")

    def compile_one(src):
        obj = os.path.join(obj_dir, os.path.splitext(src)[0] + ".o")
        r = subprocess.run([nvcc] + flags + ["-c", os.path.join(CSRC, src), "-o", obj],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        return obj, r.stderr

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    log = "".join(err for _, err in results)
    with open(os.path.join(obj_dir, "ptxas.log"), "w") as f:
        f.write(log)
    if verbose:
        print(log)
    bad = spill_report(log)
    if bad and not checked:                 # the checked build is a debugging aid: spills there are tolerated
        raise RuntimeError("register spills (north_star demands none):\n" + "\n".join(f"{k}: {l}" for k, l in bad))
    subprocess.run([nvcc, "-shared", "-Wno-deprecated-gpu-targets", "-o", lib + ".tmp"] + [o for o, _ in results] + ["-lcudart_static", "-ldl", "-lrt", "-lpthread"],
                   check=True)
    os.replace(lib + ".tmp", lib)
    if checked:
        return lib
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
