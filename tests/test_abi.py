"""CPU-only checks of the boundary: libmc.so builds/loads, exports every symbol include/mc.h declares,
struct layouts agree, argument validation runs before any CUDA call.  No compute here."""
import ctypes
import os
import re

import pytest

from paper_1802_00147_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mc.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mc_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = binding.load_library()
    names = declared_functions()
    assert names == sorted(binding.EXPORTS), names
    for n in names:
        assert hasattr(lib, n), n


def test_bench_instruments_are_a_library_of_their_own():
    """include/mc_bench.h (FP64 probes, flop model) is served by benchlib/libmc_bench.so; libmc.so, the product, exports
    none of it, and the product package does not import the bench package."""
    import benchlib
    src = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "mc_bench.h")).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(mc_[a-z0-9_]+)\s*\(", src)))
    assert names == sorted(benchlib.EXPORTS), names
    blib, lib = benchlib.load_library(), binding.load_library()
    for n in names:
        assert hasattr(blib, n), n
        assert not hasattr(lib, n), n
    pkg = os.path.join(ROOT, "paper_1802_00147_b200")
    for f in os.listdir(pkg):
        if f.endswith(".py"):
            assert "benchlib" not in open(os.path.join(pkg, f)).read(), f


def test_header_is_plain_c(tmp_path):
    """The boundary header must compile as C (no C++ types in the signatures)."""
    c = tmp_path / "t.c"
    c.write_text('#include "mc.h"\n#include "mc_bench.h"\nint main(void){ mc_params p; return (int)sizeof(p) * 0; }\n')
    import subprocess
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_params_default_and_struct_size_agree():
    p = binding.params_default()
    assert p.struct_size == ctypes.sizeof(binding.mc_params)
    assert p.terms == 15 and p.renorm_interval == 100 and p.newton_iters == 4
    assert p.newton_tol == 1e-10 and p.r_merge == 2.0 and p.r_escape == 1e4
    assert p.beta == p.chi1 == p.chi2 == p.kq1 == p.kq2 == 1.0


@pytest.mark.parametrize("field,value", [("struct_size", 8), ("terms", 64), ("beta", 0.0), ("beta", 1.5),
                                         ("chi1", -0.1), ("chi2", 1.01), ("renorm_interval", 0),
                                         ("newton_iters", 0), ("newton_iters", 17), ("r_escape", 1.0)])
def test_create_rejects_bad_params_before_touching_cuda(field, value):
    lib = binding.load_library()
    p = binding.params_default()
    setattr(p, field, value)
    h = ctypes.c_void_p()
    assert lib.mc_create(ctypes.byref(p), ctypes.byref(h)) == binding.MC_EINVAL
    assert not h.value


def test_null_arguments_are_einval():
    lib = binding.load_library()
    assert lib.mc_create(None, None) == binding.MC_EINVAL
    assert lib.mc_integrate(None, None, 1, 1.0, 1, 3, 0.0, None, None, None) == binding.MC_EINVAL
    assert lib.mc_destroy(None) == binding.MC_EINVAL
    assert lib.mc_params_default(None) == binding.MC_EINVAL
    assert lib.mc_strerror(binding.MC_EINVAL) == b"invalid argument"
    assert lib.mc_strerror(0) == b"ok"


def test_no_cpu_fallback_exists():
    """The product package must not reach the oracle (or any CPU implementation)."""
    pkg = os.path.join(ROOT, "paper_1802_00147_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "pn_oracle" not in text or f == "mc_math.cuh" or f.endswith(".cuh"), f


def test_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = binding.load_library()
    p = binding.params_default()
    h = ctypes.c_void_p()
    rc = lib.mc_create(ctypes.byref(p), ctypes.byref(h))
    assert rc in (binding.MC_ECUDA, binding.MC_EINVAL) and not h.value
