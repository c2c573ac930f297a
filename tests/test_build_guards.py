"""Build guards (ADVICE): a failed compile must never fall back to a stale libmc.so, and a
kernel that spills registers must stop the build (north_star: zero register spills).  CPU only."""
import os

import pytest

from paper_1802_00147_b200 import binding, build


def test_spill_report_flags_any_stack_frame_or_spill_of_a_kernel():
    log = open(os.path.join(build.OBJ, "ptxas.log")).read()
    assert log.count("Compiling entry function") >= 70 and build.spill_report(log) == []      # the library as built
    k = "_ZN2mc16integrate_kernelILi0ELb0ELi3ELi0ELb0ELi3EEEv8McConstsNS_13IntegrateArgsE"
    clean = ("ptxas info    : Function properties for %s\n    0 bytes stack frame, 0 bytes spill stores, 0 bytes spill loads\n" % k)
    for bad_line in ("    8 bytes stack frame, 0 bytes spill stores, 0 bytes spill loads",
                     "    0 bytes stack frame, 4 bytes spill stores, 0 bytes spill loads",
                     "    0 bytes stack frame, 0 bytes spill stores, 12 bytes spill loads"):
        doctored = clean + "ptxas info    : Function properties for %s\n%s\n" % (k.replace("Li3ELi0", "Li2ELi0"), bad_line)
        rep = build.spill_report(doctored)
        assert len(rep) == 1 and "Li2ELi0" in rep[0][0]
    # helper subroutines (slow paths of sqrt / division) may own a stack frame; only kernels count
    helper = "ptxas info    : Function properties for $__internal_0_$__cuda_sm20_dsqrt_rn_f64\n    16 bytes stack frame, 0 bytes spill stores, 0 bytes spill loads\n"
    assert build.spill_report(clean + helper) == []


def test_failed_build_never_falls_back_to_a_stale_library(monkeypatch):
    assert os.path.exists(build.LIB)
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.delenv("MC_LIBMC_PATH", raising=False)

    def compile_error(*a, **k):
        raise RuntimeError("nvcc failed on mc_kernel_mode3.cu: error: expected a ';'")
    monkeypatch.setattr(build, "build", compile_error)
    with pytest.raises(binding.MCLibraryError, match="could not be built"):
        binding.load_library()

    def no_nvcc(*a, **k):
        raise FileNotFoundError("nvcc")
    monkeypatch.setattr(build, "build", no_nvcc)
    monkeypatch.setattr(build, "sources_newer_than_library", lambda: True)
    with pytest.raises(binding.MCLibraryError, match="older than its sources"):
        binding.load_library()
    monkeypatch.setattr(build, "sources_newer_than_library", lambda: False)    # no nvcc, library up to date: usable
    assert binding.load_library() is not None
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setenv("MC_LIBMC_PATH", "/nonexistent/libmc.so")
    with pytest.raises(binding.MCLibraryError, match="cannot load"):
        binding.load_library()
