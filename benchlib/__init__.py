"""Measurement instruments of bench.py (include/mc_bench.h, libmc_bench.so) -- not part of the product.

fp64_peak / fp64_probe measure the FP64 pipe of the device; flop_model counts the operations of the kernels' own
formulation with a counting scalar (host only); sass_mix reads the instruction mix of the built kernel.  bench.py and
the tests use them; paper_1802_00147_b200 does not import this package.
"""
import ctypes

from . import build as _build

MC_OK = 0
_lib = None


class mc_op_counts(ctypes.Structure):
    _fields_ = [("fma", ctypes.c_int64), ("mul", ctypes.c_int64), ("add", ctypes.c_int64), ("special", ctypes.c_int64)]


class mc_flop_model_t(ctypes.Structure):
    _fields_ = [(k, mc_op_counts) for k in ("rhs", "base_step", "correct_fixed", "gn_step", "status", "references", "renorm")]


EXPORTS = ["mc_fp64_peak", "mc_fp64_probe", "mc_flop_model"]     # every symbol include/mc_bench.h declares


def load_library():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        i32, dbl = ctypes.c_int32, ctypes.c_double
        lib.mc_fp64_peak.argtypes = [i32, dbl, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
        lib.mc_fp64_probe.argtypes = [i32, dbl, i32, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
        lib.mc_flop_model.argtypes = [ctypes.c_uint32, i32, i32, i32, ctypes.POINTER(mc_flop_model_t)]
        for name in EXPORTS:
            getattr(lib, name).restype = ctypes.c_int
        _lib = lib
    return _lib


def _check(rc, what):
    if rc != MC_OK:
        raise RuntimeError(f"libmc_bench: {what} failed with mc_error {rc}")


def fp64_peak(device: int = 0, millis: float = 200.0):
    """(TFLOP/s, implied SM clock in MHz) of the DFMA probe."""
    t, c = ctypes.c_double(), ctypes.c_double()
    _check(load_library().mc_fp64_peak(device, millis, ctypes.byref(t), ctypes.byref(c)), "mc_fp64_peak")
    return t.value, c.value


FP64_PROBE_KINDS = {0: "fma(y,z,x): 3 registers", 1: "fma(y,s,x): 2 registers + reused", 2: "fma(y,c[],x): 2 registers + constant",
                    3: "x*y: DMUL"}


def fp64_probe(device: int = 0, millis: float = 100.0) -> dict:
    """mc_fp64_probe for every kind: {kind name: (cycles per warp instruction per sub-partition, TFLOP/s)}."""
    out = {}
    for kind, name in FP64_PROBE_KINDS.items():
        c, t = ctypes.c_double(), ctypes.c_double()
        _check(load_library().mc_fp64_probe(device, millis, kind, ctypes.byref(c), ctypes.byref(t)), "mc_fp64_probe")
        out[name] = (c.value, t.value)
    return out


def flop_model(terms=15, correction_mode=3, integrator=0, newton_iters=4) -> dict:
    """mc_flop_model: operation counts of the kernels' own formulation, per trajectory (host-only, no GPU needed).
    Returns {part: {"fma", "mul", "add", "special", "flop"}} with flop = 2 fma + mul + add + special."""
    m = mc_flop_model_t()
    _check(load_library().mc_flop_model(int(terms), int(correction_mode), int(integrator), int(newton_iters), ctypes.byref(m)),
           "mc_flop_model")
    out = {}
    for part, _ in mc_flop_model_t._fields_:
        c = getattr(m, part)
        out[part] = dict(fma=c.fma, mul=c.mul, add=c.add, special=c.special, flop=2 * c.fma + c.mul + c.add + c.special)
    return out
