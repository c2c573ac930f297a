"""Thin Python binding of libmc.so (include/mc.h): argument marshalling only.

torch is used for device memory and streams; every step of the path runs in the CUDA kernels behind
the C ABI.  There is no CPU fallback: if the library cannot be loaded or built, import of the symbols
fails loudly (MCLibraryError).
"""
import ctypes
import os
from dataclasses import dataclass
from typing import Optional

from . import build as _build

MC_TERM_1PN, MC_TERM_2PN, MC_TERM_SO, MC_TERM_S1S2, MC_TERM_QM, MC_TERM_RR = 1, 2, 4, 8, 16, 32
TERMS_DEFAULT = MC_TERM_1PN | MC_TERM_2PN | MC_TERM_SO | MC_TERM_S1S2
MC_OK, MC_EINVAL, MC_ECUDA, MC_EARCH, MC_ENOMEM, MC_ELIMIT = 0, -1, -2, -3, -4, -5
MC_STATIC_MAX_TRAJECTORIES = 32768   # include/mc.h: the fixed scratch of mc_integrate_static
MC_INTEG_RK4, MC_INTEG_RK5 = 0, 1

# every symbol include/mc.h declares (tests/test_abi.py checks the header against this list)
EXPORTS = ["mc_params_default", "mc_create", "mc_integrate", "mc_integrate_sampled", "mc_integrate_ex", "mc_carry_bytes", "mc_integrate_host", "mc_integrate_static", "mc_get_status", "mc_get_work", "mc_get_warp_work", "mc_get_dissipation", "mc_debug_check", "mc_eval",
           "mc_last_launch_info", "mc_destroy", "mc_strerror"]


class MCLibraryError(RuntimeError):
    pass


class MCError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libmc error {code}: {msg}")
        self.code = code


class mc_params(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("terms", ctypes.c_uint32), ("device", ctypes.c_int32),
                ("per_orbit", ctypes.c_int32), ("beta", ctypes.c_double), ("chi1", ctypes.c_double),
                ("chi2", ctypes.c_double), ("kq1", ctypes.c_double), ("kq2", ctypes.c_double),
                ("d_beta", ctypes.c_void_p), ("d_chi1", ctypes.c_void_p), ("d_chi2", ctypes.c_void_p),
                ("d_kq1", ctypes.c_void_p), ("d_kq2", ctypes.c_void_p), ("renorm_interval", ctypes.c_int32),
                ("newton_iters", ctypes.c_int32), ("newton_tol", ctypes.c_double), ("r_merge", ctypes.c_double),
                ("r_escape", ctypes.c_double), ("cuda_stream", ctypes.c_void_p), ("chunk_steps", ctypes.c_int32), ("integrator", ctypes.c_int32),
                ("wait_budget_s", ctypes.c_double), ("regroup", ctypes.c_int32), ("reserved_", ctypes.c_int32)]


class mc_launch_info(ctypes.Structure):
    _fields_ = [("grid", ctypes.c_int32), ("block", ctypes.c_int32), ("regs_per_thread", ctypes.c_int32),
                ("local_bytes", ctypes.c_int32), ("blocks_per_sm", ctypes.c_int32), ("num_sms", ctypes.c_int32),
                ("smem_bytes", ctypes.c_int32), ("variant", ctypes.c_int32), ("trajectories", ctypes.c_int64),
                ("chunk_steps", ctypes.c_int32), ("n_chunks", ctypes.c_int32)]


_lib = None


def library_path() -> str:
    return _build.LIB


def load_library():
    """dlopen libmc.so (building it with nvcc first if it is missing or stale). Never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    path = os.environ.get("MC_LIBMC_PATH")      # a prebuilt libmc.so (e.g. a box without nvcc) instead of building in-tree
    if not path:
        try:
            path = _build.build()
        except FileNotFoundError as e:           # no nvcc on this box: an existing library is all there can be
            if os.path.exists(_build.LIB) and not _build.sources_newer_than_library():
                path = _build.LIB
            else:
                raise MCLibraryError(f"libmc.so is missing or older than its sources and nvcc is not available: {e}") from e
        except Exception as e:                   # nvcc ran and failed: never fall back to a stale binary
            raise MCLibraryError(f"libmc.so could not be built from the current sources: {e}") from e
    try:
        lib = ctypes.CDLL(path)
    except OSError as e:
        raise MCLibraryError(f"cannot load {path}: {e}") from e
    vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    lib.mc_params_default.argtypes = [ctypes.POINTER(mc_params)]
    lib.mc_create.argtypes = [ctypes.POINTER(mc_params), ctypes.POINTER(vp)]
    lib.mc_integrate.argtypes = [vp, vp, i64, dbl, i64, i32, dbl, vp, vp, vp]
    lib.mc_integrate_sampled.argtypes = [vp, vp, i64, dbl, i64, i32, dbl, vp, vp, vp, i64, vp]
    lib.mc_integrate_ex.argtypes = [vp, vp, i64, dbl, i64, i32, dbl, vp, vp, vp, vp, i32]
    lib.mc_carry_bytes.argtypes = [i64, i32]
    lib.mc_integrate_host.argtypes = [vp, vp, i64, dbl, i64, i32, dbl, vp, vp, vp, vp, vp]
    lib.mc_integrate_static.argtypes = [ctypes.POINTER(mc_params), vp, i64, dbl, i64, i32, dbl, vp, vp, vp, vp, vp]
    lib.mc_get_status.argtypes = [vp, vp, vp]
    lib.mc_get_work.argtypes = [vp, vp]
    lib.mc_get_dissipation.argtypes = [vp, vp]
    lib.mc_get_warp_work.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
    lib.mc_debug_check.argtypes = [vp, ctypes.POINTER(ctypes.c_int64)]
    lib.mc_eval.argtypes = [vp, i32, vp, i64, dbl, i32, vp, vp]
    lib.mc_last_launch_info.argtypes = [vp, ctypes.POINTER(mc_launch_info)]
    lib.mc_destroy.argtypes = [vp]
    lib.mc_strerror.argtypes = [ctypes.c_int]
    lib.mc_strerror.restype = ctypes.c_char_p
    for name in EXPORTS:
        if name not in ("mc_strerror", "mc_carry_bytes"):
            getattr(lib, name).restype = ctypes.c_int
    lib.mc_carry_bytes.restype = ctypes.c_int64
    _lib = lib
    return lib


def _check(rc):
    if rc != MC_OK:
        raise MCError(rc, load_library().mc_strerror(rc).decode())


def params_default() -> mc_params:
    p = mc_params()
    _check(load_library().mc_params_default(ctypes.byref(p)))
    return p


@dataclass
class IntegrateResult:
    states: "object"                 # torch.Tensor (12, n) float64, device
    invariants: Optional["object"]   # (12, n) or None
    fli: Optional["object"]          # (n,) or None
    status: "object"                 # (n,) int32
    steps_done: "object"             # (n,) int64
    samples: Optional["object"] = None   # (n_steps // sample_interval, 12, n) with sample_interval > 0
    carry: Optional["object"] = None     # checkpoint buffer of integrate_ex


class Integrator:
    """mc_create / mc_integrate / mc_destroy with torch tensors as device buffers."""

    def __init__(self, terms=TERMS_DEFAULT, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0, device=0,
                 renorm_interval=100, newton_iters=4, newton_tol=1e-10, r_merge=2.0, r_escape=1e4, stream=None,
                 chunk_steps=0, integrator=0, wait_budget_s=600.0, per_orbit=None, regroup=0):
        import torch
        self._torch = torch
        self._lib = load_library()
        p = params_default()
        p.terms, p.device = int(terms), int(device)
        p.renorm_interval, p.newton_iters, p.newton_tol = int(renorm_interval), int(newton_iters), float(newton_tol)
        p.r_merge, p.r_escape = float(r_merge), float(r_escape)
        p.chunk_steps = int(chunk_steps)
        p.integrator = int(integrator)
        p.wait_budget_s = float(wait_budget_s)
        p.regroup = int(regroup)
        self.device = torch.device("cuda", device)
        vals = dict(beta=beta, chi1=chi1, chi2=chi2, kq1=kq1, kq2=kq2)

        def uniform_value(v):
            """The scalar all orbits share, or None if the parameter really varies."""
            if not hasattr(v, "__len__"):
                return float(v)
            if isinstance(v, torch.Tensor):          # device tensors stay where they are: tested with torch, no host copy of the array
                t = v.detach().reshape(-1)
                return float(t[0]) if t.numel() and bool((t == t[0]).all()) else None
            import numpy as np
            a = np.asarray(v, dtype=np.float64)
            return float(a.flat[0]) if a.size and (a == a.flat[0]).all() else None

        uni = {k: uniform_value(v) for k, v in vals.items()}
        self._keep = []
        self.n_params = None
        arrays = [k for k, u in uni.items() if u is None]
        if per_orbit == 1:                               # forced: every parameter as a device array (tests)
            arrays = [k for k, v in vals.items() if hasattr(v, "__len__")] + ["beta"]
            uni = {k: None for k in vals}
        if not arrays:                                   # mc_params.per_orbit = 0
            for name, u in uni.items():
                setattr(p, name, u)
        elif set(arrays) <= {"kq1", "kq2"}:              # per_orbit = 2: one binary model, per-orbit quadrupole coefficients
            self.n_params = max(len(vals[k]) for k in arrays)
            p.per_orbit = 2
            for name in ("beta", "chi1", "chi2"):
                setattr(p, name, uni[name])
            for name in ("kq1", "kq2"):
                t = torch.as_tensor(vals[name], dtype=torch.float64).expand(self.n_params).contiguous().to(self.device)
                self._keep.append(t)                     # must outlive the handle (include/mc.h)
                setattr(p, "d_" + name, t.data_ptr())
        else:                                            # per_orbit = 1
            n = max([len(v) for v in vals.values() if hasattr(v, "__len__")] + [1])
            self.n_params = n
            p.per_orbit = 1
            for name, v in vals.items():
                t = torch.as_tensor(v, dtype=torch.float64).expand(n).contiguous().to(self.device)
                self._keep.append(t)            # must outlive the handle (include/mc.h)
                setattr(p, "d_" + name, t.data_ptr())
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        p.cuda_stream = stream.cuda_stream
        self.params = p
        self._h = ctypes.c_void_p()
        _check(self._lib.mc_create(ctypes.byref(p), ctypes.byref(self._h)))

    def close(self):
        h = getattr(self, "_h", None)
        if h is not None and h.value:
            self._h = None                     # before the call: safe against re-entry and interpreter shutdown
            self._lib.mc_destroy(h)

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _dev(self, x):
        torch = self._torch
        t = torch.as_tensor(x, dtype=torch.float64)
        if t.device != self.device:
            t = t.to(self.device)
        return t.contiguous()

    def integrate(self, states, h, n_steps, correction_mode=3, shadow_eps=0.0, want_invariants=True,
                  out_states=None, sample_interval=0) -> IntegrateResult:
        """states: (12, n) float64 (device tensor, or anything torch.as_tensor accepts)."""
        torch = self._torch
        z = self._dev(states)
        assert z.dim() == 2 and z.shape[0] == 12, z.shape
        n = z.shape[1]
        if self.n_params is not None and n > self.n_params:
            raise ValueError("more orbits than per-orbit parameters")
        out = torch.empty_like(z) if out_states is None else out_states
        inv = torch.empty_like(z) if want_invariants else None
        fli = torch.empty(n, dtype=torch.float64, device=self.device) if shadow_eps != 0.0 else None
        samples = None
        if sample_interval > 0:
            samples = torch.empty((int(n_steps) // int(sample_interval), 12, n), dtype=torch.float64, device=self.device)
        _check(self._lib.mc_integrate_sampled(self._h, z.data_ptr(), n, float(h), int(n_steps), int(correction_mode),
                                              float(shadow_eps), out.data_ptr(),
                                              inv.data_ptr() if inv is not None else None,
                                              fli.data_ptr() if fli is not None else None, int(sample_interval),
                                              samples.data_ptr() if samples is not None else None))
        status = torch.empty(n, dtype=torch.int32, device=self.device)
        steps = torch.empty(n, dtype=torch.int64, device=self.device)
        _check(self._lib.mc_get_status(self._h, status.data_ptr(), steps.data_ptr()))
        return IntegrateResult(out, inv, fli, status, steps, samples)

    def integrate_ex(self, states, h, n_steps, correction_mode=3, shadow_eps=0.0, carry=None, resume=False,
                     n_orbits=None, invariants=None) -> IntegrateResult:
        """mc_integrate_ex: checkpoint / resume.  First call: carry=None allocates the checkpoint buffer (returned
        as result.carry); later calls pass it back with resume=True (states may then be None)."""
        torch = self._torch
        if resume:
            n = int(n_orbits)
            zptr = None
        else:
            z = self._dev(states)
            n = z.shape[1]
            zptr = z.data_ptr()
        if carry is None:
            nbytes = self._lib.mc_carry_bytes(n, int(shadow_eps != 0.0))
            carry = torch.empty(max(nbytes, 8) // 8, dtype=torch.float64, device=self.device)
        out = torch.empty((12, n), dtype=torch.float64, device=self.device)
        inv = invariants if invariants is not None else torch.empty((12, n), dtype=torch.float64, device=self.device)
        fli = torch.empty(n, dtype=torch.float64, device=self.device) if shadow_eps != 0.0 else None
        _check(self._lib.mc_integrate_ex(self._h, zptr, n, float(h), int(n_steps), int(correction_mode), float(shadow_eps),
                                         out.data_ptr(), inv.data_ptr(), fli.data_ptr() if fli is not None else None,
                                         carry.data_ptr(), int(bool(resume))))
        status = torch.empty(n, dtype=torch.int32, device=self.device)
        steps = torch.empty(n, dtype=torch.int64, device=self.device)
        _check(self._lib.mc_get_status(self._h, status.data_ptr(), steps.data_ptr()))
        res = IntegrateResult(out, inv, fli, status, steps)
        res.carry = carry
        return res

    def integrate_host(self, states_np, h, n_steps, correction_mode=3, shadow_eps=0.0):
        """mc_integrate_host: numpy (host) in, numpy out; copies are inside the call."""
        import numpy as np
        z = np.ascontiguousarray(states_np, dtype=np.float64)
        n = z.shape[1]
        out, inv = np.empty_like(z), np.empty_like(z)
        fli = np.empty(n) if shadow_eps != 0.0 else None
        status, steps = np.empty(n, dtype=np.int32), np.empty(n, dtype=np.int64)
        _check(self._lib.mc_integrate_host(self._h, z.ctypes.data, n, float(h), int(n_steps), int(correction_mode),
                                           float(shadow_eps), out.ctypes.data, inv.ctypes.data,
                                           fli.ctypes.data if fli is not None else None, status.ctypes.data,
                                           steps.ctypes.data))
        return IntegrateResult(out, inv, fli, status, steps)

    def integrate_static(self, states, h, n_steps, correction_mode=3, shadow_eps=0.0, out=None) -> IntegrateResult:
        """mc_integrate_static: the same integration for callers that must not allocate device memory (a process whose
        own pool owns the whole GPU, a latency-bound loop that cannot afford cudaMalloc's stall, code running while a
        stream is being captured).  The library keeps its bookkeeping in a fixed array inside libmc.so instead of
        cudaMalloc'ed handle buffers, so the batch is limited to MC_STATIC_MAX_TRAJECTORIES trajectories (orbits, or
        2 x orbits with a shadow; MCError with code MC_ELIMIT beyond that) and calls on different streams must not
        overlap.  It takes this Integrator's parameters but not its handle.

        `states` must already be a contiguous float64 device tensor (12, n) -- converting it would allocate.  `out`,
        an IntegrateResult of preallocated device tensors (states, invariants or None, fli if shadow_eps != 0, status
        int32, steps_done int64), receives the outputs; without it this wrapper allocates them through torch, which
        is fine for a test and defeats the purpose in production."""
        torch = self._torch
        z = states
        if not (isinstance(z, torch.Tensor) and z.device == self.device and z.dtype == torch.float64 and z.is_contiguous()
                and z.dim() == 2 and z.shape[0] == 12):
            raise ValueError("integrate_static needs a contiguous float64 (12, n) tensor on the integrator's device")
        n = z.shape[1]
        if self.n_params is not None and n > self.n_params:
            raise ValueError("more orbits than per-orbit parameters")
        if out is None:
            out = IntegrateResult(torch.empty_like(z), torch.empty_like(z),
                                  torch.empty(n, dtype=torch.float64, device=self.device) if shadow_eps != 0.0 else None,
                                  torch.empty(n, dtype=torch.int32, device=self.device),
                                  torch.empty(n, dtype=torch.int64, device=self.device))
        _check(self._lib.mc_integrate_static(ctypes.byref(self.params), z.data_ptr(), n, float(h), int(n_steps),
                                             int(correction_mode), float(shadow_eps), out.states.data_ptr(),
                                             out.invariants.data_ptr() if out.invariants is not None else None,
                                             out.fli.data_ptr() if out.fli is not None else None,
                                             out.status.data_ptr(), out.steps_done.data_ptr()))
        return out

    _WHAT = {"H": (0, 1), "rhs": (1, 12), "integrals": (2, 6), "rk4_step": (3, 12), "correct": (4, 12)}

    def eval(self, what, states, h=0.0, mode=0, refs=None):
        """mc_eval: what in {"H","rhs","integrals","rk4_step","correct"} -> tensor (rows, n)."""
        torch = self._torch
        z = self._dev(states)
        n = z.shape[1]
        code, rows = self._WHAT[what]
        if (self.params.terms & MC_TERM_RR) and what in ("rhs", "rk4_step"):
            rows = 16                                   # + the dissipation integrals / their rates (include/mc.h)
        out = torch.empty((rows, n), dtype=torch.float64, device=self.device)
        r = self._dev(refs) if refs is not None else None
        _check(self._lib.mc_eval(self._h, code, z.data_ptr(), n, float(h), int(mode),
                                 r.data_ptr() if r is not None else None, out.data_ptr()))
        return out

    def work(self, n):
        """mc_get_work: Gauss-Newton steps per orbit (orbit + shadow) of the last integrate -> int64 tensor (n,)."""
        torch = self._torch
        out = torch.empty(n, dtype=torch.int64, device=self.device)
        _check(self._lib.mc_get_work(self._h, out.data_ptr()))
        return out

    def warp_work(self) -> dict:
        """mc_get_warp_work: Gauss-Newton loop passes counted per warp and warp-steps of the last integrate."""
        out = (ctypes.c_int64 * 2)()
        _check(self._lib.mc_get_warp_work(self._h, out))
        return {"gn_warp_passes": int(out[0]), "warp_steps": int(out[1])}

    def debug_check(self) -> int:
        """mc_debug_check: -1 for the product library; checked build: 0 = clean, else the source line of the failed test."""
        out = ctypes.c_int64()
        _check(self._lib.mc_debug_check(self._h, ctypes.byref(out)))
        return int(out.value)

    def dissipation(self, n):
        """mc_get_dissipation: the moving references E0 + W, J0 + G per orbit at the end of the last integrate (handle
        created with MC_TERM_RR) -> (4, n); subtract rows 0-3 of the invariants to get W, G."""
        torch = self._torch
        out = torch.empty((4, n), dtype=torch.float64, device=self.device)
        _check(self._lib.mc_get_dissipation(self._h, out.data_ptr()))
        return out

    def launch_info(self) -> dict:
        info = mc_launch_info()
        _check(self._lib.mc_last_launch_info(self._h, ctypes.byref(info)))
        return {k: getattr(info, k) for k, _ in mc_launch_info._fields_}
