"""CPU ORACLE -- test infrastructure, NOT the product.

ctypes front end of oracle/libpn_oracle.so (pn_oracle.hpp: plain long-double restatement of
arXiv 1802.00147 as read in DESIGN.md).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this package; paper_1802_00147_b200 never does.

All state arrays are float64 SoA of shape (12, n): rx ry rz px py pz s1x s1y s1z s2x s2y s2z.
Parameters are per-orbit float64 arrays of length n (scalars are broadcast).
"""
import ctypes
from dataclasses import dataclass

import numpy as np

from . import build as _build

LONG_DOUBLE = 0
DOUBLE = 1

TERM_1PN, TERM_2PN, TERM_SO, TERM_S1S2, TERM_QM, TERM_RR = 1, 2, 4, 8, 16, 32
TERMS_DEFAULT = TERM_1PN | TERM_2PN | TERM_SO | TERM_S1S2

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.oracle_max_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _states(z):
    z = np.ascontiguousarray(z, dtype=np.float64)
    if z.ndim == 1:
        z = z.reshape(12, 1)
    assert z.ndim == 2 and z.shape[0] == 12, z.shape
    return z


def _par(x, n):
    return np.ascontiguousarray(np.broadcast_to(np.asarray(x, dtype=np.float64), (n,)))


def _params(n, beta, chi1, chi2, kq1, kq2):
    return [_par(v, n) for v in (beta, chi1, chi2, kq1, kq2)]


_WHAT = {"H": (0, 1), "J": (1, 3), "rhs": (2, 12), "gradient": (3, 12), "integrals": (4, 6), "rhs16": (5, 16)}


def evaluate(what, z, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0, terms=TERMS_DEFAULT,
             precision=LONG_DOUBLE):
    """what in {"H","J","rhs","gradient","integrals","rhs16"}; returns array of shape (rows, n).
    rhs16 = rhs plus the rates of the dissipation integrals (dW/dt, dG/dt; zero without TERM_RR)."""
    z = _states(z)
    n = z.shape[1]
    code, rows = _WHAT[what]
    out = np.empty((rows, n), dtype=np.float64)
    pa = _params(n, beta, chi1, chi2, kq1, kq2)
    lib().oracle_eval(ctypes.c_int(precision), ctypes.c_int(code), ctypes.c_int64(n), _p(z),
                      *[_p(a) for a in pa], ctypes.c_uint32(terms), _p(out))
    return out


def hamiltonian(z, **kw):
    return evaluate("H", z, **kw)[0]


def total_J(z, **kw):
    return evaluate("J", z, **kw)


def rhs(z, **kw):
    return evaluate("rhs", z, **kw)


def gradient(z, **kw):
    """rows 0-2 dH/dr, 3-5 dH/dp, 6-8 dH/dS1, 9-11 dH/dS2 (S_i = physical spin vectors)."""
    return evaluate("gradient", z, **kw)


def integrals(z, **kw):
    """rows: E, Jx, Jy, Jz, |S1hat|, |S2hat|."""
    return evaluate("integrals", z, **kw)


RK4, RK5 = 0, 1     # integrator codes (RK5: Butcher's six-stage fifth-order method, R9)


def tableau(integrator=RK4):
    """(c, A, b) of the Butcher tableau the oracle really integrates with."""
    c, a, b = np.zeros(8), np.zeros(64), np.zeros(8)
    lib().oracle_tableau.restype = ctypes.c_int
    s = lib().oracle_tableau(ctypes.c_int(integrator), _p(c), _p(a), _p(b))
    return c[:s].copy(), a[:s * s].reshape(s, s).copy(), b[:s].copy()


def rk_step(z, h, integrator=RK4, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0, terms=TERMS_DEFAULT,
            precision=LONG_DOUBLE):
    """One uncorrected step of the base integrator (RK4 or RK5)."""
    z = _states(z)
    n = z.shape[1]
    out = np.empty_like(z)
    pa = _params(n, beta, chi1, chi2, kq1, kq2)
    lib().oracle_rk4_step(ctypes.c_int(precision), ctypes.c_int64(n), _p(z), *[_p(a) for a in pa],
                          ctypes.c_uint32(terms), ctypes.c_double(h), ctypes.c_int(integrator), _p(out))
    return out


def rk4_step(z, h, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0, terms=TERMS_DEFAULT,
             precision=LONG_DOUBLE):
    z = _states(z)
    n = z.shape[1]
    out = np.empty_like(z)
    pa = _params(n, beta, chi1, chi2, kq1, kq2)
    lib().oracle_rk4_step(ctypes.c_int(precision), ctypes.c_int64(n), _p(z), *[_p(a) for a in pa],
                          ctypes.c_uint32(terms), ctypes.c_double(h), ctypes.c_int(RK4), _p(out))
    return out


def correct(z, E0, J0, mode, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0, terms=TERMS_DEFAULT,
            newton_iters=4, newton_tol=1e-10, precision=LONG_DOUBLE):
    """Apply the correction operator C_mode once. Returns (z_corrected, ok[n])."""
    z = _states(z)
    n = z.shape[1]
    out = np.empty_like(z)
    ok = np.empty(n, dtype=np.int32)
    E0 = _par(E0, n)
    J0 = np.ascontiguousarray(np.broadcast_to(np.asarray(J0, dtype=np.float64).reshape(3, -1), (3, n)))
    pa = _params(n, beta, chi1, chi2, kq1, kq2)
    lib().oracle_correct(ctypes.c_int(precision), ctypes.c_int64(n), _p(z), *[_p(a) for a in pa],
                         ctypes.c_uint32(terms), _p(E0), _p(J0), ctypes.c_int(mode),
                         ctypes.c_int(newton_iters), ctypes.c_double(newton_tol), _p(out), _p(ok))
    return out, ok


@dataclass
class Result:
    states: np.ndarray       # (12, n) final / frozen states
    invariants: np.ndarray   # (12, n): six integrals at start, six at end
    fli: np.ndarray          # (n,)
    status: np.ndarray       # (n,) int32
    steps_done: np.ndarray   # (n,) int64
    gn_steps: np.ndarray     # (n,) int64: Gauss-Newton steps of mode 3 over accepted steps, orbit + shadow
    samples: np.ndarray = None   # (n_steps // sample_interval, 12, n): orbit states after steps interval, 2 interval, ...
    diss: np.ndarray = None      # (4, n): W, Gx, Gy, Gz, the work and torque integrals of the 2.5PN force (zero without TERM_RR)
    shadow: np.ndarray = None    # (16, n) with want_shadow: the shadow's final state (12 rows), then E0', J0' it is corrected onto


def integrate(z, h, n_steps, mode, shadow_eps=0.0, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0,
              terms=TERMS_DEFAULT, renorm_interval=100, newton_iters=4, newton_tol=1e-10,
              r_merge=2.0, r_escape=1e4, precision=LONG_DOUBLE, n_threads=0, integrator=RK4, sample_interval=0,
              want_shadow=False):
    """The oracle's statement of mc_integrate (include/mc.h), orbit by orbit."""
    z = _states(z)
    n = z.shape[1]
    pa = _params(n, beta, chi1, chi2, kq1, kq2)
    res = Result(np.empty_like(z), np.empty((12, n)), np.empty(n), np.empty(n, dtype=np.int32),
                 np.empty(n, dtype=np.int64), np.empty(n, dtype=np.int64))
    if sample_interval > 0:
        res.samples = np.empty((n_steps // sample_interval, 12, n))
    if want_shadow:
        res.shadow = np.empty((16, n))
    res.diss = np.empty((4, n))
    lib().oracle_integrate(ctypes.c_int(precision), ctypes.c_int64(n), _p(z), *[_p(a) for a in pa],
                           ctypes.c_uint32(terms), ctypes.c_double(h), ctypes.c_int64(n_steps),
                           ctypes.c_int(mode), ctypes.c_double(shadow_eps), ctypes.c_int(renorm_interval),
                           ctypes.c_int(newton_iters), ctypes.c_double(newton_tol),
                           ctypes.c_double(r_merge), ctypes.c_double(r_escape), _p(res.states),
                           _p(res.invariants), _p(res.fli), _p(res.status), _p(res.steps_done),
                           _p(res.gn_steps), ctypes.c_int(n_threads), ctypes.c_int(integrator),
                           ctypes.c_int64(sample_interval), _p(res.samples), _p(res.shadow), _p(res.diss))
    return res


def count_flops(z12, beta=1.0, chi1=1.0, chi2=1.0, kq1=1.0, kq2=1.0, terms=TERMS_DEFAULT, mode=3,
                newton_iters=2):
    """Exact flop counts of the oracle's formulation: dict(rhs, rk4_step, correct, H, gradient)."""
    z = np.ascontiguousarray(np.asarray(z12, dtype=np.float64).reshape(12))
    c = (ctypes.c_longlong * 5)()
    lib().oracle_count_flops(_p(z), ctypes.c_double(beta), ctypes.c_double(chi1), ctypes.c_double(chi2),
                             ctypes.c_double(kq1), ctypes.c_double(kq2), ctypes.c_uint32(terms),
                             ctypes.c_int(mode), ctypes.c_int(newton_iters), c)
    return dict(rhs=c[0], rk4_step=c[1], correct=c[2], H=c[3], gradient=c[4])


def max_threads():
    return lib().oracle_max_threads()
