"""Seeded synthetic inputs for the BASELINE.json configs.

This module holds NO arithmetic of the method (no Hamiltonian, no integrator): it only lays out
initial conditions and dynamic parameters.  It is the one module shared by the CUDA path's tests,
bench.py and the oracle's tests; it imports numpy only.

Layout: states are float64 SoA of shape (12, n): rx ry rz px py pz s1x s1y s1z s2x s2y s2z
(unit spins).  Units G = c = M = 1, r in M, p in mu.  Seeds: 1802001470 + config.
"""
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 1802001470
TERM_1PN, TERM_2PN, TERM_SO, TERM_S1S2, TERM_QM, TERM_RR = 1, 2, 4, 8, 16, 32
TERMS_DEFAULT = TERM_1PN | TERM_2PN | TERM_SO | TERM_S1S2


@dataclass
class Workload:
    name: str
    states: np.ndarray                 # (12, n) float64
    beta: np.ndarray                   # (n,) mass ratio m1/m2 in (0, 1]
    chi1: np.ndarray                   # (n,)
    chi2: np.ndarray                   # (n,)
    kq1: np.ndarray                    # (n,) quadrupole coefficient body 1 (1 = black hole)
    kq2: np.ndarray                    # (n,)
    terms: int = TERMS_DEFAULT
    h: float = 1.0
    n_steps: int = 10_000
    correction_mode: int = 3
    shadow_eps: float = 0.0
    renorm_interval: int = 100
    uniform: bool = True               # all orbits share one parameter set
    meta: dict = field(default_factory=dict)

    @property
    def n_orbits(self) -> int:
        return self.states.shape[1]

    def params(self) -> dict:
        return dict(beta=self.beta, chi1=self.chi1, chi2=self.chi2, kq1=self.kq1, kq2=self.kq2,
                    terms=self.terms)

    def subset(self, idx) -> "Workload":
        idx = np.asarray(idx)
        return Workload(self.name + "[subset]", np.ascontiguousarray(self.states[:, idx]),
                        self.beta[idx].copy(), self.chi1[idx].copy(), self.chi2[idx].copy(),
                        self.kq1[idx].copy(), self.kq2[idx].copy(), self.terms, self.h, self.n_steps,
                        self.correction_mode, self.shadow_eps, self.renorm_interval, self.uniform,
                        dict(self.meta))


def _full(n, v):
    return np.full(n, float(v))


def _sphere(rng, n):
    """Unit vectors uniform on the sphere: z ~ U[-1,1], phi ~ U[0, 2 pi)."""
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(1.0 - z * z)
    return np.stack([s * np.cos(phi), s * np.sin(phi), z])


def random_orbits(n, rng):
    """Config-0 initial conditions: r0 = (a,0,0), a ~ U[15,30]; p0 = (0, f/sqrt(a), 0),
    f ~ U[0.85,1] (1/sqrt(a) = Newtonian circular momentum per unit mu); spins uniform on the sphere."""
    a = rng.uniform(15.0, 30.0, n)
    f = rng.uniform(0.85, 1.0, n)
    z = np.zeros((12, n))
    z[0] = a
    z[4] = f / np.sqrt(a)
    z[6:9] = _sphere(rng, n)
    z[9:12] = _sphere(rng, n)
    return z


def config0(n=64, n_steps=10_000):
    """64 orbits, equal masses, chi = 1, N+1PN+2PN+SO+SS, RK4 h = 1, correction on, no shadow."""
    rng = np.random.default_rng(SEED_BASE + 0)
    return Workload("config0", random_orbits(n, rng), _full(n, 1), _full(n, 1), _full(n, 1), _full(n, 1),
                    _full(n, 1), n_steps=n_steps)


def config1(n=1024, n_steps=100_000):
    """1024 orbits, per-orbit beta ~ U[0.5,1], chi_i ~ U[0.5,1], shadow 1e-8 in x, renorm every 100."""
    rng = np.random.default_rng(SEED_BASE + 1)
    z = random_orbits(n, rng)
    beta = rng.uniform(0.5, 1.0, n)
    chi1 = rng.uniform(0.5, 1.0, n)
    chi2 = rng.uniform(0.5, 1.0, n)
    return Workload("config1", z, beta, chi1, chi2, _full(n, 1), _full(n, 1), n_steps=n_steps,
                    shadow_eps=1e-8, uniform=False)


def scan_grid(n_r=314, n_theta=314, r_lo=10.0, r_hi=60.0, py_factor=0.9):
    """Config-2 grid: r0_i = r_lo + (r_hi-r_lo) i/(n_r-1), theta_j = pi j/(n_theta-1);
    r = (r0,0,0), p = (0, py_factor/sqrt(r0), 0), S1hat = (sin theta, 0, cos theta) (rotated about y
    from +z, which is parallel to L), S2hat = (0,0,-1).  Orbit index = i*n_theta + j (r0-major)."""
    i = np.arange(n_r, dtype=np.float64)
    j = np.arange(n_theta, dtype=np.float64)
    r0 = r_lo + (r_hi - r_lo) * i / max(n_r - 1, 1)
    th = np.pi * j / max(n_theta - 1, 1)
    R, TH = np.meshgrid(r0, th, indexing="ij")
    R = R.ravel()
    TH = TH.ravel()
    n = R.size
    z = np.zeros((12, n))
    z[0] = R
    z[4] = py_factor / np.sqrt(R)
    z[6] = np.sin(TH)
    z[8] = np.cos(TH)
    z[11] = -1.0
    return z, R, TH


def config2(n_r=314, n_theta=314, n_steps=100_000):
    """314 x 314 phase-space scan (shape of PAPER.md:227, Fig 7), equal mass, chi = 1, shadow + FLI."""
    z, R, TH = scan_grid(n_r, n_theta)
    n = z.shape[1]
    return Workload("config2", z, _full(n, 1), _full(n, 1), _full(n, 1), _full(n, 1), _full(n, 1),
                    n_steps=n_steps, shadow_eps=1e-8, meta=dict(shape=(n_r, n_theta), r0=R, theta=TH))


def config3(n_r=314, n_theta=314, n_steps=100_000, qm=True):
    """Same grid, beta = 0.8, chi = 0.9, per-body quadrupole coefficient ~ U[1,8]; QM on or off."""
    z, R, TH = scan_grid(n_r, n_theta)
    n = z.shape[1]
    rng = np.random.default_rng(SEED_BASE + 3)
    kq1 = rng.uniform(1.0, 8.0, n)
    kq2 = rng.uniform(1.0, 8.0, n)
    terms = TERMS_DEFAULT | (TERM_QM if qm else 0)
    return Workload("config3-qm" + ("on" if qm else "off"), z, _full(n, 0.8), _full(n, 0.9), _full(n, 0.9),
                    kq1, kq2, terms=terms, n_steps=n_steps, shadow_eps=1e-8, uniform=False,
                    meta=dict(shape=(n_r, n_theta), r0=R, theta=TH))


def config4(log2_n=12, n_steps=20_000):
    """Throughput sweep member: 2^log2_n random orbits as config 0, shadow on, correction on."""
    n = 1 << log2_n
    rng = np.random.default_rng(SEED_BASE + 4)
    return Workload(f"config4-2^{log2_n}", random_orbits(n, rng), _full(n, 1), _full(n, 1), _full(n, 1),
                    _full(n, 1), _full(n, 1), n_steps=n_steps, shadow_eps=1e-8)


def _spin_xz(theta):
    """Unit vector at angle theta from +z in the x-z plane: (sin theta, 0, cos theta)."""
    theta = np.asarray(theta, dtype=np.float64)
    return np.stack([np.sin(theta), np.zeros_like(theta), np.cos(theta)])


def paper_scan_theta2(theta1=np.pi / 2, n=314, dtheta=0.01, n_steps=100_000):
    """The paper's 1-D scan (Fig 6): beta = 1/3, r = (5.65,0,0), p = (0,0.765,0), chi = 1,
    theta1 fixed (pi/2 for Fig 6a, 0 for Fig 6b), theta2 = 0, 0.01, ..., 3.13 (314 orbits), t = 1e5, FLI."""
    th2 = dtheta * np.arange(n)
    z = np.zeros((12, n))
    z[0] = 5.65
    z[4] = 0.765
    z[6:9] = _spin_xz(np.full(n, theta1))
    z[9:12] = _spin_xz(th2)
    return Workload(f"paper-scan-theta2(theta1={theta1:.4f})", z, _full(n, 1.0 / 3.0), _full(n, 1), _full(n, 1),
                    _full(n, 1), _full(n, 1), n_steps=n_steps, shadow_eps=1e-8, meta=dict(theta2=th2))


def paper_scan_plane(n1=314, n2=314, dtheta=0.01, n_steps=100_000):
    """The paper's 2-D scan (Fig 7): (theta1, theta2) plane, 314 x 314 orbits, r = (10.14,0,0),
    p = (0,0.365,0) (orbit 2's initial state, hence beta = 1; R20), chi = 1.  Index = i1*n2 + i2."""
    T1, T2 = np.meshgrid(dtheta * np.arange(n1), dtheta * np.arange(n2), indexing="ij")
    T1, T2 = T1.ravel(), T2.ravel()
    n = T1.size
    z = np.zeros((12, n))
    z[0] = 10.14
    z[4] = 0.365
    z[6:9] = _spin_xz(T1)
    z[9:12] = _spin_xz(T2)
    return Workload("paper-scan-plane", z, _full(n, 1), _full(n, 1), _full(n, 1), _full(n, 1), _full(n, 1),
                    n_steps=n_steps, shadow_eps=1e-8, meta=dict(shape=(n1, n2), theta1=T1, theta2=T2))


def shard_range(n_units: int, rank: int, world_size: int):
    """Contiguous, balanced [lo, hi) range of orbit indices owned by `rank` (no collective needed)."""
    base, rem = divmod(n_units, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


# The paper's own worked examples: (beta, r0, p_y, S1hat, S2hat, chi1, chi2)
def paper_orbit(which: int) -> Workload:
    d2r = np.pi / 180.0
    table = {
        1: (1.0 / 3.0, 20.0, 0.2461, (np.sin(60 * d2r), 0, np.cos(60 * d2r)),
            (np.sin(45 * d2r), 0, np.cos(45 * d2r)), 0.75, 0.75),
        2: (1.0, 10.14, 0.365, (0.13036, 0.262852, -0.955989), (0.118966, -0.13459, -0.983734), 1.0, 1.0),
        3: (1.0, 50.0, 0.140, (np.sin(45 * d2r), 0, np.cos(45 * d2r)),
            (np.sin(30 * d2r), 0, np.cos(30 * d2r)), 1.0, 0.85),
        4: (1.0, 10.0, 0.274, (np.sin(1.0), 0, np.cos(1.0)), (np.sin(1.325), 0, np.cos(1.325)), 1.0, 1.0),
    }
    beta, r0, py, s1, s2, c1, c2 = table[which]
    z = np.zeros((12, 1))
    z[0] = r0
    z[4] = py
    z[6:9, 0] = s1
    z[9:12, 0] = s2
    return Workload(f"paper-orbit{which}", z, _full(1, beta), _full(1, c1), _full(1, c2), _full(1, 1),
                    _full(1, 1), n_steps=10_000)
