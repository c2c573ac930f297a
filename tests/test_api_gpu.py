"""GPU tests of the boundary's host logic (not of the arithmetic): what a handle reports after a refused call, the
chunk policy that keeps the kernel's 32-bit per-item counters from wrapping, device tensors as per-orbit parameters."""
import ctypes

import numpy as np
import pytest

from paper_1802_00147_b200 import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1802_00147_b200 import binding
    return binding


def test_a_refused_call_leaves_the_record_of_the_last_launch_alone(mc):
    """mc_get_status / mc_get_work copy `last_n` entries.  A call that is refused (here: a mode that does not exist, then
    the one kernel combination that is not built) must not set last_n to the size of a batch no kernel ever wrote."""
    w = workloads.config0(8)
    with mc.Integrator() as I:
        good = I.integrate(w.states, 1.0, 50, 3)
        big = torch.zeros((12, 100_000), dtype=torch.float64, device=I.device)
        out = torch.empty_like(big)
        rc = I._lib.mc_integrate(I._h, big.data_ptr(), 100_000, 1.0, 10, 7, 0.0, out.data_ptr(), None, None)
        assert rc == mc.MC_EINVAL
        status = torch.full((8,), -7, dtype=torch.int32, device=I.device)     # 8 entries: a 100 000-entry copy would overrun
        steps = torch.full((8,), -7, dtype=torch.int64, device=I.device)
        assert I._lib.mc_get_status(I._h, status.data_ptr(), steps.data_ptr()) == mc.MC_OK
        torch.cuda.synchronize()
        assert torch.equal(status, good.status) and torch.equal(steps, good.steps_done)
    n = 16
    rng = np.random.default_rng(5)
    par = dict(beta=rng.uniform(0.5, 1, n), chi1=rng.uniform(0, 1, n), chi2=rng.uniform(0, 1, n), kq1=np.ones(n), kq2=np.ones(n))
    with mc.Integrator(terms=15 | mc.MC_TERM_RR, integrator=mc.MC_INTEG_RK5, **par) as I:     # per_orbit = 1 + RK5 + RR: not built
        z = torch.as_tensor(workloads.config0(n).states, device=I.device)
        out = torch.empty_like(z)
        assert I._lib.mc_integrate(I._h, z.data_ptr(), n, 1.0, 10, 3, 0.0, out.data_ptr(), None, None) == mc.MC_EINVAL
        status = torch.full((n,), -7, dtype=torch.int32, device=I.device)
        assert I._lib.mc_get_status(I._h, status.data_ptr(), None) == mc.MC_OK
        torch.cuda.synchronize()
        assert (status == -7).all()                  # nothing ran, nothing is reported


def test_chunks_are_short_enough_for_the_32_bit_item_counters(mc):
    """The kernel counts Gauss-Newton steps per work item in 32 bits, at most newton_iters per step.  A run of 2^31 - 1
    steps with newton_iters = 16 could wrap them in one chunk; the host splits it.  The orbit is non-finite from the
    start, so every chunk ends at once and the launch takes no time."""
    z = np.full((12, 1), np.nan)
    with mc.Integrator(newton_iters=16) as I:
        g = I.integrate(z, 1.0, 2 ** 31 - 1, 3, shadow_eps=1e-8)
        torch.cuda.synchronize()
        info = I.launch_info()
    assert int(g.status[0]) == 3 and int(g.steps_done[0]) == 0
    assert info["chunk_steps"] * 16 < 2 ** 32
    assert info["n_chunks"] * info["chunk_steps"] >= 2 ** 31 - 1


def test_device_tensors_as_per_orbit_parameters(mc):
    """Integrator() accepts CUDA tensors for beta, chi, kq (it used to pass them through numpy, which raises)."""
    w = workloads.config1().subset(np.arange(40))
    par = {k: v for k, v in w.params().items() if k != "terms"}
    with mc.Integrator(terms=w.terms, **par) as I:
        want = I.integrate(w.states, w.h, 200, 3, shadow_eps=w.shadow_eps)
    dev = {k: torch.as_tensor(v, dtype=torch.float64).cuda() for k, v in par.items()}
    with mc.Integrator(terms=w.terms, **dev) as I:
        got = I.integrate(w.states, w.h, 200, 3, shadow_eps=w.shadow_eps)
        assert I.params.per_orbit == 1
    assert torch.equal(got.states, want.states) and torch.equal(got.fli, want.fli)
    uni = dict(beta=torch.full((40,), 0.8, dtype=torch.float64).cuda(), chi1=0.9, chi2=0.9)
    with mc.Integrator(**uni) as I:
        assert I.params.per_orbit == 0 and I.params.beta == 0.8          # a device tensor of equal values is a uniform parameter
