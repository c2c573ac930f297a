"""mc_integrate_static -- the entry point for callers that may not allocate device memory.

Collected last on purpose (the "zz"): `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.

Who needs it: a program whose own pool has taken the whole GPU (a library's cudaMalloc then fails), a loop with a
latency budget (cudaMalloc / cudaFree stall every stream of the process), code that runs while a stream is being
captured (allocation is refused there).  mc_integrate cannot serve them because its handle cudaMallocs the kernel's
bookkeeping; mc_integrate_static keeps that bookkeeping in a fixed array inside libmc.so, which limits the batch to
MC_STATIC_MAX_TRAJECTORIES and makes all calls on a device share one array.  What is checked here:
  * CPU: batches beyond the limit are refused, with an error text that names the limit, before any CUDA call;
  * GPU: two calls in a row (different batch sizes, so the second one meets the leftovers of the first in the shared
    array) give what mc_integrate gives on the same inputs, and the second call leaves the device's free memory as it
    found it.
"""
import ctypes

import numpy as np
import pytest

from paper_1802_00147_b200 import binding, workloads

STATE_RTOL = 1e-10      # the state tolerance of tests/test_parity_gpu.py (north_star)
FLI_VALUE_TOL = 3e-3    # its FLI value tolerance


def test_batches_beyond_the_fixed_scratch_are_refused_in_words():
    lib = binding.load_library()
    p = binding.params_default()
    limit = binding.MC_STATIC_MAX_TRAJECTORIES
    one = ctypes.c_void_p(8)     # never dereferenced: the size check comes before any CUDA call
    # without a shadow the limit counts orbits, with one it counts orbit + shadow
    assert lib.mc_integrate_static(ctypes.byref(p), one, limit + 1, 1.0, 10, 3, 0.0, one, None, None, one, one) == binding.MC_ELIMIT
    assert lib.mc_integrate_static(ctypes.byref(p), one, limit // 2 + 1, 1.0, 10, 3, 1e-8, one, None, one, one, one) == binding.MC_ELIMIT
    text = lib.mc_strerror(binding.MC_ELIMIT).decode()
    assert str(limit) in text and "mc_integrate_static" in text
    # the other refusals: bad parameters, missing required outputs, the term whose outputs need a handle
    assert lib.mc_integrate_static(None, one, 1, 1.0, 10, 3, 0.0, one, None, None, one, one) == binding.MC_EINVAL
    assert lib.mc_integrate_static(ctypes.byref(p), one, 4, 1.0, 10, 3, 0.0, one, None, None, None, one) == binding.MC_EINVAL
    assert lib.mc_integrate_static(ctypes.byref(p), one, 4, 1.0, 10, 3, 1e-8, one, None, None, one, one) == binding.MC_EINVAL
    p.terms |= binding.MC_TERM_RR
    assert lib.mc_integrate_static(ctypes.byref(p), one, 4, 1.0, 10, 3, 0.0, one, None, None, one, one) == binding.MC_EINVAL
    # an empty batch is valid and touches nothing
    p = binding.params_default()
    assert lib.mc_integrate_static(ctypes.byref(p), None, 0, 1.0, 10, 3, 0.0, None, None, None, None, None) == binding.MC_OK


def _rel_state_err(a, b):
    worst = 0.0
    for s in (slice(0, 3), slice(3, 6), slice(6, 9), slice(9, 12)):
        worst = max(worst, float((np.linalg.norm(a[s] - b[s], axis=0) / np.linalg.norm(b[s], axis=0)).max()))
    return worst


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_mc_integrate_on_two_calls_in_a_row():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    # BASELINE config 1's kind of batch: per-orbit parameters, shadow + FLI, six-integral correction
    w = workloads.config1()
    par = {k: v for k, v in w.params().items() if k != "terms"}
    n_steps = 700                                    # not a multiple of renorm_interval: the final FLI term is non-zero
    with binding.Integrator(terms=w.terms, **par) as I:
        # second batch smaller than the first and of ragged size: it runs on the array as the first call left it
        for n in (1000, 333):
            z = torch.as_tensor(w.states[:, :n], dtype=torch.float64).contiguous().to(I.device)
            want = I.integrate(z, w.h, n_steps, 3, shadow_eps=w.shadow_eps)
            out = binding.IntegrateResult(torch.empty_like(z), torch.empty_like(z),
                                          torch.empty(n, dtype=torch.float64, device=I.device),
                                          torch.full((n,), -7, dtype=torch.int32, device=I.device),
                                          torch.full((n,), -7, dtype=torch.int64, device=I.device))
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info(I.device)[0]
            got = I.integrate_static(z, w.h, n_steps, 3, shadow_eps=w.shadow_eps, out=out)
            torch.cuda.synchronize()
            free_after = torch.cuda.mem_get_info(I.device)[0]
            if n != 1000:                            # the first call may make the driver load the kernel
                assert free_after == free_before, (free_before, free_after)
            assert torch.equal(got.status, want.status)
            assert torch.equal(got.steps_done, want.steps_done)
            assert int((want.status == 0).sum()) > n // 2     # the comparison is not about dropped orbits only
            live = (want.status == 0).cpu().numpy()            # dropped orbits keep their last good state; FLI may be NaN
            gs, ws = got.states.cpu().numpy(), want.states.cpu().numpy()
            gf, wf = got.fli.cpu().numpy(), want.fli.cpu().numpy()
            gi, wi = got.invariants.cpu().numpy(), want.invariants.cpu().numpy()
            assert np.isfinite(gs[:, live]).all() and np.isfinite(gf[live]).all()
            assert _rel_state_err(gs[:, live], ws[:, live]) <= STATE_RTOL
            assert np.abs(gf[live] - wf[live]).max() <= FLI_VALUE_TOL
            assert np.abs(gi[:, live] - wi[:, live]).max() <= 1e-13 * max(1.0, np.abs(wi[:, live]).max())
            # same kernel, same single chunk: in fact nothing differs at all, dropped orbits included
            assert np.array_equal(gs, ws, equal_nan=True) and np.array_equal(gf, wf, equal_nan=True)
    # a uniform-parameter batch without a shadow, at the limit itself, goes through the same array afterwards
    limit = binding.MC_STATIC_MAX_TRAJECTORIES
    w0 = workloads.config0(64)
    z = torch.as_tensor(np.tile(w0.states, (1, limit // 64)), dtype=torch.float64).contiguous().cuda()
    par0 = {k: v for k, v in w0.params().items() if k != "terms"}
    with binding.Integrator(terms=w0.terms, **par0) as I:
        want = I.integrate(z, w0.h, 50, 3)
        got = I.integrate_static(z, w0.h, 50, 3)
        torch.cuda.synchronize()
        assert torch.equal(got.status, want.status) and torch.equal(got.steps_done, want.steps_done)
        live = (want.status == 0).cpu().numpy()
        assert live.any()
        assert _rel_state_err(got.states.cpu().numpy()[:, live], want.states.cpu().numpy()[:, live]) <= STATE_RTOL
        with pytest.raises(binding.MCError) as ei:
            I.integrate_static(torch.cat([z, z[:, :1]], dim=1).contiguous(), w0.h, 50, 3)
        assert ei.value.code == binding.MC_ELIMIT
