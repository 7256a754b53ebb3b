"""phylino_variable_metric_step_static: the variable-metric step (R30) for users who cannot
let this library allocate on the GPU -- a fit living next to a framework whose allocator already owns the device
memory, a minimiser loop that cannot pay for the device-wide stall of a cudaMalloc, a service that forbids allocation
after start-up.  The entry point has no context and keeps its scratch in one fixed array inside the library, shared by
every call on a device and never cleared.

What is checked here: the new entry point returns the SAME BITS as the existing, allocating one
(phylino_variable_metric_step, itself compared bit for bit with the oracle in test_gpu_consumers.py -- the bar of that
test is kept), on several calls in a row that reuse the array with whatever the call before left in it (a larger N
first, then smaller ones, with and without the update), and sizes beyond the fixed maximum are refused with a text
that says so.  The file sorts last on purpose: with `pytest -x` a failure here hides nothing behind it.  It must pass
alone in a fresh process (its first call is then the one that looks the array up) and after all other tests.
"""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def _case(rng, N, vscale):
    A = rng.normal(size=(N, N))
    V = (A @ A.T / N + np.eye(N)) * vscale
    H = rng.normal(size=(N, N))
    H = H @ H.T / N + np.eye(N)
    g = rng.normal(size=N)
    dx = rng.normal(size=N) * 0.1
    return V, g, dx, H @ dx


def test_static_step_equals_the_allocating_one_call_after_call(gpu):
    import torch
    rng = np.random.default_rng(23)
    calls = 0
    with gpu.Phylino() as ph:
        # consecutive calls share one scratch array: N shrinks and grows, the update is on and off, so every call
        # finds the leftovers of a different one in it
        for N, vscale in ((301, 1.0), (37, 1e-3), (3, 1.0), (gpu.binding.STATIC_MAX_N, 1.0), (301, 1e-3)):
            V, g, dx, dg = _case(rng, N, vscale)
            for use_move in (True, False, True):
                mv = (_dev(dx), _dev(dg)) if use_move else (None, None)
                V_ref, V_new = _dev(V), _dev(V)
                d_ref, edm_ref = ph.variable_metric_step(V_ref, _dev(g), *mv)
                d_new, edm_new = gpu.variable_metric_step_static(V_new, _dev(g), *mv)
                torch.cuda.synchronize()
                calls += 1
                assert np.array_equal(V_new.cpu().numpy(), V_ref.cpu().numpy()), (N, use_move)
                assert np.array_equal(d_new.cpu().numpy(), d_ref.cpu().numpy()), (N, use_move)
                assert np.array_equal(edm_new.cpu().numpy(), edm_ref.cpu().numpy()), (N, use_move)
                assert edm_new.cpu().numpy()[1] == 0.0
                if use_move:
                    assert not np.array_equal(V_new.cpu().numpy(), V)        # the update did happen
        # the skip branch (no positive curvature) reads the two scalars of the array: same answer as the other path
        V_new = _dev(np.eye(4))
        d_new, edm_new = gpu.variable_metric_step_static(V_new, _dev(np.ones(4)), _dev(np.array([1.0, 0, 0, 0])),
                                                         _dev(np.array([-1.0, 0, 0, 0])))
        assert edm_new.cpu().numpy()[1] == 1.0 and np.array_equal(V_new.cpu().numpy(), np.eye(4))
        assert np.array_equal(d_new.cpu().numpy(), -np.ones(4))
    assert calls >= 2


def test_static_step_allocates_nothing(gpu):
    """With every buffer preallocated by the caller, two calls in a row leave the device's free memory where it was
    (cudaMemGetInfo sees any cudaMalloc, whoever makes it)."""
    import torch
    rng = np.random.default_rng(5)
    N = 128
    V, g, dx, dg = _case(rng, N, 1.0)
    dV, dg_, ddx, ddg = _dev(V), _dev(g), _dev(dx), _dev(dg)
    direction, edm = torch.empty(N, dtype=torch.float64, device="cuda"), torch.empty(2, dtype=torch.float64, device="cuda")
    gpu.variable_metric_step_static(dV, dg_, ddx, ddg, direction=direction, edm=edm)     # first use on this device, if alone
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        gpu.variable_metric_step_static(dV, dg_, ddx, ddg, direction=direction, edm=edm)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_step_refuses_what_does_not_fit(gpu):
    lib = gpu.load_library()
    err = C.create_string_buffer(256)
    too_big = gpu.binding.STATIC_MAX_N + 1
    # the size check comes before any pointer is touched
    assert lib.phylino_variable_metric_step_static(None, too_big, None, None, None, None, None, None, err, len(err)) == 2
    assert b"PHYLINO_STATIC_MAX_N" in err.value and str(gpu.binding.STATIC_MAX_N).encode() in err.value
    assert lib.phylino_variable_metric_step_static(None, -1, None, None, None, None, None, None, err, len(err)) == 2
    assert lib.phylino_variable_metric_step_static(None, 4, None, None, None, None, None, None, err, len(err)) == 1
    assert err.value
    assert lib.phylino_variable_metric_step_static(None, 0, None, None, None, None, None, None, None, 0) == 0
    import torch
    with pytest.raises(gpu.PhylinoError, match="PHYLINO_STATIC_MAX_N"):
        gpu.variable_metric_step_static(torch.zeros((too_big, too_big), dtype=torch.float64, device="cuda"),
                                        torch.zeros(too_big, dtype=torch.float64, device="cuda"))
