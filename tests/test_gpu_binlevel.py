"""-m gpu: the paper's own signal steps 2-3 on the binned spectrum and the fine-grid reactor-flux
model through the CUDA path against the oracle (R27, R28).  Bars: per bin 1e-7, NLL 1e-6."""
import numpy as np
import pytest

import workloads
from workloads.spec import FluxModel

pytestmark = pytest.mark.gpu
REL_BIN, ABS_NLL = 1e-7, 1e-6


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def _check(h, h_o, floor=0.0):
    """per-bin relative error; `floor`: bins whose content is a tiny remainder of a cancellation are compared on the
    scale of their neighbours (the smoothing parabola can leave 1e-3 events where the plain histogram has none)"""
    assert h.shape == h_o.shape
    scale = np.maximum(np.abs(h_o), floor)
    ok = scale > 0
    assert np.array_equal(h[~ok], h_o[~ok])
    assert (np.abs(h - h_o)[ok] / scale[ok]).max() <= REL_BIN


def _data(orc, wl):
    mu0 = orc.expectation(wl.theta0[None, :], orc.spectra_raw(wl.theta0[None, :]))[0]
    return workloads.poisson_counts(np.clip(mu0, 0, None), wl.seed + 7)


@pytest.mark.parametrize("k,scale,n_points", [(1, 1.0, 1), (2, 0.05, 5), (2, 0.05, 64), (3, 0.01, 41), (5, 0.05, 70)])
def test_bin_level_energy_correction(gpu, oracle_mod, k, scale, n_points):
    wl = workloads.make_config(k, scale=scale, n_points=n_points)
    if k == 5:              # the grid scan has no energy-scale parameters of its own: give every point one
        rng = np.random.default_rng(5)
        wl.model.n_params = 12
        for d, ds in enumerate(wl.model.datasets):
            ds.idx_a = (6 + 3 * d, 7 + 3 * d, 8 + 3 * d)
        ext = np.tile([0.0, 1.0, 0.0, 0.0, 1.0, 0.0], (wl.n_points, 1)) + rng.normal(size=(wl.n_points, 6)) * np.array([0.02, 0.01, 1e-3] * 2)
        wl.params = np.ascontiguousarray(np.hstack([wl.params, ext]))
        wl.theta0 = np.r_[wl.theta0, 0.0, 1.0, 0.0, 0.0, 1.0, 0.0]
        wl.model.prior_mean = np.r_[wl.model.prior_mean, np.zeros(6)]
        wl.model.prior_sigma = np.r_[wl.model.prior_sigma, np.zeros(6)]
    wl.model.energy_correction = 1
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    h_o = orc.spectra(wl.params)
    mu_o = orc.expectation(wl.params, orc.spectra_raw(wl.params))
    nll_o = orc.nll(wl.params, data)
    floor = 1e-6 * np.abs(h_o).max()
    with gpu.Phylino() as ph:
        ph.load_workload(wl)                      # sets mode 1 from the model
        h = ph.spectra(_dev(wl.params)).cpu().numpy()
        mu = ph.expectation(_dev(wl.params)).cpu().numpy()
        nll = ph.nll(_dev(wl.params), _dev(data)).cpu().numpy()
        nll_h = ph.nll_host(wl.params, data)
        ph.set_caching(True)
        nll_c = ph.nll_host(wl.params, data)
        vp, classes = ph.last_plan()
        ph.set_caching(False)
        # the raw step-1 spectrum is the identity-binned one: bins bit-exact against the oracle's
        assert np.array_equal(ph.event_bins(_dev(wl.params[:2])).cpu().numpy(), orc.event_bins(wl.params[:2]))
        # back to per-event mode on the same context
        ph.set_energy_correction_mode(0)
        h0 = ph.spectra(_dev(wl.params)).cpu().numpy()
    _check(h, h_o, floor)
    _check(mu, mu_o, floor)
    fin = np.isfinite(nll_o)
    assert np.array_equal(np.isfinite(nll), fin) and np.abs(nll[fin] - nll_o[fin]).max() <= ABS_NLL
    assert np.array_equal(nll, nll_h)
    if vp:
        assert classes == 1 and np.abs(nll_c[fin] - nll_o[fin]).max() <= ABS_NLL     # no event work depends on the scale
    wl.model.energy_correction = 0
    _check(h0, oracle_mod.Oracle(wl.model, wl.events).spectra(wl.params))


def test_bin_level_and_per_event_agree_where_they_must(gpu, oracle_mod):
    """identity scale: identical spectra in both modes (to rounding of the parabola's integral)"""
    wl = workloads.make_config(2, scale=0.03, n_points=9)
    wl.params[:, 4:10] = (0.0, 1.0, 0.0, 0.0, 1.0, 0.0)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        h0 = ph.spectra(_dev(wl.params)).cpu().numpy()
        ph.set_energy_correction_mode(1)
        h1 = ph.spectra(_dev(wl.params)).cpu().numpy()
    assert np.allclose(h1, h0, rtol=1e-12, atol=1e-9)


@pytest.mark.parametrize("mode", [0, 1])
def test_fine_grid_flux_model(gpu, oracle_mod, mode):
    """3 x 41 flux parameters on 0.25-MeV bins instead of the 3 x 38 per-bin scales of config 3"""
    wl = workloads.make_config(3, scale=0.01, n_points=33)
    NP0 = wl.model.n_params
    rng = np.random.default_rng(6)
    for d, ds in enumerate(wl.model.datasets):
        ds.idx_flux = None
        ds.flux_model = FluxModel(idx_par=np.arange(NP0 + 41 * d, NP0 + 41 * (d + 1), dtype=np.int32))
    wl.model.n_params = NP0 + 123
    wl.params = np.ascontiguousarray(np.hstack([wl.params, 1.0 + 0.02 * rng.normal(size=(wl.n_points, 123))]))
    wl.theta0 = np.r_[wl.theta0, np.ones(123)]
    wl.model.prior_mean = np.r_[wl.model.prior_mean, np.ones(123)]
    wl.model.prior_sigma = np.r_[wl.model.prior_sigma, np.full(123, 0.02)]
    wl.model.energy_correction = mode
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    mu_o = orc.expectation(wl.params, orc.spectra_raw(wl.params))
    nll_o = orc.nll(wl.params, data)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        mu = ph.expectation(_dev(wl.params)).cpu().numpy()
        nll = ph.nll(_dev(wl.params), _dev(data)).cpu().numpy()
        ph.set_flux_model(1, [])                 # dataset 1 back to "no flux scales"
        mu_without = ph.expectation(_dev(wl.params[:3])).cpu().numpy()
    _check(mu, mu_o, 1e-6 * np.abs(mu_o).max())
    assert np.abs(nll - nll_o).max() <= ABS_NLL
    wl.model.datasets[1].flux_model = None
    orc2 = oracle_mod.Oracle(wl.model, wl.events)
    _check(mu_without, orc2.expectation(wl.params[:3], orc2.spectra_raw(wl.params[:3])), 1e-6 * np.abs(mu_o).max())


def test_bin_level_mode_needs_the_staged_layout(gpu):
    from workloads.spec import DatasetSpec, ModelSpec, OSC_EQ1
    model = ModelSpec(osc_model=OSC_EQ1, n_params=4, idx_osc=(0, 1, 2, 3, -1, -1), fixed_osc=(0,) * 6,
                      datasets=[DatasetSpec(n_bins=2001)])
    with gpu.Phylino() as ph:
        ph.set_model(model)
        with pytest.raises(gpu.PhylinoError) as e:
            ph.set_energy_correction_mode(1)
        assert e.value.status == 2
        with pytest.raises(gpu.PhylinoError) as e:
            ph.set_flux_model(0, [0, 1, 2])
        assert e.value.status == 2
