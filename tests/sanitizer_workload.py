"""A tiny workload that reaches every kernel path, for `compute-sanitizer`:

    compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_workload.py

Paths: ticket schedule with full groups, a ragged group and sub-streams (70 points), the small-batch kernel with its
in-CTA tables (1, 5, 16 points), weighted and unit-weight records, bin edges inside units (per-event slow path, general
sub-stream flush), the edge-first unit order of the single-launch kernel (capped warps), component mode (caching),
prior blocks over parameters and over functions of them, ensembles, pseudo-data, the ordering scan, the gradient (dense
and through the structural plan) and the variable-metric step, the bin-level energy correction with a flux model, the diagnostic instantiation.
Results are checked against the oracle so that a sanitizer-clean run is also a correct one."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

import oracle  # noqa: E402
import workloads  # noqa: E402
import paper_2502_15253_b200 as pkg  # noqa: E402
from workloads.spec import FluxModel  # noqa: E402


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def close(h, h_o, nll, nll_o):
    nz = h_o != 0
    assert np.array_equal(h[~nz], h_o[~nz]) and (np.abs(h - h_o)[nz] / np.abs(h_o[nz])).max() <= 1e-7
    assert np.abs(nll - nll_o).max() <= 1e-6


def main():
    n = 0
    for osc, n_pts, weights in ((0, 70, True), (1, 5, False), (2, 16, True), (0, 1, False), (2, 33, False)):
        wl = workloads.make_tiny(seed=900 + n_pts, osc_model=osc, n_events=1500 + 13 * n_pts, n_points=n_pts, n_datasets=2,
                                 ordering=-1 if osc == 1 else 1)
        if not weights:
            for e in wl.events:
                e.w[:] = 1.0
        orc = oracle.Oracle(wl.model, wl.events)
        data = np.arange(orc.total_bins, dtype=np.float64) * 2.0 + 1.0
        h_o, nll_o = orc.spectra(wl.params), orc.nll(wl.params, data)
        with pkg.Phylino() as ph:
            ph.load_workload(wl)
            for schedule in (0, 1, 2):
                ph.set_schedule(schedule)
                h = ph.spectra(dev(wl.params)).cpu().numpy()
                nll = ph.nll(dev(wl.params), dev(data)).cpu().numpy()
                close(h, h_o, nll, nll_o)
                n += 2
            ph.set_schedule(0)
            assert np.array_equal(ph.event_bins(dev(wl.params)).cpu().numpy(), orc.event_bins(wl.params))
            ph.set_caching(True)
            p2 = np.vstack([wl.params, wl.params])
            p2[n_pts:, 0] *= 0.98
            assert np.abs(ph.nll_host(p2, data) - orc.nll(p2, data)).max() <= 1e-6
            ph.set_caching(False)
            mu0 = ph.expectation(dev(wl.theta0[None, :]))
            pseudo = ph.draw_pseudo_data(mu0[0].contiguous(), 5, seed=3)
            ens = ph.nll_ensemble(dev(wl.params), pseudo).cpu().numpy()
            assert np.array_equal(pseudo.cpu().numpy(), oracle.draw_pseudo_data(mu0.cpu().numpy()[0], 5, seed=3))
            assert np.abs(ens[:, 2] - orc.nll(wl.params, pseudo.cpu().numpy()[2])).max() <= 1e-6
            step = np.full(wl.model.n_params, 1e-4)
            nll0, grad = ph.nll_gradient(dev(wl.theta0), dev(step), dev(data))
            scan = ph.ordering_scan(1, dev(np.linspace(2.4e-3, 2.6e-3, 7)), dev(wl.theta0), dev(data))
            torch.cuda.synchronize()
            assert np.isfinite(grad.cpu().numpy()).all() and np.isfinite(scan.cpu().numpy()).all()
            n += 8
    # prior blocks over parameters and over functions of them; the single-launch kernel with few warps (unit order
    # table); the cached gradient through its structural plan
    wl = workloads.make_config(3, scale=0.002, n_points=40)
    NP0 = wl.model.n_params
    i32 = lambda *a: np.array(a, np.int32)      # noqa: E731
    wl.model.functions = [workloads.FunctionSpec(terms=[(1.0, i32(127, 130), i32(1, 1))]),
                          workloads.FunctionSpec(terms=[(2.0, i32(13), i32(1)), (-1.0, i32(5, 8), i32(2, -1))], offset=0.5)]
    b0 = oracle.Oracle(wl.model, wl.events).function_values(wl.theta0)
    wl.model.prior_blocks = [workloads.PriorBlock(i32(NP0, 30, NP0 + 1), np.array([b0[0], 1.0, b0[1]]),
                                                  np.array([[4e2, 1e1, 0.0], [1e1, 9e2, -2e1], [0.0, -2e1, 1e2]]))]
    orc = oracle.Oracle(wl.model, wl.events)
    data = np.full(orc.total_bins, 40.0)
    with pkg.Phylino() as ph:
        ph.load_workload(wl)
        assert np.abs(ph.nll(dev(wl.params), dev(data)).cpu().numpy() - orc.nll(wl.params, data)).max() <= 1e-6
        ph.set_tuning(0, 0, 8)
        assert np.abs(ph.nll(dev(wl.params[:3]), dev(data)).cpu().numpy() - orc.nll(wl.params[:3], data)).max() <= 1e-6
        assert np.array_equal(ph.event_bins(dev(wl.params[:1])).cpu().numpy(), orc.event_bins(wl.params[:1]))
        ph.set_tuning(0, 0, 0)
        ph.set_caching(True)
        step = np.full(NP0, 1e-4)
        nll0, grad = ph.nll_gradient(dev(wl.theta0), dev(step), dev(data))
        assert ph.last_plan()[0] > 0
        assert abs(nll0.cpu().numpy()[0] - orc.nll(wl.theta0[None, :], data)[0]) <= 1e-6
        V = np.diag(np.full(NP0, 1e-4))
        dV = dev(V)
        dxs, dgs = np.full(NP0, 1e-3), np.linspace(0.5, 2.0, NP0)
        d, edm = ph.variable_metric_step(dV, grad, dev(dxs), dev(dgs))
        V_o, d_o, edm_o, _ = oracle.variable_metric_step(V, grad.cpu().numpy(), dxs, dgs)
        assert np.array_equal(dV.cpu().numpy(), V_o) and np.array_equal(d.cpu().numpy(), d_o) and edm.cpu().numpy()[0] == edm_o
        n += 6
    # the paper's bin-level steps with a flux model
    wl = workloads.make_config(3, scale=0.001, n_points=20)
    NP0 = wl.model.n_params
    wl.model.datasets[0].idx_flux = None
    wl.model.datasets[0].flux_model = FluxModel(idx_par=np.arange(NP0, NP0 + 41, dtype=np.int32))
    wl.model.n_params = NP0 + 41
    wl.params = np.ascontiguousarray(np.hstack([wl.params, np.full((20, 41), 1.01)]))
    wl.theta0 = np.r_[wl.theta0, np.ones(41)]
    wl.model.prior_mean = np.r_[wl.model.prior_mean, np.ones(41)]
    wl.model.prior_sigma = np.r_[wl.model.prior_sigma, np.zeros(41)]
    wl.model.energy_correction = 1
    orc = oracle.Oracle(wl.model, wl.events)
    data = np.full(orc.total_bins, 50.0)
    with pkg.Phylino() as ph:
        ph.load_workload(wl)
        assert np.abs(ph.nll(dev(wl.params), dev(data)).cpu().numpy() - orc.nll(wl.params, data)).max() <= 1e-6
        assert np.abs(ph.nll(dev(wl.params[:2]), dev(data)).cpu().numpy() - orc.nll(wl.params[:2], data)).max() <= 1e-6
        n += 2
    torch.cuda.synchronize()
    print(f"sanitizer workload: {n} library calls checked against the oracle, all within the parity bars")


if __name__ == "__main__":
    main()
