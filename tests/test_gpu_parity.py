"""-m gpu: the CUDA path (through the C-ABI binding) against the CPU oracle on the same seeded inputs.

Tolerances are north_star's: bin assignment bit-exact, per-bin relative error <= 1e-7,
NLL absolute error <= 1e-6."""
import numpy as np
import pytest

import workloads
from workloads.spec import OSC_EQ1, OSC_FULL3, OSC_STERILE4

pytestmark = pytest.mark.gpu

REL_BIN = 1e-7
ABS_NLL = 1e-6


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def _data_for(orc, wl, oracle_mod):
    """Pseudo-data n ~ Poisson(mu(theta0)) with mu from the ORACLE (never from the CUDA path)."""
    h0 = orc.spectra(wl.theta0[None, :])
    mu0 = orc.expectation(wl.theta0[None, :], h0)[0]
    return workloads.poisson_counts(mu0, wl.seed + 7)


def _check_hist(h_gpu, h_orc):
    assert h_gpu.shape == h_orc.shape
    zero = h_orc == 0.0
    assert np.array_equal(h_gpu[zero], h_orc[zero])              # empty bins are exactly empty
    rel = np.abs(h_gpu[~zero] - h_orc[~zero]) / np.abs(h_orc[~zero])
    assert rel.size == 0 or rel.max() <= REL_BIN, rel.max()
    return 0.0 if rel.size == 0 else float(rel.max())


def _run_case(gpu, oracle_mod, wl, check_bins=True, points=None, tuning=None):
    import torch
    params = wl.params if points is None else wl.params[points]
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        if tuning:
            ph.set_tuning(*tuning)
        dp = _dev(params)
        h = ph.spectra(dp).cpu().numpy()
        nll = ph.nll(dp, _dev(data)).cpu().numpy()
        bins = ph.event_bins(dp).cpu().numpy() if check_bins else None
        torch.cuda.synchronize()
    h_o = orc.spectra(params)
    nll_o = orc.nll(params, data)
    rel = _check_hist(h, h_o)
    fin = np.isfinite(nll_o)
    assert np.array_equal(np.isfinite(nll), fin)
    assert np.array_equal(nll[~fin], nll_o[~fin], equal_nan=True)
    err = np.abs(nll[fin] - nll_o[fin]).max() if fin.any() else 0.0
    assert err <= ABS_NLL, err
    if check_bins:
        assert np.array_equal(bins, orc.event_bins(params))       # bit-exact bin assignment
    return rel, err


@pytest.mark.parametrize("osc,ordering", [(OSC_EQ1, +1), (OSC_FULL3, +1), (OSC_FULL3, -1), (OSC_STERILE4, +1)])
@pytest.mark.parametrize("n_datasets", [1, 3])
def test_tiny_inputs(gpu, oracle_mod, osc, ordering, n_datasets):
    wl = workloads.make_tiny(seed=40 + osc, osc_model=osc, n_events=100, n_points=5, n_datasets=n_datasets,
                             ordering=ordering)
    _run_case(gpu, oracle_mod, wl)


def test_inverted_ordering_is_a_different_spectrum(gpu, oracle_mod):
    """PAPER.md:226 (section 4.3): the mass ordering flips the sign of the Delta m^2_21 share in Delta m^2_31/32
    (R5).  The CUDA path must follow the flag: both orderings against the oracle, and the two
    differ by far more than the parity bar, so a kernel that ignored the flag could not pass."""
    import torch
    hists = {}
    for o in (+1, -1):
        wl = workloads.make_config(4, scale=0.004, n_points=7, ordering=o)
        orc = oracle_mod.Oracle(wl.model, wl.events)
        with gpu.Phylino() as ph:
            ph.load_workload(wl)
            h = ph.spectra(_dev(wl.params)).cpu().numpy()
            torch.cuda.synchronize()
        _check_hist(h, orc.spectra(wl.params))
        hists[o] = h
    nz = hists[+1] != 0
    assert (np.abs(hists[+1] - hists[-1])[nz] / hists[+1][nz]).max() > 1e-3


@pytest.mark.parametrize("osc", [OSC_EQ1, OSC_STERILE4])
def test_weighted_events_full_point_groups(gpu, oracle_mod, osc):
    """Random weights U(0.5, 1.5) with 70 points: two full groups of 32 lanes (the weighted straight-line
    path; the BASELINE configs all have weight 1 and take the unit-weight one) plus a ragged group of 6."""
    wl = workloads.make_tiny(seed=91 + osc, osc_model=osc, n_events=3001, n_points=70, n_datasets=2)
    assert any(np.any(e.w != 1.0) for e in wl.events)
    _run_case(gpu, oracle_mod, wl)
    _run_case(gpu, oracle_mod, wl, tuning=(64, 1, 0))


# scaled-down copies of the five BASELINE.json configs: several CTA tiles (2048 events) per dataset
# and a ragged tail, a point count that is not a multiple of the point chunk
@pytest.mark.parametrize("k,scale,n_points,ordering", [(1, 0.137, 3, +1), (2, 0.0123, 19, +1), (3, 0.0051, 41, +1),
                                                        (4, 0.00217, 9, +1), (4, 0.00217, 9, -1), (5, 0.0097, 37, +1)])
def test_configs_scaled(gpu, oracle_mod, k, scale, n_points, ordering):
    wl = workloads.make_config(k, scale=scale, n_points=n_points, ordering=ordering)
    _run_case(gpu, oracle_mod, wl)


def test_config1_full(gpu, oracle_mod):
    _run_case(gpu, oracle_mod, workloads.make_config(1))


def test_bitwise_reproducible(gpu, oracle_mod):
    import torch
    wl = workloads.make_config(2, scale=0.02, n_points=23)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _dev(_data_for(orc, wl, oracle_mod))
    dp = _dev(wl.params)
    outs = {}
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        for tun in ((0, 0, 0), (0, 0, 0), (64, 0, 0), (0, 0, 37), (4096, 3, 1000), (0, 0, 37), (64, 0, 0), (0, 0, 0)):
            ph.set_tuning(*tun)
            outs.setdefault(tun, []).append((ph.spectra(dp).cpu().numpy(), ph.nll(dp, data).cpu().numpy()))
    torch.cuda.synchronize()
    # same inputs, same launch configuration => the same bits, call after call
    for tun, runs in outs.items():
        for h, n in runs[1:]:
            assert h.tobytes() == runs[0][0].tobytes() and n.tobytes() == runs[0][1].tobytes(), tun
    # another unit length / grid changes which events a lane sums in fp64 before the (exact) integer
    # accumulation: rounding-level differences only
    for tun, runs in outs.items():
        assert np.allclose(runs[0][0], outs[(0, 0, 0)][0][0], rtol=1e-13, atol=0)
        assert np.allclose(runs[0][1], outs[(0, 0, 0)][0][1], rtol=0, atol=1e-9)
    outs = [(outs[(0, 0, 0)][0][0].tobytes(), None)]
    # a second context on a permuted copy of the events gives the same bits: the fixed-point
    # accumulators do not depend on arrival order, the sort is by E_vis
    wl2 = workloads.make_config(2, scale=0.02, n_points=23)
    rng = np.random.Generator(np.random.PCG64(5))
    for e in wl2.events:
        perm = rng.permutation(e.n)
        e.e_nu, e.e_vis, e.w, e.core = e.e_nu[perm], e.e_vis[perm], e.w[perm], e.core[perm]
    with gpu.Phylino() as ph:
        ph.load_workload(wl2)
        h2 = ph.spectra(dp).cpu().numpy()
    h1 = np.frombuffer(outs[0][0], dtype=np.float64).reshape(h2.shape)
    # equal E_vis keys may be ordered differently inside a thread's run -> allow rounding-level difference
    assert np.allclose(h1, h2, rtol=1e-13, atol=0)


def test_host_entry_points_match_device_ones(gpu, oracle_mod):
    wl = workloads.make_config(2, scale=0.01, n_points=7)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        dp = _dev(wl.params)
        h_d = ph.spectra(dp).cpu().numpy()
        n_d = ph.nll(dp, _dev(data)).cpu().numpy()
        h_h = ph.spectra_host(wl.params)
        n_h = ph.nll_host(wl.params, data)
        assert ph.launch_count == 8              # small batch: (setup fused into spectra) + finalize per call
    assert h_d.tobytes() == h_h.tobytes() and n_d.tobytes() == n_h.tobytes()


# ---- edge cases ------------------------------------------------------------------------------
def _one_dataset_model(n_bins, osc=OSC_EQ1, idx_a=(-1, -1, -1), n_params=4):
    from workloads.spec import DatasetSpec, ModelSpec
    return ModelSpec(osc_model=osc, n_params=n_params, idx_osc=(0, 1, 2, 3, -1, -1), fixed_osc=(0,) * 6,
                     datasets=[DatasetSpec(n_bins=n_bins, idx_a=idx_a)])


THETA = np.array([[0.1, 2.5e-3, 0.85, 7.5e-5]])


def _events(e_nu, e_vis, w, edges, L=(1050.0,), core=None):
    from workloads.spec import DatasetEvents
    n = len(e_nu)
    return DatasetEvents(e_nu=np.asarray(e_nu, np.float32), e_vis=np.asarray(e_vis, np.float32),
                         w=np.asarray(w, np.float32),
                         core=np.zeros(n, np.int32) if core is None else np.asarray(core, np.int32),
                         L_m=np.asarray(L, np.float64), edges=np.asarray(edges, np.float64))


def _both(gpu, oracle_mod, model, evs, params, check_bins=True):
    from workloads.spec import Workload
    wl = Workload(name="edge", model=model, events=evs, params=np.asarray(params, np.float64),
                  theta0=np.asarray(params[0], np.float64), seed=1)
    orc = oracle_mod.Oracle(model, evs)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        dp = _dev(wl.params)
        h = ph.spectra(dp).cpu().numpy()
        b = ph.event_bins(dp).cpu().numpy() if (check_bins and wl.n_events) else None
    h_o = orc.spectra(wl.params)
    if b is not None:
        assert np.array_equal(b, orc.event_bins(wl.params))
    return h, h_o


def test_empty_dataset_and_single_event(gpu, oracle_mod):
    edges = np.linspace(1.0, 8.0, 8)
    h, h_o = _both(gpu, oracle_mod, _one_dataset_model(7), [_events([], [], [], edges)], THETA, check_bins=False)
    assert np.array_equal(h, np.zeros((1, 7))) and np.array_equal(h_o, h)
    h, h_o = _both(gpu, oracle_mod, _one_dataset_model(7), [_events([3.5], [2.7], [1.25], edges)], THETA)
    _check_hist(h, h_o)
    assert np.count_nonzero(h) == 1


def test_all_datasets_empty_large_batch(gpu, oracle_mod):
    """Every dataset empty and more points than the single-launch kernel takes: no setup and no spectra kernel is
    launched, the finalize kernel runs alone (as an ordinary launch -- it has no spectra kernel in front of it to order
    it behind the producer of params and data, which here is the device op enqueued right before the call).
    mu = backgrounds only, NLL = deviance against them + priors."""
    import torch
    from workloads.spec import BkgSpec, DatasetSpec, ModelSpec, Workload
    rng = np.random.Generator(np.random.PCG64(41))
    edges = np.linspace(1.0, 8.0, 8)
    model = ModelSpec(osc_model=OSC_EQ1, n_params=5, idx_osc=(0, 1, 2, 3, -1, -1), fixed_osc=(0,) * 6,
                      datasets=[DatasetSpec(n_bins=7, bkg=[BkgSpec(tmpl=rng.uniform(5.0, 50.0, 7), idx_rate=4)]),
                                DatasetSpec(n_bins=7, bkg=[BkgSpec(tmpl=rng.uniform(5.0, 50.0, 7), idx_rate=4)])],
                      prior_mean=np.array([0.1, 2.5e-3, 0.85, 7.5e-5, 1.0]), prior_sigma=np.array([0, 1e-4, 0.02, 2e-6, 0.1]))
    evs = [_events([], [], [], edges), _events([], [], [], edges)]
    P = 40
    params = np.array([0.1, 2.5e-3, 0.85, 7.5e-5, 1.0])[None, :] * (1.0 + 0.05 * rng.standard_normal((P, 5)))
    data = rng.poisson(25.0, 14).astype(np.float64)
    orc = oracle_mod.Oracle(model, evs)
    with gpu.Phylino() as ph:
        ph.load_workload(Workload("empty", model, evs, params, params[0], 1))
        for _ in range(3):
            half = _dev(params * 0.5)
            dp = half + half                        # produced on the stream right before the call
            nll = ph.nll(dp, _dev(data))
            h = ph.spectra(dp)
        nll, h = nll.cpu().numpy(), h.cpu().numpy()
    assert np.array_equal(h, np.zeros((P, 14)))
    assert np.abs(nll - orc.nll(params, data)).max() <= ABS_NLL


def test_edges_underflow_overflow_nan(gpu, oracle_mod):
    edges = np.array([1.0, 1.5, 2.25, 3.0, 3.5, 4.75, 6.0, 9.0])
    below = np.nextafter(np.float32(1.0), np.float32(0.0))
    e_vis = [1.0, below, 9.0, np.nextafter(np.float32(9.0), np.float32(0.0)), 2.25, 3.5, np.nan, -1.0, 50.0, 6.0]
    n = len(e_vis)
    h, h_o = _both(gpu, oracle_mod, _one_dataset_model(7), [_events([3.0 + 0.1 * i for i in range(n)], e_vis,
                                                                     [1.0 + 0.01 * i for i in range(n)], edges)], THETA)
    _check_hist(h, h_o)
    # all events out of range
    h, h_o = _both(gpu, oracle_mod, _one_dataset_model(7), [_events([3.0] * 5, [0.1, 0.2, 20.0, 30.0, np.nan],
                                                                     [1.0] * 5, edges)], THETA)
    assert np.array_equal(h, np.zeros((1, 7))) and np.array_equal(h_o, h)


def test_energy_scale_moves_events_across_edges(gpu, oracle_mod):
    """events sit exactly on edges; a0 shifts of +-1 ulp-scale and of one bin width."""
    rng = np.random.Generator(np.random.PCG64(3))
    edges = 1.0 + 0.25 * np.arange(30)
    e_vis = np.concatenate([edges[:-1], edges[:-1] + 0.125, rng.uniform(0.5, 9.0, 3000)]).astype(np.float32)
    n = len(e_vis)
    evs = [_events(rng.uniform(2.0, 8.0, n), e_vis, rng.uniform(0.5, 1.5, n), edges, L=(400.0, 1100.0),
                   core=rng.integers(0, 2, n))]
    model = _one_dataset_model(29, idx_a=(4, 5, 6), n_params=7)
    base = np.array([0.1, 2.5e-3, 0.85, 7.5e-5, 0.0, 1.0, 0.0])
    pts = [base.copy() for _ in range(9)]
    pts[1][4] = 0.25; pts[2][4] = -0.25; pts[3][4] = 1e-16; pts[4][4] = -1e-16
    pts[5][5] = 1.0 + 2 ** -52; pts[6][5] = 1.0 - 2 ** -53; pts[7][6] = 1e-3; pts[8][5:7] = (-1.0, 0.3)
    h, h_o = _both(gpu, oracle_mod, model, evs, np.array(pts))
    _check_hist(h, h_o)


def test_nan_and_unphysical_points_propagate(gpu, oracle_mod):
    wl = workloads.make_tiny(seed=77, osc_model=OSC_EQ1, n_events=100, n_points=6)
    wl.params[1, 0] = np.nan           # sin^2 2theta13 = NaN
    wl.params[2, 2] = 1.5              # sin^2 2theta12 > 1: sqrt of a negative
    wl.params[3, 1] = np.nan           # dm2_ee = NaN
    wl.params[4, 6] = np.nan           # a0 = NaN: every event of dataset 0 leaves the histogram
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        dp = _dev(wl.params)
        h = ph.spectra(dp).cpu().numpy()
        nll = ph.nll(dp, _dev(data)).cpu().numpy()
        # the accumulators were left clean: a following good batch is unaffected
        good = workloads.make_tiny(seed=77, osc_model=OSC_EQ1, n_events=100, n_points=6).params
        h2 = ph.spectra(_dev(good)).cpu().numpy()
    h_o = orc.spectra(wl.params)
    assert np.array_equal(np.isnan(h), np.isnan(h_o))
    ok = ~np.isnan(h_o)
    _check_hist(h[ok], h_o[ok])
    nll_o = orc.nll(wl.params, data)
    assert np.array_equal(np.isnan(nll), np.isnan(nll_o))
    fin = np.isfinite(nll_o)
    assert np.abs(nll[fin] - nll_o[fin]).max() <= ABS_NLL
    _check_hist(h2, orc.spectra(good))


def test_zero_count_and_zero_mu_bins(gpu, oracle_mod):
    wl = workloads.make_tiny(seed=78, osc_model=OSC_EQ1, n_events=60, n_points=3)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    data[::2] = 0.0
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        nll = ph.nll(_dev(wl.params), _dev(data)).cpu().numpy()
    assert np.abs(nll - orc.nll(wl.params, data)).max() <= ABS_NLL
    # no backgrounds + an empty bin with observed counts -> mu = 0, n > 0 -> +inf on both sides
    edges = np.linspace(1.0, 8.0, 8)
    model = _one_dataset_model(7)
    evs = [_events([3.5, 4.0], [2.7, 2.8], [1.0, 1.0], edges)]
    orc = oracle_mod.Oracle(model, evs)
    d = np.array([0, 2, 0, 0, 3, 0, 0], dtype=np.float64)
    from workloads.spec import Workload
    with gpu.Phylino() as ph:
        ph.load_workload(Workload("z", model, evs, THETA, THETA[0], 1))
        nll = ph.nll(_dev(THETA), _dev(d)).cpu().numpy()
    assert np.isposinf(nll).all() and np.isposinf(orc.nll(THETA, d)).all()


def test_eighteen_datasets_and_odd_bin_counts(gpu, oracle_mod):
    """splitting gives 18 histograms; bin counts that are not multiples of 32."""
    from workloads.spec import DatasetSpec, ModelSpec, Workload
    rng = np.random.Generator(np.random.PCG64(18))
    D = 18
    evs, dss = [], []
    for d in range(D):
        B = 5 + 3 * d
        edges = np.sort(rng.uniform(0.8, 9.5, B + 1))
        edges[0], edges[-1] = 0.8, 9.5
        evs.append(workloads.reactor_events(rng, 300 + 411 * d, [355.0, 469.0, 1050.0], [0.3, 0.3, 0.4], 0.08,
                                            edges, weights="uniform"))
        dss.append(DatasetSpec(n_bins=B, idx_a=(4 + 3 * (d % 2), 5 + 3 * (d % 2), 6 + 3 * (d % 2)), norm=0.5))
    model = ModelSpec(osc_model=OSC_EQ1, n_params=10, idx_osc=(0, 1, 2, 3, -1, -1), fixed_osc=(0,) * 6, datasets=dss)
    base = np.array([0.1, 2.5e-3, 0.85, 7.5e-5, 0.0, 1.0, 0.0, 0.01, 0.99, 0.001])
    params = base[None, :] + rng.standard_normal((11, 10)) * np.array([0.01, 5e-5, 0.02, 2e-6, .02, .01, .001, .02, .01, .001])
    h, h_o = _both(gpu, oracle_mod, model, evs, params)
    _check_hist(h, h_o)


def test_error_reporting(gpu):
    import torch
    wl = workloads.make_tiny(seed=5, n_events=10, n_points=2, n_datasets=2)
    with gpu.Phylino() as ph:
        dp = _dev(wl.params)
        with pytest.raises(gpu.PhylinoError) as e:
            ph.load_events(0, wl.events[0].e_nu, wl.events[0].e_vis, None, None, [1000.0], wl.events[0].edges)
        assert e.value.status == 3                                   # ERR_STATE: no model
        ph.set_model(wl.model)
        ph.load_events(0, wl.events[0].e_nu, wl.events[0].e_vis, None, None, [1000.0], wl.events[0].edges)
        out = torch.empty((2, ph.total_bins), dtype=torch.float64, device="cuda")
        with pytest.raises(gpu.PhylinoError) as e:
            ph.spectra(dp, out)
        assert e.value.status == 3 and "dataset 1" in str(e.value)    # dataset 1 not loaded
        with pytest.raises(gpu.PhylinoError) as e:
            ph.load_events(1, wl.events[1].e_nu, wl.events[1].e_vis, None, None, [1000.0], wl.events[1].edges[:-1])
        assert e.value.status == 2                                   # ERR_SHAPE: n_bins
        with pytest.raises(gpu.PhylinoError) as e:
            ph.load_events(5, wl.events[1].e_nu, wl.events[1].e_vis, None, None, [1000.0], wl.events[1].edges)
        assert e.value.status == 2
        bad = wl.events[1].e_nu.copy(); bad[3] = -1.0
        with pytest.raises(gpu.PhylinoError) as e:
            ph.load_events(1, bad, wl.events[1].e_vis, None, None, [1000.0], wl.events[1].edges)
        assert e.value.status == 1                                   # ERR_ARG
        with pytest.raises(gpu.PhylinoError) as e:
            ph.load_events(1, wl.events[1].e_nu, wl.events[1].e_vis, None, None, [1000.0], wl.events[1].edges[::-1])
        assert e.value.status == 1


def test_peak_fp64_microbenchmark_runs(gpu):
    with gpu.Phylino() as ph:
        r = ph.peak_fp64(2048)
    assert 1e12 < r < 1e14


def test_correlated_prior_blocks(gpu, oracle_mod):
    """PAPER.md:121-123 (Eq. 9, third factor): blocks of 3 and 41 parameters (the size of the paper's flux
    covariance) on config 3's 301-parameter model, dense and cached entry points, against the oracle."""
    wl = workloads.make_config(3, scale=0.003, n_points=75)
    rng = np.random.default_rng(77)
    A3, A41 = rng.normal(size=(3, 3)), rng.normal(size=(41, 41))
    V3 = (A3 @ A3.T + 0.5 * np.eye(3)) * 1e-4
    V41 = (A41 @ A41.T / 41 + 0.2 * np.eye(41)) * 4e-4
    i3 = np.array([4, 7, 10], np.int32)                    # energy-scale a0 of the three datasets
    i41 = np.arange(13, 54, dtype=np.int32)                # 41 flux parameters
    wl.model.prior_sigma = wl.model.prior_sigma.copy()
    wl.model.prior_sigma[i3] = 0.0
    wl.model.prior_sigma[i41] = 0.0
    wl.model.prior_blocks = [workloads.PriorBlock(i3, wl.theta0[i3], np.linalg.inv(V3)),
                             workloads.PriorBlock(i41, wl.theta0[i41], np.linalg.inv(V41))]
    params = wl.params.copy()
    params[:, i41] += rng.normal(0, 0.02, (params.shape[0], 41))
    params[:, i3] += rng.normal(0, 0.01, (params.shape[0], 3))
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    nll_o = orc.nll(params, data)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        nll = ph.nll(_dev(params), _dev(data)).cpu().numpy()
        nll_h = ph.nll_host(params, data)
        ph.set_caching(True)
        nll_c = ph.nll_host(params, data)
        ph.set_prior_blocks([])                            # cleared: back to the plain model
        nll_plain = ph.nll(_dev(params), _dev(data)).cpu().numpy()
    assert np.abs(nll - nll_o).max() <= ABS_NLL
    assert np.array_equal(nll, nll_h)
    assert np.abs(nll_c - nll_o).max() <= ABS_NLL
    wl.model.prior_blocks = []
    assert np.abs(nll_plain - oracle_mod.Oracle(wl.model, wl.events).nll(params, data)).max() <= ABS_NLL
    assert np.abs(nll_plain - nll).max() > 1.0             # the blocks did contribute


def test_reactor_off_rate_only_dataset(gpu, oracle_mod):
    """PAPER.md:109, :121 (Eq. 9, second factor P(n_off, mu_off)): the reactor-off period is a dataset of ONE
    bin with no MC signal events and background templates only; mu_off = sum_k r_k T_k."""
    from workloads.spec import BkgSpec, DatasetSpec, ModelSpec, Workload
    edges = 1.0 + 0.5 * np.arange(9)
    rng = np.random.default_rng(8)
    on = _events(rng.uniform(2.0, 7.0, 500), rng.uniform(0.5, 6.0, 500), np.ones(500), edges)
    off = _events([], [], [], np.array([1.0, 20.0]))
    # theta = (s13, mee, s12, m21, r_li, r_acc)
    ds_on = DatasetSpec(n_bins=8, norm=0.3, bkg=[BkgSpec(tmpl=np.full(8, 2.0), idx_rate=4)])
    ds_off = DatasetSpec(n_bins=1, norm=1.0, bkg=[BkgSpec(tmpl=np.array([6.5]), idx_rate=4),
                                                  BkgSpec(tmpl=np.array([1.25]), idx_rate=5)])
    model = ModelSpec(osc_model=OSC_EQ1, n_params=6, idx_osc=(0, 1, 2, 3, -1, -1), fixed_osc=(0,) * 6,
                      datasets=[ds_on, ds_off], prior_mean=np.array([0, 0, 0, 0, 1.0, 1.0]),
                      prior_sigma=np.array([0, 0, 0, 0, 0.0, 0.3]))
    params = np.array([[0.1, 2.5e-3, 0.85, 7.5e-5, r1, r2] for r1, r2 in ((1.0, 1.0), (0.7, 1.4), (1.3, 0.2))])
    wl = Workload(name="off", model=model, events=[on, off], params=params, theta0=params[0], seed=1)
    orc = oracle_mod.Oracle(model, wl.events)
    data = np.concatenate([np.round(orc.expectation(params[:1], orc.spectra(params[:1]))[0][:8]), [7.0]])
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        mu = ph.expectation(_dev(params)).cpu().numpy()
        nll = ph.nll(_dev(params), _dev(data)).cpu().numpy()
    assert np.allclose(mu[:, 8], 6.5 * params[:, 4] + 1.25 * params[:, 5], rtol=1e-15)
    assert np.abs(nll - orc.nll(params, data)).max() <= ABS_NLL
    # the off term alone: dev(7, mu_off) is what distinguishes the points beyond the on-data and the prior
    assert np.isfinite(nll).all()


def test_pseudo_experiment_ensemble(gpu, oracle_mod):
    """nll[p, e] for E pseudo-experiments against one batch of expectations == the plain NLL
    call per experiment (oracle), including priors, an E that is not a multiple of anything, and E = 1."""
    import torch
    wl = workloads.make_config(5, scale=0.004, n_points=45)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    mu0 = orc.expectation(wl.theta0[None, :], orc.spectra(wl.theta0[None, :]))[0]
    E = 131
    data = np.stack([workloads.poisson_counts(mu0, 500 + e) for e in range(E)])
    want = np.stack([orc.nll(wl.params, data[e]) for e in range(E)], axis=1)            # [P, E]
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        got = ph.nll_ensemble(_dev(wl.params), _dev(data)).cpu().numpy()
        one = ph.nll_ensemble(_dev(wl.params), _dev(data[:1])).cpu().numpy()
        again = ph.nll_ensemble(_dev(wl.params), _dev(data)).cpu().numpy()
        plain = ph.nll(_dev(wl.params), _dev(data[7])).cpu().numpy()
        torch.cuda.synchronize()
    assert got.shape == (45, E)
    assert np.abs(got - want).max() <= ABS_NLL
    assert np.array_equal(got, again)                      # reproducible
    assert np.abs(one[:, 0] - want[:, 0]).max() <= ABS_NLL
    assert np.abs(plain - got[:, 7]).max() <= 1e-9         # same expectations, another summation tree


def test_ensemble_with_priors_config3(gpu, oracle_mod):
    wl = workloads.make_config(3, scale=0.002, n_points=9)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    mu0 = orc.expectation(wl.theta0[None, :], orc.spectra(wl.theta0[None, :]))[0]
    data = np.stack([workloads.poisson_counts(mu0, 900 + e) for e in range(5)])
    want = np.stack([orc.nll(wl.params, data[e]) for e in range(5)], axis=1)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        got = ph.nll_ensemble(_dev(wl.params), _dev(data)).cpu().numpy()
    assert np.abs(got - want).max() <= ABS_NLL


def test_infinite_reconstructed_energies(gpu, oracle_mod):
    """E_vis = +-inf (and NaN) land in no bin on both sides, with a fixed and with a per-point energy scale,
    at the start, in the middle and at the end of the sorted store."""
    edges = np.array([1.0, 1.5, 2.25, 3.0, 3.5, 4.75, 6.0, 9.0])
    rng = np.random.default_rng(4)
    e_vis = np.concatenate([rng.uniform(0.5, 10.0, 300), [np.inf, -np.inf, np.nan, np.inf, -np.inf]]).astype(np.float32)
    rng.shuffle(e_vis)
    n = len(e_vis)
    evs = [_events(rng.uniform(2.0, 8.0, n), e_vis, rng.uniform(0.5, 1.5, n), edges)]
    h, h_o = _both(gpu, oracle_mod, _one_dataset_model(7), evs, THETA)
    _check_hist(h, h_o)
    params = np.array([[0.1, 2.5e-3, 0.85, 7.5e-5, 0.02, 1.01, -0.001], [0.1, 2.5e-3, 0.85, 7.5e-5, -0.03, 0.98, 0.002]])
    h, h_o = _both(gpu, oracle_mod, _one_dataset_model(7, idx_a=(4, 5, 6), n_params=7), evs, params)
    _check_hist(h, h_o)


def _transform_for_config3(wl, rng):
    """u = (4 oscillation, 7 energy-response, the other 288 parameters): the 9 energy-scale coefficients of the
    three datasets come from 7 parameters, a 41-parameter flux block goes through the Cholesky
    factor of its covariance, everything else is copied."""
    NP = wl.model.n_params
    n_u = NP - 2
    copy_src = np.full(NP, -1, np.int32)
    copy_src[:4] = np.arange(4)
    copy_src[13:] = np.arange(11, n_u)                   # theta[13:] <- u[11:]
    M97 = np.zeros((9, 7))
    for d in range(3):
        M97[3 * d + 2, 0] = 1.0
        M97[3 * d + 0, 1 + 2 * d] = 1.0
        M97[3 * d + 1, 2 + 2 * d] = 1.0
    M97 += 0.05 * rng.normal(size=M97.shape)
    A = rng.normal(size=(41, 41))
    L = np.linalg.cholesky((A @ A.T / 41 + 0.2 * np.eye(41)) * 4e-4)
    flux_out = np.arange(13, 54, dtype=np.int32)
    flux_in = flux_out - 2
    blocks = [workloads.TransformBlock(np.arange(4, 13, dtype=np.int32), np.arange(4, 11, dtype=np.int32),
                                       np.tile([0.0, 1.0, 0.0], 3), np.zeros(7), M97),
              workloads.TransformBlock(flux_out, flux_in, np.ones(41), np.zeros(41), L)]
    return workloads.TransformSpec(n_u=n_u, copy_src=copy_src, copy_const=np.zeros(NP), blocks=blocks)


def test_transformation_layer(gpu, oracle_mod):
    """batches of the minimiser's vectors u through the device and the host entry points,
    dense and cached, against oracle.transform followed by the oracle's NLL; then the layer removed."""
    wl = workloads.make_config(3, scale=0.003, n_points=40)
    rng = np.random.default_rng(21)
    spec = _transform_for_config3(wl, rng)
    P = 40
    u = np.zeros((P, spec.n_u))
    u[:, :4] = wl.params[:P, :4]
    u[:, 4:11] = rng.normal(0, 0.004, (P, 7))            # energy-response parameters
    u[:, 11:] = wl.params[:P, 13:]
    u[:, 11:52] = rng.normal(0, 1.0, (P, 41))            # whitened flux parameters
    u[20:] = u[:20]                                      # repeated energy scales: something for the cache
    u[20:, 0] *= 1.05
    theta = oracle_mod.transform(spec, wl.model.n_params, u)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    nll_o = orc.nll(theta, data)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        assert ph.param_width == wl.model.n_params
        ph.set_transform(spec)
        assert ph.param_width == spec.n_u
        nll_d = ph.nll(_dev(u), _dev(data)).cpu().numpy()
        h_d = ph.spectra(_dev(u)).cpu().numpy()
        nll_h = ph.nll_host(u, data)
        ph.set_caching(True)
        nll_c = ph.nll_host(u, data)
        cached_vp = ph.last_plan()[0]
        ph.set_caching(False)
        with pytest.raises(ValueError):
            ph.nll(_dev(theta), _dev(data))              # theta-wide batches are refused while the layer is set
        ph.set_transform(None)
        nll_plain = ph.nll(_dev(theta), _dev(data)).cpu().numpy()
    assert np.abs(nll_d - nll_o).max() <= ABS_NLL
    assert np.array_equal(nll_d, nll_h)                  # host and device transform: identical bits
    assert np.array_equal(nll_d, nll_plain)              # and identical to handing in the oracle's theta
    assert cached_vp > 0 and np.abs(nll_c - nll_o).max() <= ABS_NLL
    _check_hist(h_d, orc.spectra(theta))


# full BASELINE.json sizes, in the launch configuration bench.py times: the spectra of EVERY point of the batch
# element by element, and its NLL -- the 4096-point grid of config 5 included (its flattened index is
# i_s14 * 64 + i_m41, so any stride that divides 64 would skip whole dm2_41 columns, the 10 eV^2 one with its
# 7.8e3-rad phase among them: every point is compared, about half a minute of oracle time).  A systematic error of the oscillation
# weight of 1e-10 relative already shows in the NLL (a degree-4 sin^2 polynomial passes every other test and
# fails this one on config 4 with 1.4e-6).  Config 4 also in the inverted ordering.
@pytest.mark.parametrize("k,stride,ordering", [(2, 1, +1), (3, 1, +1), (4, 1, +1), (4, 1, -1), (5, 1, +1)])
def test_configs_full_size_all_points(gpu, oracle_mod, k, stride, ordering):
    import torch
    wl = workloads.make_config(k, ordering=ordering)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    pts = np.arange(0, wl.n_points, stride)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        dp = _dev(wl.params)
        nll = ph.nll(dp, _dev(data)).cpu().numpy()
        h = ph.spectra(dp)[torch.as_tensor(pts, device="cuda")].cpu().numpy()
    # one pass of the oracle over the events: spectra, then expectation and likelihood from them
    h_o = orc.spectra(wl.params[pts])
    nll_o = orc.nll_from_mu(wl.params[pts], orc.expectation(wl.params[pts], h_o), data)
    _check_hist(h, h_o)
    err = np.abs(nll[pts] - nll_o).max()
    assert err <= ABS_NLL, err
    assert err <= 1e-7, err            # where the shipped kernel actually is: ten times inside the bar
    # properties that hold at any size: every point finite, NLL >= 0 (half-deviance + priors)
    assert np.isfinite(nll).all() and (nll >= 0).all()


def test_function_priors(gpu, oracle_mod):
    """PAPER.md:80 ("the constrained parameters b_i(theta) are functions of the actually fitted nuisance parameters";
    DESIGN.md R29: polynomials with integer powers): on config 3's 301-parameter model a Gaussian constraint on the
    product (signal normalisation x background rate) of each dataset, one on a ratio of two energy-scale slopes, and a
    correlated pair (an affine combination of two flux parameters, a square) in one block together with a raw
    parameter -- dense, host, cached, single-launch and ensemble entry points against the oracle."""
    wl = workloads.make_config(3, scale=0.003, n_points=75)
    NP = wl.model.n_params
    rng = np.random.default_rng(91)
    i32 = lambda *a: np.array(a, np.int32)
    F = workloads.FunctionSpec
    th0 = wl.theta0
    fns = [F(terms=[(1.0, i32(127 + d, 130 + 3 * d), i32(1, 1))]) for d in range(3)]         # eps_d x rate_d0
    fns.append(F(terms=[(1.0, i32(5, 8), i32(1, -1))]))                                      # a1(FD-I) / a1(FD-II)
    fns.append(F(terms=[(2.0, i32(13), i32(1)), (-1.0, i32(14), i32(1))], offset=0.25))      # 2 f_0 - f_1 + 1/4
    fns.append(F(terms=[(3.0, i32(20), i32(2))]))                                            # 3 f_7^2
    wl.model.functions = fns
    orc0 = oracle_mod.Oracle(wl.model, wl.events)
    b0 = orc0.function_values(th0)
    A = rng.normal(size=(3, 3))
    V = (A @ A.T + 0.5 * np.eye(3)) * 1e-3
    blocks = [workloads.PriorBlock(i32(NP + k), b0[k:k + 1], np.array([[1.0 / (0.05 * abs(b0[k])) ** 2]])) for k in range(4)]
    blocks.append(workloads.PriorBlock(i32(NP + 4, 30, NP + 5), np.array([b0[4], th0[30], b0[5]]), np.linalg.inv(V)))
    wl.model.prior_blocks = blocks
    params = wl.params.copy()
    params[:, 13:54] += rng.normal(0, 0.02, (params.shape[0], 41))
    params[:, 127:139] *= 1.0 + rng.normal(0, 0.03, (params.shape[0], 12))
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data_for(orc, wl, oracle_mod)
    nll_o = orc.nll(params, data)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        nll = ph.nll(_dev(params), _dev(data)).cpu().numpy()
        nll_h = ph.nll_host(params, data)
        nll_1 = np.concatenate([ph.nll(_dev(params[i:i + 3]), _dev(data)).cpu().numpy() for i in (0, 30)])
        ens = ph.nll_ensemble(_dev(params[:5]), _dev(np.stack([data, data + 1.0]))).cpu().numpy()
        ph.set_caching(True)
        nll_c = ph.nll_host(params, data)
        ph.set_caching(False)
        # removing functions that blocks still name is refused; blocks first, then functions
        with pytest.raises(gpu.PhylinoError):
            ph.set_functions([])
        ph.set_prior_blocks([])
        ph.set_functions([])
        nll_plain = ph.nll(_dev(params), _dev(data)).cpu().numpy()
        with pytest.raises(gpu.PhylinoError):                   # no functions any more: the index is out of range
            ph.set_prior_blocks(blocks[:1])
    assert np.abs(nll - nll_o).max() <= ABS_NLL
    assert np.array_equal(nll, nll_h)
    assert np.abs(nll_1 - nll_o[[0, 1, 2, 30, 31, 32]]).max() <= ABS_NLL
    assert np.abs(nll_c - nll_o).max() <= ABS_NLL
    assert np.abs(ens[:, 0] - nll_o[:5]).max() <= ABS_NLL
    assert np.abs(ens[:, 1] - orc.nll(params[:5], data + 1.0)).max() <= ABS_NLL
    wl.model.prior_blocks, wl.model.functions = [], []
    assert np.abs(nll_plain - oracle_mod.Oracle(wl.model, wl.events).nll(params, data)).max() <= ABS_NLL
    assert np.abs(nll_plain - nll).max() > 0.1              # the constraints did contribute
