"""-m gpu: the launch schedules, the hot loop's own bin assignment, contexts side by side, sharding on one GPU.

Bars as everywhere: bins bit-exact, per-bin relative error <= 1e-7, |dNLL| <= 1e-6 against the oracle."""
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


def _check_hist(h_gpu, h_orc):
    zero = h_orc == 0.0
    assert np.array_equal(h_gpu[zero], h_orc[zero])
    rel = np.abs(h_gpu[~zero] - h_orc[~zero]) / np.abs(h_orc[~zero])
    assert rel.size == 0 or rel.max() <= REL_BIN, rel.max()


def _data(orc, wl):
    mu0 = orc.expectation(wl.theta0[None, :], orc.spectra(wl.theta0[None, :]))[0]
    return workloads.poisson_counts(mu0, wl.seed + 7)


# ---- bit-exact bins FROM THE HOT LOOP (north_star "bin assignment bit-exact") ------------------------------------
# phylino_event_bins runs the production kernels of the batch size in their diagnostic instantiation: every
# event is reported with the bin the lane that accumulated it put it in -- through the hint walk, the forward
# scan, the whole-batch test, the 2-/4-batch straight-line paths, the per-event path and the sub-stream split.
# 1 / 5 points: small-batch kernel (32 / 4 sub-streams); 17: one full group with 15 shadow lanes; 33: a full group
# and a 1-point group of 32 sub-streams; 70: two full groups and a ragged one of 6.
@pytest.mark.parametrize("k,scale", [(2, 0.02), (3, 0.004), (4, 0.004), (5, 0.02)])
@pytest.mark.parametrize("n_points", [1, 5, 17, 33, 70])
def test_hot_loop_bins_scaled_configs(gpu, oracle_mod, k, scale, n_points):
    import torch
    wl = workloads.make_config(k, scale=scale)
    rng = np.random.default_rng(7 * k + n_points)
    sel = rng.choice(wl.n_points, size=n_points, replace=wl.n_points < n_points)
    params = wl.params[sel].copy()
    orc = oracle_mod.Oracle(wl.model, wl.events)
    want = orc.event_bins(params)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        for schedule in ((0, 1, 2) if n_points <= 16 else (0,)):
            ph.set_schedule(schedule)
            got = ph.event_bins(_dev(params)).cpu().numpy()
            assert np.array_equal(got, want), (schedule, int((got != want).sum()))
            # the diagnostic pass left the accumulators clean
            _check_hist(ph.spectra(_dev(params)).cpu().numpy(), orc.spectra(params))
        torch.cuda.synchronize()


@pytest.mark.parametrize("n_points", [1, 5, 17, 33, 70])
@pytest.mark.parametrize("osc", [OSC_EQ1, OSC_FULL3])
def test_hot_loop_bins_weighted_store(gpu, oracle_mod, osc, n_points):
    """random weights (the 96-byte records), per-point energy scales, three datasets, ragged event counts"""
    wl = workloads.make_tiny(seed=300 + n_points + osc, osc_model=osc, n_events=2500 + 37 * n_points, n_points=n_points,
                             n_datasets=3, ordering=-1 if osc == OSC_FULL3 else +1)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        for tuning in ((0, 0, 0), (64, 1, 0), (256, 2, 16)):
            ph.set_tuning(*tuning)
            assert np.array_equal(ph.event_bins(_dev(wl.params)).cpu().numpy(), orc.event_bins(wl.params)), tuning


# ---- schedules -----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k,scale,n_points", [(1, 1.0, 1), (2, 0.05, 3), (3, 0.01, 16), (4, 0.01, 2), (5, 0.05, 4), (5, 0.05, 11)])
def test_small_batches_every_schedule(gpu, oracle_mod, k, scale, n_points):
    """the small-batch kernel (setup fused in, finalize prologue overlapped) and the three-kernel ticket path
    against the oracle, device and host entry points; the schedules differ from each other by rounding only"""
    wl = workloads.make_config(k, scale=scale, n_points=n_points)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    h_o, nll_o = orc.spectra(wl.params), orc.nll(wl.params, data)
    mu_o = orc.expectation(wl.params, h_o)
    out = {}
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        for schedule in (0, 1, 2):
            ph.set_schedule(schedule)
            n0 = ph.launch_count
            h = ph.spectra(_dev(wl.params)).cpu().numpy()
            launches = ph.launch_count - n0
            assert launches == (3 if schedule == 1 else 2) or schedule == 0
            nll = ph.nll(_dev(wl.params), _dev(data)).cpu().numpy()
            mu = ph.expectation(_dev(wl.params)).cpu().numpy()
            nll_h = ph.nll_host(wl.params, data)
            h_h = ph.spectra_host(wl.params)
            _check_hist(h, h_o)
            _check_hist(mu, mu_o)
            assert np.abs(nll - nll_o).max() <= ABS_NLL
            assert np.array_equal(nll, nll_h) and np.array_equal(h, h_h)     # same kernels, same bits
            out[schedule] = (h, nll)
    assert np.allclose(out[1][0], out[2][0], rtol=1e-12, atol=0) and np.allclose(out[1][1], out[2][1], rtol=0, atol=1e-8)


def test_model_switch_on_one_context(gpu, oracle_mod):
    """A context that goes from a two-term model to a three-term one and back (the cached occupancy
    and the shared-memory opt-in belonged to the first model's kernels)."""
    with gpu.Phylino() as ph:
        for k, scale, n_points in ((2, 0.01, 40), (4, 0.002, 40), (2, 0.01, 3), (5, 0.01, 3), (2, 0.01, 40)):
            wl = workloads.make_config(k, scale=scale, n_points=n_points)
            orc = oracle_mod.Oracle(wl.model, wl.events)
            data = _data(orc, wl)
            ph.load_workload(wl)
            nll = ph.nll(_dev(wl.params), _dev(data)).cpu().numpy()
            assert np.abs(nll - orc.nll(wl.params, data)).max() <= ABS_NLL, k


def test_unphysical_amplitudes_near_the_fixed_point_bound(gpu, oracle_mod):
    """phylino.h "Errors": finite but unphysical mixings.  sin^2 2theta13 = -1 gives cos^4 theta13 = 1.457 and
    sum |A_k| = 2.24 <= 3: still inside the fixed-point range, parity with the oracle holds.  sin^2 2theta13 = -3
    gives sum |A_k| = 4.9 > 3: the documented NaN (the oracle, which has no fixed point, stays finite)."""
    wl = workloads.make_tiny(seed=83, osc_model=OSC_EQ1, n_events=400, n_points=4)
    wl.params[1, 0] = -1.0
    wl.params[2, 0] = -3.0
    orc = oracle_mod.Oracle(wl.model, wl.events)
    A, _ = orc.terms(wl.params[1])
    assert 2.0 < np.abs(A).sum() <= 3.0
    A, _ = orc.terms(wl.params[2])
    assert np.abs(A).sum() > 3.0
    h_o = orc.spectra(wl.params)
    assert np.isfinite(h_o).all()
    for schedule in (1, 2):
        with gpu.Phylino() as ph:
            ph.load_workload(wl)
            ph.set_schedule(schedule)
            h = ph.spectra(_dev(wl.params)).cpu().numpy()
        ok = [0, 1, 3]
        _check_hist(h[ok], h_o[ok])
        assert np.isnan(h[2]).all()


def test_two_contexts_on_two_streams(gpu, oracle_mod):
    """phylino.h "Threads": any number of contexts may coexist (independent fits).  Two contexts on
    two streams, calls interleaved with no synchronisation in between, each against the oracle."""
    import torch
    wls = [workloads.make_config(2, scale=0.05, n_points=40), workloads.make_config(5, scale=0.05, n_points=70)]
    orcs = [oracle_mod.Oracle(w.model, w.events) for w in wls]
    datas = [_data(o, w) for o, w in zip(orcs, wls)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs, outs = [], [[], []]
    for w, st in zip(wls, streams):
        ph = gpu.Phylino(stream=st.cuda_stream)
        ph.load_workload(w)
        ctxs.append(ph)
    dev = []
    for w, d, st in zip(wls, datas, streams):
        with torch.cuda.stream(st):
            dev.append((_dev(w.params), _dev(d)))
    torch.cuda.synchronize()
    for rep in range(3):
        for i in (0, 1):
            with torch.cuda.stream(streams[i]):
                outs[i].append((ctxs[i].nll(*dev[i]), ctxs[i].spectra(dev[i][0])))
    torch.cuda.synchronize()
    for i in (0, 1):
        nll_o, h_o = orcs[i].nll(wls[i].params, datas[i]), orcs[i].spectra(wls[i].params)
        for nll, h in outs[i]:
            assert np.abs(nll.cpu().numpy() - nll_o).max() <= ABS_NLL
            _check_hist(h.cpu().numpy(), h_o)
        assert all(np.array_equal(outs[i][0][0].cpu().numpy(), o[0].cpu().numpy()) for o in outs[i][1:])
    for ph in ctxs:
        ph.close()


def test_reserve_then_cuda_graph(gpu, oracle_mod):
    """phylino.h "Async": after phylino_reserve the device entry points neither allocate nor synchronise, so a
    call can be captured into a CUDA graph and replayed (the launch-bound inner loop of a minimiser)."""
    import torch
    for k, scale, n_points in ((2, 0.02, 64), (2, 0.02, 1)):
        wl = workloads.make_config(k, scale=scale, n_points=n_points)
        orc = oracle_mod.Oracle(wl.model, wl.events)
        data = _data(orc, wl)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            ph = gpu.Phylino(stream=st.cuda_stream)
            ph.load_workload(wl)
            ph.reserve(n_points)
            dp, dd = _dev(wl.params), _dev(data)
            out = torch.zeros(n_points, dtype=torch.float64, device="cuda")
            ph.nll(dp, dd, out)                       # warm: occupancy queries and attributes are set
            st.synchronize()
            first = out.cpu().numpy().copy()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                ph.nll(dp, dd, out)
            for shift in (0.0, 1e-3):
                dp[:, 0] = torch.as_tensor(wl.params[:, 0] * (1.0 + shift), device="cuda")
                out.zero_()
                g.replay()
                st.synchronize()
                p = wl.params.copy()
                p[:, 0] *= 1.0 + shift
                assert np.abs(out.cpu().numpy() - orc.nll(p, data)).max() <= ABS_NLL
                if shift == 0.0:
                    assert np.array_equal(out.cpu().numpy(), first)
        ph.close()


# ---- the multi-GPU split, with the REAL library, on one GPU -------------
@pytest.mark.parametrize("k,scale,n_points", [(2, 0.05, 64), (3, 0.01, 603)])
@pytest.mark.parametrize("world", [2, 3, 8])
def test_point_shards_agree_with_the_unsharded_batch(gpu, oracle_mod, k, scale, n_points, world):
    """Every rank evaluates a contiguous slice of the batch (sharding.shard_points).  A slice is another batch
    size, hence possibly another schedule and another grouping of the fp64 partial sums before the exact integer
    accumulation: the slices agree with the unsharded call to rounding (<= 1e-13 relative per bin, <= 1e-9 in the
    NLL), not bit for bit -- and each meets the parity bars against the oracle on its own."""
    from paper_2502_15253_b200 import sharding
    wl = workloads.make_config(k, scale=scale, n_points=n_points)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        h_all = ph.spectra(_dev(wl.params)).cpu().numpy()
        nll_all = ph.nll(_dev(wl.params), _dev(data)).cpu().numpy()
        h_parts, nll_parts = [], []
        for rank in range(world):
            lo, hi = sharding.shard_points(n_points, world, rank)
            h_parts.append(ph.spectra(_dev(wl.params[lo:hi])).cpu().numpy())
            nll_parts.append(ph.nll(_dev(wl.params[lo:hi]), _dev(data)).cpu().numpy())
    h_sh, nll_sh = np.concatenate(h_parts), np.concatenate(nll_parts)
    assert h_sh.shape == h_all.shape
    assert np.allclose(h_sh, h_all, rtol=1e-13, atol=0.0)
    assert np.abs(nll_sh - nll_all).max() <= 1e-9
    _check_hist(h_sh, orc.spectra(wl.params))
    assert np.abs(nll_sh - orc.nll(wl.params, data)).max() <= ABS_NLL


# ---- the 41 -> 38 flux block through the transformation layer --------------------------------------
def test_flux_rebinning_block_through_set_transform(gpu, oracle_mod):
    """41 flux parameters on uniform 0.25-MeV bins (1-11.25 MeV) drive the 38 per-bin flux scales of each of config
    3's datasets through one 38 x 41 area-conserving block per dataset of phylino_set_transform; NLL and
    expectations against oracle.transform followed by the oracle."""
    wl = workloads.make_config(3, scale=0.004, n_points=24)
    NP = wl.model.n_params
    edges = workloads.dc_edges()
    fine = 1.0 + 0.25 * np.arange(42)
    M = np.zeros((38, 41))
    off = np.zeros(38)
    for b in range(38):
        lo, hi = edges[b], edges[b + 1]
        for j in range(41):
            M[b, j] = max(0.0, min(hi, fine[j + 1]) - max(lo, fine[j])) / (hi - lo)
        off[b] = 1.0 - M[b].sum()
    # u = theta without the 3 x 38 flux scales (theta[13:127]) + 3 x 41 flux-model parameters at the end
    keep = np.r_[0:13, 127:NP]
    n_keep = keep.size
    n_u = n_keep + 3 * 41
    copy_src = np.full(NP, -1, np.int32)
    copy_src[keep] = np.arange(n_keep)
    blocks = [workloads.TransformBlock(np.arange(13 + 38 * d, 13 + 38 * (d + 1), dtype=np.int32),
                                       np.arange(n_keep + 41 * d, n_keep + 41 * (d + 1), dtype=np.int32),
                                       off, np.zeros(41), M) for d in range(3)]
    spec = workloads.TransformSpec(n_u=n_u, copy_src=copy_src, copy_const=np.zeros(NP), blocks=blocks)
    rng = np.random.default_rng(12)
    u = np.zeros((24, n_u))
    u[:, :n_keep] = wl.params[:, keep]
    u[:, n_keep:] = 1.0 + 0.02 * rng.normal(size=(24, 123))
    theta = oracle_mod.transform(spec, NP, u)
    assert np.allclose(theta[:, 13:13 + 28], u[:, n_keep:n_keep + 28], rtol=1e-14)     # 1-8 MeV: bins coincide
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_transform(spec)
        nll = ph.nll(_dev(u), _dev(data)).cpu().numpy()
        mu = ph.expectation(_dev(u)).cpu().numpy()
        nll_h = ph.nll_host(u, data)
    assert np.abs(nll - orc.nll(theta, data)).max() <= ABS_NLL
    assert np.array_equal(nll, nll_h)
    _check_hist(mu, orc.expectation(theta, orc.spectra(theta)))


# ---- the cheaper forms of a term where they are exact (devmath.cuh: folded / no-reduction / small-phase) ----------
# The kernel may take them only where the result is the general form's: the first term without range reduction where
# |phase| <= 1/2 half-turn for every event of a work item and every point of the group, the last term as a cubic where
# it stays below 1/8 over a dataset.  Checked here: the forms are actually reached on the Double-Chooz-like stores and
# not on the 52-km one, batches of at most 16 points (single-launch kernel) never take the first, and every one of these
# batches matches the oracle far inside the per-bin bar (a dropped parity count or constant part would be O(1)).
@pytest.mark.parametrize("k,scale,n_points", [(2, 0.05, 64), (3, 0.02, 40), (5, 0.05, 96), (4, 0.01, 64), (2, 0.05, 8)])
def test_cheaper_forms_are_reached_and_exact(gpu, oracle_mod, k, scale, n_points):
    wl = workloads.make_config(k, scale=scale, n_points=n_points)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        h = ph.spectra(_dev(wl.params)).cpu().numpy()
        med, small = ph.last_medium_phase(), ph.last_small_phase()
        h_o = orc.spectra(wl.params)
        nz = h_o != 0.0
        assert np.array_equal(h[~nz], h_o[~nz])
        assert (np.abs(h - h_o)[nz] / np.abs(h_o[nz])).max() <= 1e-10
        if k == 4:                      # 52 km: the dm2_ee phase is hundreds of radians, the solar term up to 5 rad
            assert med == 0.0 and small == 0.0
        elif n_points <= 16:            # single-launch kernel: small-phase form only
            assert med == 0.0 and small == 1.0
        else:                           # near detector fully, far detector above 4-4.5 MeV
            assert 0.25 < med < 0.9 and small == 1.0, (med, small)
        # determinism of the count and of the bits
        h2 = ph.spectra(_dev(wl.params)).cpu().numpy()
        assert np.array_equal(h, h2) and ph.last_medium_phase() == med


# ---- the single-launch kernel's edge-first unit order (api.cu build_unit_order) -----------------------------------
# The order table exists only where warps claim tickets (more than two units per warp); a cap on the warps forces
# that on small stores.  The order must change no result: bins bit-exact, spectra and NLL at the usual bars, and the
# same bits as the uncapped launch (integer accumulators: the walk order is immaterial).
@pytest.mark.parametrize("k,scale", [(2, 0.05), (3, 0.02), (4, 0.01), (5, 0.05)])
@pytest.mark.parametrize("n_points", [1, 5])
def test_edge_first_unit_order_changes_nothing(gpu, oracle_mod, k, scale, n_points):
    wl = workloads.make_config(k, scale=scale)
    params = wl.params[:n_points].copy()
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        h_free = ph.spectra(_dev(params)).cpu().numpy()
        ph.set_tuning(0, 0, 8)                              # 8 warps: every warp claims dozens of tickets
        h = ph.spectra(_dev(params)).cpu().numpy()
        nll = ph.nll(_dev(params), _dev(data)).cpu().numpy()
        bins = ph.event_bins(_dev(params)).cpu().numpy()
    assert np.array_equal(bins, orc.event_bins(params))
    _check_hist(h, orc.spectra(params))
    assert np.abs(nll - orc.nll(params, data)).max() <= ABS_NLL
    single_launch = n_points <= (16 if wl.model.osc_model == OSC_EQ1 else 4)
    if single_launch:       # the same cut into units, another walk order: the same bits
        assert np.array_equal(h, h_free)
    else:                   # the ticket schedule cuts the units by the number of warps: rounding only
        assert np.allclose(h, h_free, rtol=1e-13, atol=0.0)


def test_one_point_over_the_full_store(gpu, oracle_mod):
    """The minimiser's single evaluation at full size (config 3: 6e6 events, 11 721 units for 2 364 warps): the
    launch configuration bench.py times, order table included, against the oracle."""
    wl = workloads.make_config(3)
    params = wl.params[:1].copy()
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        h = ph.spectra(_dev(params)).cpu().numpy()
        nll = ph.nll(_dev(params), _dev(data)).cpu().numpy()
        bins = ph.event_bins(_dev(params)).cpu().numpy()
        assert ph.launch_count == 6                          # 3 calls x (single launch + finalize)
    assert np.array_equal(bins, orc.event_bins(params))
    _check_hist(h, orc.spectra(params))
    assert np.abs(nll - orc.nll(params, data)).max() <= ABS_NLL


def test_reserve_leaves_nothing_to_set_up_for_a_single_evaluation(gpu, oracle_mod):
    """phylino.h: after phylino_reserve the DEVICE entry points never synchronise -- also not the FIRST one-point call,
    which needs kernel occupancies and the single-launch kernel's unit order: captured into a CUDA graph cold (a
    synchronisation or a blocking copy inside the call would fail the capture), replayed, checked against the oracle."""
    import torch
    wl = workloads.make_config(2, scale=0.05)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    params = wl.params[:1].copy()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        ph = gpu.Phylino(stream=st.cuda_stream)
        ph.load_workload(wl)
        ph.set_tuning(0, 0, 8)                  # few warps: the unit order table is needed
        ph.reserve(4)
        dp, dd = _dev(params), _dev(data)
        out = torch.zeros(1, dtype=torch.float64, device="cuda")
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            ph.nll(dp, dd, out)                 # the first call of this context
        g.replay()
        st.synchronize()
        assert np.abs(out.cpu().numpy() - orc.nll(params, data)).max() <= ABS_NLL
    ph.close()


def test_reserve_covers_the_consumers_and_the_cached_gradient(gpu, oracle_mod):
    """phylino.h (phylino_reserve): after reserve(2 W + 1) with caching on, the FIRST calls of phylino_nll_gradient (cached
    through the structural plan, which reserve has built), phylino_nll_ensemble, phylino_draw_pseudo_data and
    phylino_variable_metric_step allocate nothing and never synchronise: all four are captured cold into one CUDA graph (an
    allocation, a synchronisation or a blocking copy inside a call would fail the capture), replayed, and checked
    against the oracle."""
    import torch
    wl = workloads.make_config(3, scale=0.01)
    N = wl.model.n_params
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    theta = wl.params[0].copy()
    h = np.array([wl.params[1 + 2 * j, j] - theta[j] for j in range(N)])
    nll_o = orc.nll(wl.params, data)
    grad_o = (nll_o[1::2] - nll_o[2::2]) / np.array([wl.params[1 + 2 * j, j] - wl.params[2 + 2 * j, j] for j in range(N)])
    mu0 = orc.expectation(theta[None, :], orc.spectra(theta[None, :]))[0]
    E = 5
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        ph = gpu.Phylino(stream=st.cuda_stream)
        ph.load_workload(wl)
        ph.set_caching(True)
        ph.reserve(2 * N + 1)
        d_theta, d_h, d_data, d_mu = _dev(theta), _dev(h), _dev(data), _dev(mu0)
        nll0 = torch.zeros(1, dtype=torch.float64, device="cuda")
        grad = torch.zeros(N, dtype=torch.float64, device="cuda")
        pseudo = torch.zeros((E, ph.total_bins), dtype=torch.float64, device="cuda")
        ens = torch.zeros((3, E), dtype=torch.float64, device="cuda")
        d_pts = _dev(wl.params[:3])
        V = _dev(np.eye(N))
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            ph.nll_gradient(d_theta, d_h, d_data, nll0, grad)           # the first calls of this context
            plan = ph.last_plan()
            ph.draw_pseudo_data(d_mu, E, seed=9, out=pseudo)
            ph.nll_ensemble(d_pts, pseudo, out=ens)
            direction, edm = ph.variable_metric_step(V, grad)
        g.replay()
        st.synchronize()
        assert plan[0] > 0                                              # cached through the structural plan
        assert abs(nll0.cpu().numpy()[0] - nll_o[0]) <= ABS_NLL
        assert np.all(np.abs(grad.cpu().numpy() - grad_o) <= 1e-6 / np.abs(h))
        want = oracle_mod.draw_pseudo_data(mu0, E, seed=9)
        assert np.array_equal(pseudo.cpu().numpy(), want)
        ens_o = np.stack([orc.nll(wl.params[:3], want[e]) for e in range(E)], axis=1)
        assert np.abs(ens.cpu().numpy() - ens_o).max() <= ABS_NLL
        assert np.array_equal(direction.cpu().numpy(), -grad.cpu().numpy())    # V = 1
    ph.close()
