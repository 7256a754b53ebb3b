"""-m gpu: on-device producers / consumers of batches: Poisson pseudo-data (bit-exact
against the oracle's generator), the ordering scan of Fig. 4, the central-difference gradient."""
import numpy as np
import pytest

import workloads
from workloads.spec import OSC_FULL3

pytestmark = pytest.mark.gpu
ABS_NLL = 1e-6


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def _data(orc, wl):
    mu0 = orc.expectation(wl.theta0[None, :], orc.spectra(wl.theta0[None, :]))[0]
    return workloads.poisson_counts(mu0, wl.seed + 7)


@pytest.mark.parametrize("k,scale,E", [(2, 0.01, 257), (3, 0.02, 64), (4, 0.01, 33), (5, 1.0, 16)])
def test_pseudo_data_bit_exact(gpu, oracle_mod, k, scale, E):
    """integer output, so the bar is bit-exact.  Expectations from tiny (scaled configs: single-event
    bins) to 1e5 per bin (config 5 at full size), drawn on the device from the ORACLE's expectation vector."""
    wl = workloads.make_config(k, scale=scale, n_points=1)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    mu = orc.expectation(wl.theta0[None, :], orc.spectra(wl.theta0[None, :]))[0]
    mu[::17] = 0.0                       # empty expectation: always 0 counts
    mu[3] = 0.37
    want = oracle_mod.draw_pseudo_data(mu, E, seed=0xC0FFEE1234567)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        got = ph.draw_pseudo_data(_dev(mu), E, seed=0xC0FFEE1234567).cpu().numpy()
        again = ph.draw_pseudo_data(_dev(mu), E, seed=0xC0FFEE1234567).cpu().numpy()
        other = ph.draw_pseudo_data(_dev(mu), E, seed=1).cpu().numpy()
    assert got.shape == want.shape == (E, mu.size)
    assert np.array_equal(got, want)
    assert np.array_equal(got, again) and not np.array_equal(got, other)
    assert np.all(got[:, ::17] == 0.0)
    big = mu > 50
    if big.any():
        assert np.abs((got[:, big] - mu[big]) / np.sqrt(mu[big])).max() < 7.0     # fluctuations of Poisson size


def test_ensemble_from_device_drawn_data(gpu, oracle_mod):
    """the whole pseudo-experiment loop on the device: expectation at the injected point -> pseudo-data -> nll[P, E]"""
    wl = workloads.make_config(5, scale=0.01, n_points=23)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    E = 19
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        mu0 = ph.expectation(_dev(wl.theta0[None, :]))
        data = ph.draw_pseudo_data(mu0[0].contiguous(), E, seed=77)
        nll = ph.nll_ensemble(_dev(wl.params), data).cpu().numpy()
        data_h, mu0_h = data.cpu().numpy(), mu0.cpu().numpy()[0]
    assert np.array_equal(data_h, oracle_mod.draw_pseudo_data(mu0_h, E, seed=77))      # same mu bits in, same counts out
    want = np.stack([orc.nll(wl.params, data_h[e]) for e in range(E)], axis=1)
    assert np.abs(nll - want).max() <= ABS_NLL


def test_ordering_scan_matches_two_models(gpu, oracle_mod):
    """PAPER.md:213, :228 (Fig. 4): dm2_ee grid x {normal, inverted}; row o of the result is the oracle's NLL of the
    model with ordering o, whatever ordering the loaded model itself carries."""
    import torch
    n_grid = 45
    for loaded in (+1, -1):
        wl = workloads.make_config(4, scale=0.004, n_points=1, ordering=loaded)
        grid = np.linspace(2.3e-3, 2.7e-3, n_grid)
        batch = np.tile(wl.theta0, (n_grid, 1))
        batch[:, 1] = grid
        orc_n = oracle_mod.Oracle(workloads.make_config(4, scale=0.004, n_points=1, ordering=+1).model, wl.events)
        orc_i = oracle_mod.Oracle(workloads.make_config(4, scale=0.004, n_points=1, ordering=-1).model, wl.events)
        data = _data(orc_n, wl)                           # injected hypothesis: normal ordering
        with gpu.Phylino() as ph:
            ph.load_workload(wl)
            nll = ph.ordering_scan(1, _dev(grid), _dev(wl.theta0), _dev(data)).cpu().numpy()
            own = ph.nll(_dev(batch), _dev(data)).cpu().numpy()       # the context's own ordering is untouched afterwards
            torch.cuda.synchronize()
        want = np.stack([orc_n.nll(batch, data), orc_i.nll(batch, data)])
        assert np.abs(nll - want).max() <= ABS_NLL
        assert np.abs(own - want[0 if loaded > 0 else 1]).max() <= ABS_NLL
        assert np.abs(want[0] - want[1]).max() > 1e-3     # the two orderings are different curves


@pytest.mark.parametrize("caching", [False, True])
def test_gradient_from_the_603_point_batch(gpu, oracle_mod, caching):
    """g_j = (nll+ - nll-) / (2 h_j) on the device against the same differences of the oracle's NLLs,
    to 1e-6 / h_j (the NLL bar divided by the step); config 3's 301 parameters at reduced event count."""
    wl = workloads.make_config(3, scale=0.01)
    N = wl.model.n_params
    assert wl.n_points == 2 * N + 1
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    theta = wl.params[0].copy()
    h = np.array([wl.params[1 + 2 * j, j] - theta[j] for j in range(N)])
    nll_o = orc.nll(wl.params, data)
    up = np.array([wl.params[1 + 2 * j, j] for j in range(N)])
    dn = np.array([wl.params[2 + 2 * j, j] for j in range(N)])
    grad_o = (nll_o[1::2] - nll_o[2::2]) / (up - dn)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(caching)
        nll0, grad = ph.nll_gradient(_dev(theta), _dev(h), _dev(data))
        if caching:
            assert ph.last_plan()[0] > 0
        nll0, grad = nll0.cpu().numpy(), grad.cpu().numpy()
    assert abs(nll0[0] - nll_o[0]) <= ABS_NLL
    assert np.all(np.abs(grad - grad_o) <= 1e-6 / np.abs(h))
    assert np.abs(grad - grad_o).max() <= 1e-3 * max(1.0, np.abs(grad_o).max())       # and tight in absolute terms


def test_cached_gradient_plans_without_the_values(gpu, oracle_mod):
    """phylino_nll_gradient with caching on takes the plan of a central-difference batch from its structure (which
    column each point perturbs), not from the values: the same 21 virtual points as the host plan of the same batch,
    the same bits, the call can be captured into a CUDA graph (nothing is copied back, nothing synchronises), and a
    step below one ulp -- structurally different, equal in value -- only loses a merge."""
    import torch
    wl = workloads.make_config(3, scale=0.01)
    N = wl.model.n_params
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    theta = wl.params[0].copy()
    h = np.array([wl.params[1 + 2 * j, j] - theta[j] for j in range(N)])
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.reserve(2 * N + 1)
        ph.set_caching(True)
        d_theta, d_h, d_data = _dev(theta), _dev(h), _dev(data)
        nll0, grad = ph.nll_gradient(d_theta, d_h, d_data)
        plan = ph.last_plan()
        # the host plan of the very same batch (values seen): same plan, same bits
        batch = np.tile(theta, (2 * N + 1, 1))
        for j in range(N):
            batch[1 + 2 * j, j] = theta[j] + h[j]
            batch[2 + 2 * j, j] = theta[j] - h[j]
        nll_host = ph.nll(_dev(batch), d_data).cpu().numpy()
        assert ph.last_plan() == plan and plan[0] == 21
        up = batch[1::2][np.arange(N), np.arange(N)]
        dn = batch[2::2][np.arange(N), np.arange(N)]
        assert np.array_equal(grad.cpu().numpy(), (nll_host[1::2] - nll_host[2::2]) / (up - dn))
        assert nll0.cpu().numpy()[0] == nll_host[0]
        # capture + replay: would fail on any synchronisation or copy back inside the call
        g = torch.cuda.CUDAGraph()
        out0 = torch.empty(1, dtype=torch.float64, device="cuda")
        outg = torch.empty(N, dtype=torch.float64, device="cuda")
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            with gpu.Phylino(stream=s.cuda_stream) as ph2:
                ph2.load_workload(wl)
                ph2.reserve(2 * N + 1)
                ph2.set_caching(True)
                ph2.nll_gradient(d_theta, d_h, d_data, out0, outg)        # warm: plan made, buffers sized
                s.synchronize()
                with torch.cuda.graph(g, stream=s):
                    ph2.nll_gradient(d_theta, d_h, d_data, out0, outg)
                outg.zero_()
                g.replay()
                s.synchronize()
                assert np.array_equal(outg.cpu().numpy(), grad.cpu().numpy())
        # a vanishing step: theta_j +- h_j == theta_j bit for bit; the structural plan keeps the points apart, the
        # values are those of the centre
        h2 = h.copy()
        h2[5] = theta[5] * 1e-20 if theta[5] != 0 else 1e-320
        nll0b, gradb = ph.nll_gradient(d_theta, _dev(h2), d_data)
        gb = gradb.cpu().numpy()
        assert np.isnan(gb[5]) or gb[5] == 0.0 or np.isinf(gb[5])       # 0 / 0 or 0 / tiny: no information, no crash
        keep = np.arange(N) != 5
        assert np.array_equal(gb[keep], grad.cpu().numpy()[keep])


def test_variable_metric_step_matches_the_oracle_bit_for_bit(gpu, oracle_mod):
    """PAPER.md:155; R30: the rank-two update of the inverse-Hessian estimate, the Newton direction and the
    estimated distance to the minimum -- every sum in index order in plain double arithmetic on both sides, so the
    comparison is bit for bit; both branches of the rule, the no-move call and the skip; then a short minimisation of
    config 3's NLL (scaled) driven by phylino_nll_gradient + this step, which must go downhill."""
    import torch
    rng = np.random.default_rng(17)
    with gpu.Phylino() as ph:
        for N, vscale in ((3, 1.0), (37, 1e-3), (301, 1.0), (301, 1e-3)):
            A = rng.normal(size=(N, N))
            V = (A @ A.T / N + np.eye(N)) * vscale
            H = rng.normal(size=(N, N))
            H = H @ H.T / N + np.eye(N)
            g = rng.normal(size=N)
            dx = rng.normal(size=N) * 0.1
            dg = H @ dx
            for use_move in (False, True):
                dV = _dev(V)
                d, edm = ph.variable_metric_step(dV, _dev(g), _dev(dx) if use_move else None, _dev(dg) if use_move else None)
                V_o, d_o, edm_o, skipped = oracle_mod.variable_metric_step(V, g, dx if use_move else None, dg if use_move else None)
                assert np.array_equal(dV.cpu().numpy(), V_o)
                assert np.array_equal(d.cpu().numpy(), d_o)
                assert edm.cpu().numpy()[0] == edm_o and edm.cpu().numpy()[1] == float(skipped) == 0.0
        dV = _dev(np.eye(4))
        d, edm = ph.variable_metric_step(dV, _dev(np.ones(4)), _dev(np.array([1.0, 0, 0, 0])), _dev(np.array([-1.0, 0, 0, 0])))
        assert edm.cpu().numpy()[1] == 1.0 and np.array_equal(dV.cpu().numpy(), np.eye(4))       # no positive curvature

    # a few steps of the loop the paper describes, on the device except for the step length
    wl = workloads.make_config(3, scale=0.01)
    N = wl.model.n_params
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = _data(orc, wl)
    sig = np.where(np.isfinite(wl.model.prior_sigma) & (wl.model.prior_sigma > 0), wl.model.prior_sigma, 1e-2)
    theta = wl.theta0 + 0.5 * sig * np.random.default_rng(4).normal(size=N)
    h = 0.01 * sig
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_caching(True)
        dV = _dev(np.diag(sig ** 2))                       # first metric: the prior covariance
        d_theta, d_h, d_data = _dev(theta), _dev(h), _dev(data)
        nll0, grad = ph.nll_gradient(d_theta, d_h, d_data)
        f = [float(nll0.cpu()[0])]
        dx = dg = None
        for it in range(4):
            d, edm = ph.variable_metric_step(dV, grad, dx, dg)
            assert float(edm.cpu()[0]) >= 0.0
            t = 1.0
            while True:                                    # backtracking: the caller's line search
                trial = d_theta + t * d
                f_t = float(ph.nll(trial[None, :].contiguous(), d_data).cpu()[0])
                if f_t < f[-1] or t < 1e-4:
                    break
                t *= 0.5
            nll1, grad1 = ph.nll_gradient(trial.contiguous(), d_h, d_data)
            dx, dg = (trial - d_theta).contiguous(), (grad1 - grad).contiguous()
            d_theta, grad = trial.contiguous(), grad1
            f.append(f_t)
        torch.cuda.synchronize()
    assert all(b < a for a, b in zip(f, f[1:])) and f[-1] < f[0] - 1.0, f
    assert abs(f[-1] - orc.nll(d_theta.cpu().numpy()[None, :], data)[0]) <= ABS_NLL


def _philox_bigint(ctr, key, rounds=10):
    """Philox4x32 round function as published (Salmon et al., SC'11, section 3.3) on Python integers -- typed here
    from the publication, shared with neither the library nor the oracle."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c, k = list(ctr), list(key)
    for _ in range(rounds):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xffffffff, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xffffffff]
        k = [(k[0] + W0) & 0xffffffff, (k[1] + W1) & 0xffffffff]
    return c


def test_device_draws_are_the_stated_function_of_the_uniforms(gpu):
    """The INDEPENDENT check of phylino_draw_pseudo_data (R26).  The oracle's sampler and the
    library's follow the same operation sequence on purpose (that is what makes the bit-exact bar of
    test_pseudo_data_bit_exact possible), so that comparison cannot find a mistake in the RULE.  This test uses neither:
    u comes from a big-integer Philox typed from the publication, the Poisson probabilities from scipy.stats, and the
    rule is R26 as stated in words -- [0, 1) is cut into pieces of length pmf(k) laid out from the mode m = floor(mu)
    outwards in the order m, m+1, m-1, m+2, m-2, ... (only upwards once 0 is passed), and the count is the piece that
    holds u.  With ring j = {m-j, ..., m+j} and F(j) = P(|X - m| <= j), the count is in the first ring with u < F(j);
    inside it m+j if u < F(j-1) + pmf(m+j), else m-j.  Every device count must be that k wherever u is farther than
    delta from a piece boundary (delta = 1e-11: the rounding of Z, 1e-13, plus scipy's cdf), and one of the two
    neighbouring pieces otherwise; >= 1e4 (bin, experiment) pairs, mu from 0.3 to 1e5 including integer mu."""
    from scipy import stats
    from workloads.spec import DatasetEvents, DatasetSpec, ModelSpec, Workload
    mu = np.concatenate([np.logspace(np.log10(0.3), 5.0, 688), [0.37, 1.0, 2.0, 2.5, 7.0, 1000.0, 99999.0, 1e5 - 0.5,
                                                                 1e-3, 0.0, 31.999999999, 32.000000001]])
    n, E, seed = mu.size, 16, 0x5EED0123456789AB
    assert n * E >= 10000
    edges = np.linspace(1.0, 8.0, n + 1)
    model = ModelSpec(osc_model=0, n_params=4, idx_osc=(0, 1, 2, 3, -1, -1), fixed_osc=(0,) * 6,
                      datasets=[DatasetSpec(n_bins=n)])
    ev = DatasetEvents(e_nu=np.zeros(0, np.float32), e_vis=np.zeros(0, np.float32), w=np.zeros(0, np.float32),
                       core=np.zeros(0, np.int32), L_m=np.array([1050.0]), edges=edges)
    theta = np.array([[0.1, 2.5e-3, 0.85, 7.5e-5]])
    with gpu.Phylino() as ph:
        ph.load_workload(Workload("draw", model, [ev], theta, theta[0], 1))
        got = ph.draw_pseudo_data(_dev(mu), E, seed=seed).cpu().numpy()
    assert got.shape == (E, n)
    key = [seed & 0xffffffff, seed >> 32]
    delta, exact, near = 1e-11, 0, 0
    for i in range(n):
        if not mu[i] > 0.0:
            assert np.all(got[:, i] == 0.0)
            continue
        m = int(np.floor(mu[i]))
        J = int(12 * np.sqrt(mu[i]) + 40)
        j = np.arange(J + 1)
        hi = stats.poisson.cdf(m + j, mu[i])
        lo = np.where(m - j - 1 >= 0, stats.poisson.cdf(m - j - 1, mu[i]), 0.0)
        F = hi - lo                                               # mass of rings 0 ... j
        for e in range(E):
            x = _philox_bigint([i, e, 0, 0], key)
            u = ((x[0] << 21) | (x[1] >> 11)) / 2.0 ** 53
            ring = int(np.searchsorted(F, u, side="right"))
            assert ring <= J, (mu[i], u)
            if ring == 0:
                want, bounds = m, (F[0],)
            else:
                cut = F[ring - 1] + stats.poisson.pmf(m + ring, mu[i])
                want = m + ring if (u < cut or m - ring < 0) else m - ring
                bounds = (F[ring - 1], cut, F[ring])
            k = got[e, i]
            assert k == np.floor(k) and k >= 0
            if min(abs(u - b) for b in bounds) > delta:
                assert k == want, (mu[i], e, u, k, want)
                exact += 1
            else:
                assert abs(abs(k - m) - ring) <= 1, (mu[i], e, u, k, want)
                near += 1
    assert exact >= 10000 and near <= 5, (exact, near)
    # outside the domain (R26): a finite mu above 1e9 gives NaN, promptly
    with gpu.Phylino() as ph:
        ph.load_workload(Workload("draw", model, [ev], theta, theta[0], 1))
        wild = np.full(n, 3.0)
        wild[:4] = [2e9, 1e15, 1e300, np.inf]
        out = ph.draw_pseudo_data(_dev(wild), 2, seed=1).cpu().numpy()
    assert np.isnan(out[:, :3]).all() and np.all(out[:, 3] == 0.0) and np.all(out[:, 4:] >= 0.0)
