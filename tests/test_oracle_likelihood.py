"""Pins for oracle steps O4 (expectation assembly) and O5 (Poisson half-deviance + Gaussian priors).

PAPER.md:67-76 (Eq. 3-5), :80-83 (Eq. 6), :96 (Eq. 8, saturated model), :105-107 (signal + backgrounds),
:119-125 (Eq. 9); R9 (normalisation), R10 (n = 0, mu <= 0).
"""
import math

import numpy as np
import pytest
from scipy.special import gammaln

import workloads as W
from workloads.spec import OSC_EQ1, BkgSpec, DatasetSpec, ModelSpec


def _logpmf(n, mu):
    """ln of PAPER.md:67 Eq. 3 through the library log-gamma: n ln mu - mu - ln n!"""
    return n * math.log(mu) - mu - float(gammaln(n + 1.0))


def test_dev_is_poisson_log_likelihood_ratio(oracle_mod):
    """dev(n, mu) == [-ln pmf(n; mu)] - [-ln pmf(n; n)]  (Eq. 3 against the saturated model of Eq. 8)."""
    rng = np.random.default_rng(0)
    for _ in range(500):
        mu = float(rng.uniform(0.05, 3e4))
        n = float(rng.poisson(mu))
        want = -_logpmf(n, mu) + (_logpmf(n, n) if n > 0 else 0.0)
        got = oracle_mod.dev(n, mu)
        assert abs(got - want) <= 1e-9 * max(1.0, abs(_logpmf(n, mu))), (n, mu)   # lgamma cancellation
        assert got >= 0.0


def test_dev_special_values(oracle_mod):
    d = oracle_mod.dev
    assert d(7.0, 7.0) == 0.0 and d(0.0, 0.0) == 0.0       # deviance zero when data == expectation
    assert d(0.0, 2.5) == 2.5                                # n = 0  =>  mu
    assert d(3.0, 0.0) == math.inf and d(3.0, -1.0) == math.inf and d(0.0, -1.0) == math.inf
    assert math.isnan(d(float("nan"), 1.0)) and math.isnan(d(1.0, float("nan")))
    assert math.isnan(d(-1.0, 1.0))
    # second-order behaviour: dev ~ (n-mu)^2 / (2 mu) near the minimum (Wilks' chi^2 / 2)
    assert d(10_000.0, 10_010.0) == pytest.approx(100.0 / (2 * 10_005.0), rel=1e-3)


def _toy_model():
    # theta = (eps, f0, f1, r, s0, s1, unused)
    ds = DatasetSpec(n_bins=2, idx_signorm=0, norm=0.5, idx_flux=np.array([1, 2], np.int32),
                     bkg=[BkgSpec(tmpl=np.array([3.0, 5.0]), idx_rate=3, idx_shape=np.array([4, 5], np.int32)),
                          BkgSpec(tmpl=np.array([0.25, 0.5]))])
    return ModelSpec(osc_model=OSC_EQ1, n_params=7, idx_osc=(-1,) * 6, fixed_osc=(0,) * 6, datasets=[ds],
                     prior_mean=np.array([1.0, 1.0, 1.0, 1.0, 1.0, 1.0, 0.0]),
                     prior_sigma=np.array([0.1, 0.02, 0.02, 0.0, 0.05, np.inf, 0.3]))


def test_expectation_closed_form_and_linearity(oracle_mod):
    """mu = eps*norm*f_b*H_b + r*s_b*T_b + T'_b on a 2-bin, 2-background toy."""
    o = oracle_mod.Oracle(_toy_model())
    th = np.array([1.1, 0.9, 1.2, 2.0, 0.5, 1.5, 0.0])
    H = np.array([[100.0, 40.0]])
    mu = o.expectation(th, H)[0]
    assert mu[0] == pytest.approx(1.1 * 0.5 * 0.9 * 100 + 2.0 * 0.5 * 3.0 + 0.25, rel=1e-15)
    assert mu[1] == pytest.approx(1.1 * 0.5 * 1.2 * 40 + 2.0 * 1.5 * 5.0 + 0.5, rel=1e-15)
    for j in range(6):                       # linear in every multiplier
        e = np.zeros(7)
        e[j] = 0.37
        m0, m1, m2 = (o.expectation(th + k * e, H)[0] for k in (0, 1, 2))
        assert np.allclose(m2 - m1, m1 - m0, rtol=1e-12, atol=1e-12)
    assert np.array_equal(o.expectation(th + np.array([0, 0, 0, 0, 0, 0, 5.0]), H)[0], mu)


def test_priors_closed_form(oracle_mod):
    """1/2 sum ((theta-mean)/sigma)^2 over sigma finite > 0; sigma = 0 / inf => unconstrained."""
    o = oracle_mod.Oracle(_toy_model())
    th = np.array([1.05, 1.01, 0.97, 9.0, 1.1, 77.0, 0.3])
    mu = np.array([[4.0, 6.0]])
    nll = o.nll_from_mu(th, mu, np.array([4.0, 6.0]))[0]
    want = 0.5 * ((0.05 / 0.1) ** 2 + (0.01 / 0.02) ** 2 + (0.03 / 0.02) ** 2 + (0.1 / 0.05) ** 2 + (0.3 / 0.3) ** 2)
    assert nll == pytest.approx(want, rel=1e-13)


def test_nll_zero_at_saturation(oracle_mod):
    """north_star pin: NLL == 0 when data == expectation and theta == prior centres."""
    wl = W.make_tiny(seed=3, n_points=1)
    o = oracle_mod.Oracle(wl.model, wl.events)
    mu = o.expectation(wl.theta0, o.spectra(wl.theta0))
    assert o.nll(wl.theta0, mu[0])[0] == 0.0
    assert o.nll_from_mu(wl.theta0, mu, mu[0])[0] == 0.0


def test_nll_is_sum_of_bins_and_priors(oracle_mod):
    wl = W.make_tiny(seed=4, n_points=6, n_datasets=2)
    o = oracle_mod.Oracle(wl.model, wl.events)
    mu = o.expectation(wl.params, o.spectra(wl.params))
    data = W.poisson_counts(mu[0], 9)
    got = o.nll(wl.params, data)
    ps, pm = wl.model.prior_sigma, wl.model.prior_mean
    for p in range(wl.n_points):
        s = math.fsum(-_logpmf(n, m) + (_logpmf(n, n) if n > 0 else 0.0) for n, m in zip(data, mu[p]))
        s += math.fsum(0.5 * ((wl.params[p, j] - pm[j]) / ps[j]) ** 2 for j in range(len(ps)) if ps[j] > 0)
        assert got[p] == pytest.approx(s, rel=1e-10, abs=1e-10)


def test_gradient_wrt_shape_parameter(oracle_mod):
    """d nll / d s = sum_b (1 - n/mu) d mu/d s + (s - mean)/sigma^2, against a central difference
    taken from a batch of points — the use the paper makes of the batch."""
    wl = W.make_tiny(seed=5, n_points=1)
    o = oracle_mod.Oracle(wl.model, wl.events)
    th = wl.theta0.copy()
    th[-3] = 1.04                                         # one shared Li-like shape parameter (bin 4)
    j = len(th) - 3
    mu = o.expectation(th, o.spectra(th))[0]
    data = W.poisson_counts(mu, 1)
    h = 1e-5
    batch = np.stack([th, th, th])
    batch[1, j] += h
    batch[2, j] -= h
    nll = o.nll(batch, data)
    num = (nll[1] - nll[2]) / (2 * h)
    b = 4
    r = th[wl.model.datasets[0].bkg[0].idx_rate]
    dmu = r * wl.model.datasets[0].bkg[0].tmpl[b]
    ana = (1 - data[b] / mu[b]) * dmu + (th[j] - wl.model.prior_mean[j]) / wl.model.prior_sigma[j] ** 2
    assert num == pytest.approx(ana, rel=1e-6)


def test_infinite_and_nan_bins_propagate(oracle_mod):
    o = oracle_mod.Oracle(_toy_model())
    th = np.array([1.0, 1.0, 1.0, 1.0, 1.0, 1.0, 0.0])
    assert o.nll_from_mu(th, np.array([[0.0, 6.0]]), np.array([2.0, 6.0]))[0] == math.inf
    assert math.isnan(o.nll_from_mu(th, np.array([[np.nan, 6.0]]), np.array([2.0, 6.0]))[0])
