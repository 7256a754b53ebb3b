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


# ---- correlated prior blocks (third factor of Eq. 9) ---------------------

def _toy_with_blocks(blocks, sigma=None):
    m = _toy_model()
    m.prior_sigma = np.zeros(7) if sigma is None else sigma      # diagonal priors off unless asked for
    m.prior_blocks = blocks
    return m


def test_prior_block_diagonal_reduces_to_uncorrelated_gaussians(oracle_mod):
    """V = diag(sigma^2): the block term is the plain sum of 1/2 z^2 (the routine pinned above)."""
    sig = np.array([0.1, 0.02, 0.02, 0.0, 0.05, np.inf, 0.3])
    idx = np.array([0, 1, 2, 4, 6], np.int32)
    mean = _toy_model().prior_mean
    blk = W.PriorBlock(idx=idx, mean=mean[idx], inv_cov=np.diag(1.0 / sig[idx] ** 2))
    a = oracle_mod.Oracle(_toy_model())                           # diagonal priors
    b = oracle_mod.Oracle(_toy_with_blocks([blk]))                # the same constraint as one block
    rng = np.random.default_rng(5)
    mu, n = np.array([[4.0, 6.0]]), np.array([3.0, 9.0])
    for _ in range(20):
        th = mean + rng.normal(0, 0.1, 7)
        assert b.nll_from_mu(th, mu, n)[0] == pytest.approx(a.nll_from_mu(th, mu, n)[0], rel=1e-13)


def test_prior_block_bivariate_closed_form(oracle_mod):
    """2 x 2 block: q = (z1^2 - 2 rho z1 z2 + z2^2) / (1 - rho^2), the textbook bivariate normal exponent."""
    s1, s2, rho = 0.03, 0.2, -0.6
    V = np.array([[s1 * s1, rho * s1 * s2], [rho * s1 * s2, s2 * s2]])
    blk = W.PriorBlock(idx=np.array([4, 1], np.int32), mean=np.array([1.0, 0.9]), inv_cov=np.linalg.inv(V))
    o = oracle_mod.Oracle(_toy_with_blocks([blk]))
    th = np.array([1.0, 0.95, 1.0, 1.0, 1.04, 1.0, 0.0])
    z1, z2 = (1.04 - 1.0) / s1, (0.95 - 0.9) / s2
    want = 0.5 * (z1 * z1 - 2 * rho * z1 * z2 + z2 * z2) / (1 - rho * rho)
    got = o.nll_from_mu(th, np.array([[4.0, 6.0]]), np.array([4.0, 6.0]))[0]
    assert got == pytest.approx(want, rel=1e-12)


def test_prior_blocks_against_scipy_multivariate_normal(oracle_mod):
    """nll(theta) - nll(b0) = -[ln N(theta; b0, V) - ln N(b0; b0, V)] for two blocks of size 3 and 41."""
    from scipy.stats import multivariate_normal
    rng = np.random.default_rng(11)
    n_par = 50
    ds = DatasetSpec(n_bins=2, norm=1.0)
    A3, A41 = rng.normal(size=(3, 3)), rng.normal(size=(41, 41))
    V3, V41 = A3 @ A3.T + 0.5 * np.eye(3), A41 @ A41.T / 41 + 0.2 * np.eye(41)   # the paper's 41 x 41 flux block size
    i3 = np.array([47, 2, 45], np.int32)
    i41 = np.arange(3, 44, dtype=np.int32)
    m3, m41 = rng.normal(size=3), rng.normal(size=41)
    model = ModelSpec(osc_model=OSC_EQ1, n_params=n_par, idx_osc=(-1,) * 6, fixed_osc=(0,) * 6, datasets=[ds],
                      prior_blocks=[W.PriorBlock(i3, m3, np.linalg.inv(V3)), W.PriorBlock(i41, m41, np.linalg.inv(V41))])
    o = oracle_mod.Oracle(model)
    mu, n = np.array([[4.0, 6.0]]), np.array([4.0, 6.0])
    th0 = np.zeros(n_par)
    th0[i3], th0[i41] = m3, m41
    assert o.nll_from_mu(th0, mu, n)[0] == 0.0
    for _ in range(10):
        th = th0 + rng.normal(0, 0.3, n_par)
        want = -(multivariate_normal(m3, V3).logpdf(th[i3]) - multivariate_normal(m3, V3).logpdf(m3)) \
               - (multivariate_normal(m41, V41).logpdf(th[i41]) - multivariate_normal(m41, V41).logpdf(m41))
        assert o.nll_from_mu(th, mu, n)[0] == pytest.approx(want, rel=1e-9)


def test_prior_block_order_and_asymmetry(oracle_mod):
    """Relabelling the parameters of a block (with the matrix permuted alike) changes nothing; an
    unsymmetrised matrix M counts as (M + M^T)/2 -- the double sum is taken as written."""
    rng = np.random.default_rng(3)
    M = rng.normal(size=(4, 4))
    idx, mean = np.array([0, 2, 4, 5], np.int32), rng.normal(size=4)
    perm = np.array([2, 0, 3, 1])
    th = rng.normal(size=7)
    mu, n = np.array([[4.0, 6.0]]), np.array([4.0, 6.0])
    f = lambda blk: oracle_mod.Oracle(_toy_with_blocks([blk])).nll_from_mu(th, mu, n)[0]
    base = f(W.PriorBlock(idx, mean, M))
    assert f(W.PriorBlock(idx[perm], mean[perm], M[np.ix_(perm, perm)])) == pytest.approx(base, rel=1e-12, abs=1e-14)
    assert f(W.PriorBlock(idx, mean, 0.5 * (M + M.T))) == pytest.approx(base, rel=1e-12, abs=1e-14)


# ---- constrained FUNCTIONS of the fitted parameters ("b_i(theta) are functions of the actually fitted
# nuisance parameters"; R29: polynomials with integer powers; a block reaches function f as n_params + f) --

def _fn(terms, offset=0.0):
    return W.FunctionSpec(terms=[(c, np.array(i, np.int32), np.array(p, np.int32)) for c, i, p in terms], offset=offset)


def _toy_with_functions(functions, blocks):
    m = _toy_with_blocks(blocks)
    m.functions = functions
    return m


def test_function_value_exact_rationals(oracle_mod):
    """b = 3/4 - 5/2 th1^2 th4 + 7 th2^-3 + 1/8 th0 th1^-1 th6^2 on dyadic arguments: every product and sum is exact
    in binary floating point, so the result must equal the rational arithmetic bit for bit -- a wrong power, a
    dropped factor, a swapped index or a sign all show."""
    from fractions import Fraction as F
    th = np.array([1.5, -0.75, 2.0, 9.0, 0.625, 3.0, -4.0])
    f = _fn([(-2.5, [1, 4], [2, 1]), (7.0, [2], [-3]), (0.125, [0, 1, 6], [1, -1, 2]), (11.0, [3], [0])], offset=0.75)
    t = [F(x) for x in th]
    want = F(3, 4) - F(5, 2) * t[1] ** 2 * t[4] + F(7) / t[2] ** 3 + F(1, 8) * t[0] / t[1] * t[6] ** 2 + 11
    o = oracle_mod.Oracle(_toy_with_functions([f], []))
    assert o.function_values(th)[0] == float(want)


def test_function_identity_is_the_raw_parameter_prior(oracle_mod):
    """b(theta) = theta_j: a block over functions must give exactly what the same block over the parameters gives."""
    s1, s2, rho = 0.03, 0.2, -0.6
    Vi = np.linalg.inv(np.array([[s1 * s1, rho * s1 * s2], [rho * s1 * s2, s2 * s2]]))
    mean = np.array([1.0, 0.9])
    raw = W.PriorBlock(idx=np.array([4, 1], np.int32), mean=mean, inv_cov=Vi)
    fns = [_fn([(1.0, [4], [1])]), _fn([(1.0, [1], [1])])]
    via = W.PriorBlock(idx=np.array([7 + 0, 7 + 1], np.int32), mean=mean, inv_cov=Vi)
    a = oracle_mod.Oracle(_toy_with_blocks([raw]))
    b = oracle_mod.Oracle(_toy_with_functions(fns, [via]))
    rng = np.random.default_rng(11)
    mu, n = np.array([[4.0, 6.0]]), np.array([3.0, 9.0])
    for _ in range(20):
        th = _toy_model().prior_mean + rng.normal(0, 0.1, 7)
        assert b.nll_from_mu(th, mu, n)[0] == a.nll_from_mu(th, mu, n)[0]


def test_function_priors_against_mpmath(oracle_mod):
    """A Gaussian constraint on a product over a ratio, b = th0 th4 / th2, and a correlated pair (b, c) with
    c = 2 th1 - th5^2 + 1/2, typed here from Eq. 6 / Eq. 9 with 50 digits."""
    import mpmath as mp
    mp.mp.dps = 50
    fb = _fn([(1.0, [0, 4, 2], [1, 1, -1])])
    fc = _fn([(2.0, [1], [1]), (-1.0, [5], [2])], offset=0.5)
    sb = 0.07
    s1, s2, rho = 0.05, 0.3, 0.4
    V = np.array([[s1 * s1, rho * s1 * s2], [rho * s1 * s2, s2 * s2]])
    blocks = [W.PriorBlock(idx=np.array([7], np.int32), mean=np.array([1.1]), inv_cov=np.array([[1.0 / sb ** 2]])),
              W.PriorBlock(idx=np.array([7, 8], np.int32), mean=np.array([1.0, 1.4]), inv_cov=np.linalg.inv(V))]
    o = oracle_mod.Oracle(_toy_with_functions([fb, fc], blocks))
    rng = np.random.default_rng(3)
    for _ in range(10):
        th = np.array([1.0, 0.95, 1.0, 1.0, 1.04, 1.0, 0.0]) + rng.normal(0, 0.05, 7)
        t = [mp.mpf(float(x)) for x in th]
        b = t[0] * t[4] / t[2]
        c = 2 * t[1] - t[5] ** 2 + mp.mpf("0.5")
        Vi = mp.matrix(np.linalg.inv(V).tolist())
        d = mp.matrix([b - 1, c - mp.mpf("1.4")])
        want = ((b - mp.mpf("1.1")) / mp.mpf(sb)) ** 2 / 2 + (d.T * Vi * d)[0] / 2
        got = o.nll_from_mu(th, np.array([[4.0, 6.0]]), np.array([4.0, 6.0]))[0]
        assert got == pytest.approx(float(want), rel=1e-12)


def test_function_prior_gradient(oracle_mod):
    """d/d theta_k of 1/2 ((b - b0)/sigma)^2 = (b - b0)/sigma^2 db/dtheta_k with db/dtheta by hand, against a central
    difference of the oracle."""
    f = _fn([(3.0, [0, 4], [2, 1]), (-1.0, [2], [-1])], offset=0.2)          # b = 3 th0^2 th4 - 1/th2 + 0.2
    b0, sg = 2.0, 0.5
    blk = W.PriorBlock(idx=np.array([7], np.int32), mean=np.array([b0]), inv_cov=np.array([[1.0 / sg ** 2]]))
    o = oracle_mod.Oracle(_toy_with_functions([f], [blk]))
    th = np.array([0.9, 1.0, 1.3, 1.0, 0.8, 1.0, 0.0])
    mu, n = np.array([[4.0, 6.0]]), np.array([4.0, 6.0])
    b = 3 * th[0] ** 2 * th[4] - 1 / th[2] + 0.2
    grad = {0: 6 * th[0] * th[4], 4: 3 * th[0] ** 2, 2: 1 / th[2] ** 2, 1: 0.0}
    for k, db in grad.items():
        h = 1e-6
        up, dn = th.copy(), th.copy()
        up[k] += h
        dn[k] -= h
        num = (o.nll_from_mu(up, mu, n)[0] - o.nll_from_mu(dn, mu, n)[0]) / (2 * h)
        assert num == pytest.approx((b - b0) / sg ** 2 * db, rel=1e-6, abs=1e-7)
