"""Pins of the oracle's pseudo-experiment generator (R26): the counter-based uniforms and
the exact Poisson inversion.  Nothing here re-types the oracle's arithmetic through the oracle: Philox is held to
the published known-answer vectors and to an independent big-integer transcription of the published round function,
the sampler to the Poisson pmf (exact rationals, scipy.stats) and to goodness of fit."""
import math
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats


# Random123 known-answer vectors for philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy
# as 1, 2, 3", SC'11; the library's kat_vectors): counter, key -> output
KAT = [
    ((0x00000000,) * 4, (0x00000000,) * 2, (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
    ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
    ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
     (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)),
]


def _philox_bigint(ctr, key, rounds=10):
    """The round function as published (SC'11, section 3.3), on Python integers."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c, k = list(ctr), list(key)
    for _ in range(rounds):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xffffffff, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xffffffff]
        k = [(k[0] + W0) & 0xffffffff, (k[1] + W1) & 0xffffffff]
    return c


@pytest.mark.parametrize("ctr,key,want", KAT)
def test_philox_known_answers(oracle_mod, ctr, key, want):
    assert tuple(oracle_mod.philox4x32_10(ctr, key)) == want
    assert tuple(_philox_bigint(ctr, key)) == want


def test_philox_against_bigint_on_random_counters(oracle_mod):
    rng = np.random.default_rng(3)
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 2 ** 32, 4)]
        key = [int(x) for x in rng.integers(0, 2 ** 32, 2)]
        assert oracle_mod.philox4x32_10(ctr, key) == _philox_bigint(ctr, key)


def test_uniform53_layout_and_range(oracle_mod):
    seed = 0x299f31d0a4093822
    for b, e in ((0, 0), (5, 17), (2 ** 31, 2 ** 32 - 1)):
        x = _philox_bigint([b, e, 0, 0], [seed & 0xffffffff, seed >> 32])
        want = ((x[0] << 21) | (x[1] >> 11)) / 2.0 ** 53
        assert oracle_mod.uniform53(seed, b, e) == want and 0.0 <= want < 1.0
    u = np.array([oracle_mod.uniform53(11, b, e) for b in range(200) for e in range(200)])
    assert stats.kstest(u, "uniform").pvalue > 1e-3
    assert len(np.unique(u)) == u.size


@pytest.mark.parametrize("mu", [1e-3, 0.3, 1.0, 2.5, 7.0, 57.3, 1234.5, 98765.4])
def test_normalisation_is_the_reciprocal_pmf_at_the_mode(oracle_mod, mu):
    """Z = sum_k pmf(k) / pmf(mode) = 1 / pmf(mode) = e^mu m! / mu^m, from mpmath at 50 digits (scipy's pmf loses
    ten digits to cancellation at mu ~ 1e5)"""
    import mpmath as mp
    mp.mp.dps = 50
    m = math.floor(mu)
    want = mp.exp(mp.mpf(mu) - m * mp.log(mp.mpf(mu)) + mp.loggamma(m + 1))
    assert oracle_mod.poisson_norm(mu) == pytest.approx(float(want), rel=2e-12)


def test_normalisation_exact_rationals_small_mu(oracle_mod):
    mu = Fraction(5, 2)
    w = {2: Fraction(1)}
    for k in range(3, 80):
        w[k] = w[k - 1] * mu / k
    for k in (1, 0):
        w[k] = w[k + 1] * (k + 1) / mu
    assert oracle_mod.poisson_norm(2.5) == pytest.approx(float(sum(w.values())), rel=1e-15)


@pytest.mark.parametrize("mu", [0.3, 2.5, 57.3])
def test_inversion_pieces_have_the_pmf_as_length(oracle_mod, mu):
    """the u-interval that maps to k has length pmf(k): walk the pieces in the stated order m, m+1, m-1, ... and probe
    just inside both ends of each"""
    Z = oracle_mod.poisson_norm(mu)
    m = math.floor(mu)
    order = [m]
    for j in range(1, 40):
        order.append(m + j)
        if m - j >= 0:
            order.append(m - j)
    lo = 0.0
    for k in order:
        p = stats.poisson.pmf(k, mu)
        if p < 1e-9:
            break
        hi = lo + p
        assert oracle_mod.poisson_inv(mu, Z, lo + 1e-12) == k
        assert oracle_mod.poisson_inv(mu, Z, hi - 1e-12) == k
        lo = hi


def test_degenerate_means(oracle_mod):
    for mu in (0.0, -1.0, float("nan"), float("inf")):
        assert oracle_mod.poisson_inv(mu, oracle_mod.poisson_norm(mu), 0.7) == 0.0
    Z = oracle_mod.poisson_norm(12.0)
    assert oracle_mod.poisson_inv(12.0, Z, 0.0) == 12.0                 # the first piece is the mode
    assert oracle_mod.poisson_inv(12.0, Z, 1.0 - 2.0 ** -53) >= 0.0     # the largest u terminates


@pytest.mark.parametrize("mu", [0.3, 4.2, 57.3, 1234.5, 98765.4])
def test_sampler_goodness_of_fit(oracle_mod, mu):
    """chi^2 of 2e5 draws against scipy.stats.poisson, bins merged to >= 20 expected; plus mean and variance"""
    n = 200_000
    d = oracle_mod.draw_pseudo_data(np.array([mu]), n, seed=42)[:, 0]
    assert np.all(d == np.floor(d)) and d.min() >= 0
    lo, hi = int(stats.poisson.ppf(1e-4, mu)), int(stats.poisson.ppf(1 - 1e-4, mu))
    ks = np.arange(lo, hi + 1)
    exp = n * stats.poisson.pmf(ks, mu)
    obs = np.array([(d == k).sum() for k in ks], dtype=float) if hi - lo < 400 else \
        np.bincount(d.astype(np.int64) - lo, minlength=hi - lo + 1)[: hi - lo + 1].astype(float) if d.min() >= lo else None
    if obs is None:
        sel = (d >= lo) & (d <= hi)
        obs = np.bincount(d[sel].astype(np.int64) - lo, minlength=hi - lo + 1).astype(float)
    # tails beyond [lo, hi] into the end bins
    exp[0] += n * stats.poisson.cdf(lo - 1, mu)
    exp[-1] += n * stats.poisson.sf(hi, mu)
    obs[0] += (d < lo).sum()
    obs[-1] += (d > hi).sum()
    # merge neighbours until every expected count is >= 20
    eo, oo, ea, oa = [], [], 0.0, 0.0
    for e_, o_ in zip(exp, obs):
        ea += e_
        oa += o_
        if ea >= 20:
            eo.append(ea); oo.append(oa); ea = oa = 0.0
    if ea > 0:
        eo[-1] += ea; oo[-1] += oa
    chi2 = float(((np.array(oo) - np.array(eo)) ** 2 / np.array(eo)).sum())
    assert stats.chi2.sf(chi2, len(eo) - 1) > 1e-4, (chi2, len(eo))
    assert d.mean() == pytest.approx(mu, abs=5 * math.sqrt(mu / n))
    assert d.var() == pytest.approx(mu, rel=0.03)


def test_draws_are_a_function_of_seed_experiment_and_bin(oracle_mod):
    mu = np.array([3.0, 50.0, 3.0, 1e4])
    a = oracle_mod.draw_pseudo_data(mu, 7, seed=5)
    assert np.array_equal(a, oracle_mod.draw_pseudo_data(mu, 7, seed=5))
    assert np.array_equal(a[:3], oracle_mod.draw_pseudo_data(mu, 3, seed=5))          # experiment e does not depend on E
    assert not np.array_equal(a, oracle_mod.draw_pseudo_data(mu, 7, seed=6))
    assert not np.array_equal(a[:, 0], a[:, 2])                                        # same mu, another bin
    for e in range(7):
        for i in range(4):
            Z = oracle_mod.poisson_norm(mu[i])
            assert a[e, i] == oracle_mod.poisson_inv(mu[i], Z, oracle_mod.uniform53(5, i, e))
