"""Pins for oracle steps O1-O2 (amplitudes, splittings) and the scalar P_ee.

Each pin is something the paper or the mathematics fixes, computed here WITHOUT the oracle
(mpmath at 50 digits from the angles themselves, PMNS textbook form, algebraic identities).
PAPER.md:34 (Eq. 1), :39 (Eq. 2), :219-226 (Eq. 10), BASELINE.json config 5 (3+1 formula).
"""
import itertools

import mpmath as mp
import numpy as np
import pytest

import workloads as W
from workloads.spec import OSC_EQ1, OSC_FULL3, OSC_STERILE4, ModelSpec, DatasetSpec
from helpers import K, angles, pee_eq1_mp, pee_full3_mp, pee_eq10_repaired_mp


def _model(osc, ordering=+1):
    return ModelSpec(osc_model=osc, ordering=ordering, n_params=6, idx_osc=(0, 1, 2, 3, 4, 5),
                     fixed_osc=(0,) * 6, datasets=[DatasetSpec(n_bins=1)])


def _pee(oracle_mod, osc, theta, L, E, ordering=+1):
    A, m = oracle_mod.Oracle(_model(osc, ordering)).terms(np.asarray(theta, dtype=np.float64))
    return oracle_mod.pee(A, m, L, E), A, m


GRID = list(itertools.product([0.0, 0.05, 0.1, 0.15], [2.3e-3, 2.5e-3], [0.0, 0.8, 0.85, 0.9],
                              [7.0e-5, 7.5e-5], [355.0, 1050.0, 52_500.0], [1.8, 3.8, 7.3]))


def test_eq1_against_mpmath_from_angles(oracle_mod):
    """PAPER.md:34 Eq. 1 with cos^4(theta13) from the angle, not from the oracle's half-angle algebra."""
    worst = 0.0
    for s13, mee, s12, m21, L, E in GRID:
        got, _, _ = _pee(oracle_mod, OSC_EQ1, [s13, mee, s12, m21, 0, 0], L, E)
        want = pee_eq1_mp(s13, mee, s12, m21, L, E)
        worst = max(worst, abs(float(got - want)))
    assert worst < 5e-14, worst          # fp64 phase rounding at 52.5 km: ~45 rad * 1e-16 * amplitude


def test_full3_against_pmns_textbook(oracle_mod):
    """Exact 3-flavour vacuum P_ee from |U_ei|^2; both orderings (R2, R5)."""
    worst = 0.0
    for ordering in (+1, -1):
        for s13, mee, s12, m21, L, E in GRID:
            got, _, _ = _pee(oracle_mod, OSC_FULL3, [s13, mee, s12, m21, 0, 0], L, E, ordering)
            want = pee_full3_mp(s13, mee, s12, m21, L, E, ordering)
            worst = max(worst, abs(float(got - want)))
    assert worst < 5e-14, worst


def test_full3_equals_repaired_eq10(oracle_mod):
    """PAPER.md:219-226 Eq. 10 (repaired, R2) is an identity of the exact formula."""
    worst = 0.0
    rng = np.random.default_rng(5)
    for ordering in (+1, -1):
        for _ in range(200):
            s13, s12 = rng.uniform(0.02, 0.2), rng.uniform(0.7, 0.95)
            mee, m21 = rng.uniform(2.2e-3, 2.8e-3), rng.uniform(6e-5, 9e-5)
            L, E = rng.choice([400.0, 52_500.0, 53_000.0, 215_000.0]), rng.uniform(1.8, 10.0)
            got, _, _ = _pee(oracle_mod, OSC_FULL3, [s13, mee, s12, m21, 0, 0], L, E, ordering)
            want = pee_eq10_repaired_mp(s13, mee, s12, m21, L, E, ordering)
            worst = max(worst, abs(float(got - want)))
    assert worst < 1e-12, worst


def test_ordering_changes_full3(oracle_mod):
    """Normal and inverted ordering must differ at medium baseline — guards against
    an ordering flag that is silently ignored."""
    th = [0.1, 2.5e-3, 0.85, 7.5e-5, 0, 0]
    pn, _, _ = _pee(oracle_mod, OSC_FULL3, th, 52_500.0, 3.0, +1)
    pi, _, _ = _pee(oracle_mod, OSC_FULL3, th, 52_500.0, 3.0, -1)
    assert abs(pn - pi) > 1e-3


def test_eq2_round_trip(oracle_mod):
    """PAPER.md:39 Eq. 2: cos^2(th12)|dm31| + sin^2(th12)|dm32| == dm_ee; |dm31 - dm32| == dm21."""
    for ordering in (+1, -1):
        for s12 in (0.3, 0.85, 0.99):
            _, A, m = _pee(oracle_mod, OSC_FULL3, [0.1, 2.5e-3, s12, 7.5e-5, 0, 0], 1.0, 1.0, ordering)
            t12 = angles(s12)
            mee = mp.cos(t12) ** 2 * m[1] + mp.sin(t12) ** 2 * m[2]
            assert abs(float(mee) - 2.5e-3) < 1e-17
            assert abs((m[1] - m[2]) - ordering * 7.5e-5) < 1e-18
            assert m[0] == 7.5e-5
            # amplitudes: the two atmospheric terms share sin^2(2th13) in the ratio cos^2 : sin^2
            assert abs(A[1] + A[2] - 0.1) < 1e-16
            assert abs(A[1] / A[2] - float(mp.cos(t12) ** 2 / mp.sin(t12) ** 2)) < 1e-12


def test_sterile4_against_mpmath(oracle_mod):
    """BASELINE.json config 5: 1 - c14^4 s13 sin^2 Dee - s14 sin^2 D41 - c13^4 s12 sin^2 D21."""
    worst = 0.0
    for s14, m41 in itertools.product([1e-3, 0.05, 0.3], [1e-2, 0.3, 10.0]):
        for L, E in [(355.0, 2.0), (1115.0, 3.8), (998.0, 9.0)]:
            s13, mee, s12, m21 = 0.1, 2.5e-3, 0.85, 7.5e-5
            got, _, _ = _pee(oracle_mod, OSC_STERILE4, [s13, mee, s12, m21, s14, m41], L, E)
            t13, t14 = angles(s13), angles(s14)
            x = mp.mpf(L) / mp.mpf(E)
            want = (1 - mp.cos(t14) ** 4 * mp.mpf(s13) * mp.sin(K * mp.mpf(mee) * x) ** 2
                    - mp.mpf(s14) * mp.sin(K * mp.mpf(m41) * x) ** 2
                    - mp.cos(t13) ** 4 * mp.mpf(s12) * mp.sin(K * mp.mpf(m21) * x) ** 2)
            worst = max(worst, abs(float(got - want)))
    # phase up to 1.267*10*1115/3.8 = 3.7e3 rad: fp64 phase rounding 4e-13 * amplitude 0.3
    assert worst < 5e-13, worst


def test_special_cases_exact(oracle_mod):
    """north_star pins: P == 1 at theta13 = theta12 = 0, at dm2 = 0, at L = 0 (exactly)."""
    for osc in (OSC_EQ1, OSC_FULL3, OSC_STERILE4):
        p, _, _ = _pee(oracle_mod, osc, [0.0, 2.5e-3, 0.0, 7.5e-5, 0.0, 1.0], 1050.0, 3.8)
        assert p == 1.0
        p, _, _ = _pee(oracle_mod, osc, [0.1, 0.0, 0.85, 0.0, 0.05, 0.0], 1050.0, 3.8)
        assert p == 1.0
        p, _, _ = _pee(oracle_mod, osc, [0.1, 2.5e-3, 0.85, 7.5e-5, 0.05, 1.0], 0.0, 3.8)
        assert p == 1.0


def test_model_reductions(oracle_mod):
    """STERILE4 at s14 = 0 == EQ1;  FULL3 at dm21 = 0 == EQ1 without its solar term."""
    rng = np.random.default_rng(11)
    for _ in range(50):
        s13, s12 = rng.uniform(0, 0.2), rng.uniform(0.5, 0.95)
        mee, m21 = rng.uniform(2e-3, 3e-3), rng.uniform(6e-5, 9e-5)
        L, E = rng.uniform(300, 1200), rng.uniform(1.8, 10)
        p1, _, _ = _pee(oracle_mod, OSC_EQ1, [s13, mee, s12, m21, 0, 0], L, E)
        p4, _, _ = _pee(oracle_mod, OSC_STERILE4, [s13, mee, s12, m21, 0.0, 0.7], L, E)
        assert abs(p1 - p4) < 2e-16
        p3, _, _ = _pee(oracle_mod, OSC_FULL3, [s13, mee, s12, 0.0, 0, 0], L, E)
        p1b, _, _ = _pee(oracle_mod, OSC_EQ1, [s13, mee, 0.0, m21, 0, 0], L, E)
        assert abs(p3 - p1b) < 1e-15


def test_eq1_close_to_full3_at_short_baseline(oracle_mod):
    """'in good approximation': |FULL3 - EQ1| stays below 6e-5 for L <= 1115 m."""
    worst = 0.0
    for L in (355.0, 469.0, 998.0, 1050.0, 1115.0):
        for E in np.linspace(1.8, 10.0, 200):
            th = [0.1, 2.5e-3, 0.85, 7.5e-5, 0, 0]
            a, _, _ = _pee(oracle_mod, OSC_EQ1, th, L, E)
            b, _, _ = _pee(oracle_mod, OSC_FULL3, th, L, E)
            worst = max(worst, abs(a - b))
    assert 1e-6 < worst < 6e-5, worst


def test_probability_range(oracle_mod):
    """0 <= P <= 1: always for FULL3; for Eq. 1 inside s13 <= 0.15, s12 <= 0.9 (R19)."""
    rng = np.random.default_rng(3)
    for _ in range(2000):
        s13, s12 = rng.uniform(0, 1), rng.uniform(0, 1)
        mee, m21 = rng.uniform(1e-3, 5e-3), rng.uniform(1e-5, 2e-4)
        L, E = rng.uniform(100, 3e5), rng.uniform(1.8, 10)
        p, _, _ = _pee(oracle_mod, OSC_FULL3, [s13, mee, s12, m21, 0, 0], L, E, rng.choice([-1, 1]))
        assert -1e-15 <= p <= 1.0
        p, _, _ = _pee(oracle_mod, OSC_EQ1, [0.15 * s13, mee, 0.9 * s12, m21, 0, 0], L, E)
        assert 0.0 <= p <= 1.0


def test_fixed_vs_indexed_parameters(oracle_mod):
    """idx_osc = -1 takes fixed_osc: same terms as reading the value from theta."""
    m_idx = _model(OSC_STERILE4)
    vals = (0.09, 2.4e-3, 0.8, 7.2e-5, 0.02, 0.4)
    m_fix = ModelSpec(osc_model=OSC_STERILE4, n_params=6, idx_osc=(-1,) * 6, fixed_osc=vals,
                      datasets=[DatasetSpec(n_bins=1)])
    A1, d1 = oracle_mod.Oracle(m_idx).terms(np.array(vals))
    A2, d2 = oracle_mod.Oracle(m_fix).terms(np.zeros(6))
    assert np.array_equal(A1, A2) and np.array_equal(d1, d2)
