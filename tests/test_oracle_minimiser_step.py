"""Pins of the oracle's variable-metric step (the minimiser's loop; R30: the paper prints no
formula, the update taken is Davidon-Fletcher-Powell plus the rank-one term that makes it BFGS where dx.dg > dg.V dg).

None of these re-types the oracle's update through the oracle: they are properties every correct rank-two
variable-metric update has, and a quadratic on which the exact answer is known."""
from fractions import Fraction as F

import numpy as np
import pytest

pytestmark = pytest.mark.filterwarnings("ignore")


def _spd(rng, n, cond=30.0):
    q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    return (q * np.geomspace(1.0, cond, n)) @ q.T


def test_direction_and_edm_are_the_plain_definitions(oracle_mod):
    rng = np.random.default_rng(1)
    V = _spd(rng, 7)
    g = rng.normal(size=7)
    V2, d, edm, skipped = oracle_mod.variable_metric_step(V, g)
    assert not skipped and np.array_equal(V2, V)                   # no move given: the metric is untouched
    assert np.allclose(d, -V @ g, rtol=1e-14, atol=0) and edm == pytest.approx(0.5 * g @ V @ g, rel=1e-14)


def test_secant_equation_symmetry_and_positive_definiteness(oracle_mod):
    """Every update of the Broyden family maps the last gradient change onto the last move, V' dg = dx, stays symmetric
    and (for dx.dg > 0) positive definite -- both branches of the rule (a > b: BFGS term on; a <= b: DFP alone)."""
    rng = np.random.default_rng(2)
    seen = set()
    for trial in range(40):
        n = int(rng.integers(2, 9))
        V = _spd(rng, n) * (1e-3 if trial % 4 < 2 else 1.0)        # a small metric makes dx.dg exceed dg.V dg
        A = _spd(rng, n)                                            # the true Hessian of a quadratic
        dx = rng.normal(size=n) * (0.2 if trial % 2 else 3.0)
        dg = A @ dx                                                 # its gradient change along dx: dx.dg > 0
        V2, d, edm, skipped = oracle_mod.variable_metric_step(V, rng.normal(size=n), dx, dg)
        assert not skipped
        seen.add(bool(dx @ dg > dg @ V @ dg))
        assert np.allclose(V2 @ dg, dx, rtol=1e-10, atol=1e-12)
        assert np.allclose(V2, V2.T, rtol=1e-13, atol=1e-15)
        assert np.linalg.eigvalsh(0.5 * (V2 + V2.T)).min() > 0
    assert seen == {True, False}                                    # both branches were exercised


def test_exact_rationals_on_a_two_parameter_case(oracle_mod):
    """Dyadic inputs chosen so that every quotient is exact in binary: the update must equal the rational arithmetic
    of the stated rule bit for bit (a = 4 > b = 2: the BFGS term is on)."""
    V = np.array([[1.0, 0.0], [0.0, 1.0]])
    dx, dg = np.array([4.0, 0.0]), np.array([1.0, 1.0])             # a = dx.dg = 4; vg = dg; b = 2
    V2, d, edm, skipped = oracle_mod.variable_metric_step(V, np.array([2.0, -1.0]), dx, dg)
    a, b = F(4), F(2)
    fx, fg = [F(4), F(0)], [F(1), F(1)]
    want = [[F(int(i == j)) + fx[i] * fx[j] / a - fg[i] * fg[j] / b + b * (fx[i] / a - fg[i] / b) * (fx[j] / a - fg[j] / b)
             for j in range(2)] for i in range(2)]
    assert [[float(x) for x in r] for r in want] == V2.tolist()
    g = [F(2), F(-1)]
    dir_want = [-(want[i][0] * g[0] + want[i][1] * g[1]) for i in range(2)]
    assert d.tolist() == [float(x) for x in dir_want]
    assert edm == float(F(1, 2) * sum(g[i] * -dir_want[i] for i in range(2)))


def test_quadratic_with_exact_line_searches_finds_the_inverse_hessian(oracle_mod):
    """On f = 1/2 x^T A x - b^T x with exact line searches a Broyden-family method terminates in n steps with
    V = A^-1 (the textbook finite-termination theorem): minimum reached, metric exact, EDM -> 0."""
    rng = np.random.default_rng(5)
    n = 6
    A, bvec = _spd(rng, n, cond=50.0), rng.normal(size=n)
    x = rng.normal(size=n)
    V = np.eye(n)
    g = A @ x - bvec
    dx = dg = None
    for it in range(n + 1):
        V, d, edm, skipped = oracle_mod.variable_metric_step(V, g, dx, dg)
        assert not skipped and edm >= 0
        if it == n:
            break
        t = -(g @ d) / (d @ A @ d)                                  # exact minimiser along d
        x_new = x + t * d
        g_new = A @ x_new - bvec
        dx, dg, x, g = x_new - x, g_new - g, x_new, g_new
    assert np.allclose(x, np.linalg.solve(A, bvec), rtol=1e-8, atol=1e-10)
    assert np.allclose(V, np.linalg.inv(A), rtol=1e-6, atol=1e-8)
    assert edm < 1e-18


def test_update_is_skipped_without_positive_curvature(oracle_mod):
    V = np.diag([1.0, 2.0, 3.0])
    g = np.array([1.0, 1.0, 1.0])
    for dx, dg in ((np.array([1.0, 0, 0]), np.array([-1.0, 0, 0])),        # dx.dg < 0
                   (np.array([1.0, 0, 0]), np.array([0.0, 1.0, 0])),        # dx.dg = 0
                   (np.array([1.0, 0, 0]), np.zeros(3))):                   # dg = 0: b = 0
        V2, d, edm, skipped = oracle_mod.variable_metric_step(V, g, dx, dg)
        assert skipped and np.array_equal(V2, V) and np.array_equal(d, -V @ g)
