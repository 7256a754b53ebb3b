"""Pins for the oracle's transformation layer ("A transformation layer applies the covariance of
any changed model parameter"; "the 9 polynomial coefficients can be expressed by 7 independent
parameters"): theta = copy(u), then theta[idx_out] = offset + M (u[idx_in] - centre) per block.
"""
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from workloads.spec import OSC_EQ1, DatasetSpec, ModelSpec


def _identity(n):
    return W.TransformSpec(n_u=n, copy_src=np.arange(n, dtype=np.int32), copy_const=np.zeros(n))


def test_identity_and_constants(oracle_mod):
    u = np.random.default_rng(0).normal(size=(4, 6))
    assert np.array_equal(oracle_mod.transform(_identity(6), 6, u), u)
    sp = W.TransformSpec(n_u=2, copy_src=np.array([1, -1, 0, -1], np.int32), copy_const=np.array([9.0, 2.5, 9.0, -1.0]))
    th = oracle_mod.transform(sp, 4, np.array([[3.0, 4.0]]))
    assert np.array_equal(th, [[4.0, 2.5, 3.0, -1.0]])        # permutation + constants; copy_const ignored where copied


def test_block_against_exact_rationals(oracle_mod):
    """A 3 <- 2 block on small dyadic numbers: the fma chain is exact, so it must equal the rational result."""
    M = np.array([[0.5, -2.0], [1.25, 0.75], [-3.0, 0.125]])
    off, cen = np.array([1.0, -0.5, 8.0]), np.array([0.25, -1.5])
    sp = W.TransformSpec(n_u=3, copy_src=np.array([0, 1, 2, -1], np.int32), copy_const=np.zeros(4),
                         blocks=[W.TransformBlock(np.array([3, 0, 1], np.int32), np.array([2, 0], np.int32), off, cen, M)])
    u = np.array([[0.75, 7.0, -2.5]])
    th = oracle_mod.transform(sp, 4, u)[0]
    d = [Fraction(-2.5) - Fraction(0.25), Fraction(0.75) - Fraction(-1.5)]
    want = [Fraction(float(off[i])) + sum(Fraction(float(M[i, j])) * d[j] for j in range(2)) for i in range(3)]
    assert [Fraction(float(th[3])), Fraction(float(th[0])), Fraction(float(th[1]))] == want
    assert th[2] == -2.5                                       # untouched entries keep the copy


def test_rectangular_nine_from_seven_against_numpy(oracle_mod):
    """9 energy-scale coefficients (3 datasets x a0, a1, a2) from 7 independent parameters: one
    fully correlated scintillator non-linearity shared by the datasets plus two uncorrelated terms each."""
    rng = np.random.default_rng(2)
    M = np.zeros((9, 7))
    for d in range(3):
        M[3 * d + 2, 0] = 1.0                # a2 of every dataset <- the shared non-linearity
        M[3 * d + 0, 1 + 2 * d] = 1.0        # a0 <- its own offset parameter
        M[3 * d + 1, 2 + 2 * d] = 1.0        # a1 <- its own scale parameter
    M += 0.01 * rng.normal(size=M.shape)
    off = np.tile([0.0, 1.0, 0.0], 3)
    sp = W.TransformSpec(n_u=11, copy_src=np.array([0, 1, 2, 3] + [-1] * 9, np.int32), copy_const=np.zeros(13),
                         blocks=[W.TransformBlock(np.arange(4, 13, dtype=np.int32), np.arange(4, 11, dtype=np.int32),
                                                  off, np.zeros(7), M)])
    u = rng.normal(size=(5, 11))
    th = oracle_mod.transform(sp, 13, u)
    assert np.array_equal(th[:, :4], u[:, :4])
    assert np.allclose(th[:, 4:], off + u[:, 4:] @ M.T, rtol=1e-14, atol=1e-15)
    # affine: second differences vanish
    t0, t1, t2 = (oracle_mod.transform(sp, 13, u + k * 0.37) for k in (0, 1, 2))
    assert np.allclose(t2 - t1, t1 - t0, rtol=1e-12, atol=1e-12)


def test_cholesky_whitening_makes_the_correlated_prior_a_unit_gaussian(oracle_mod):
    """theta = b0 + L u with L L^T = V (numpy's Cholesky): the correlated prior 1/2 (theta-b0)^T V^-1 (theta-b0)
    of PAPER.md:121-123 becomes 1/2 |u|^2 -- what lets the minimiser treat its parameters as uncorrelated."""
    rng = np.random.default_rng(6)
    A = rng.normal(size=(5, 5))
    V = A @ A.T + 0.3 * np.eye(5)
    L = np.linalg.cholesky(V)
    b0 = rng.normal(size=5)
    idx = np.array([6, 1, 4, 2, 5], np.int32)
    sp = W.TransformSpec(n_u=7, copy_src=np.arange(7, dtype=np.int32), copy_const=np.zeros(7),
                         blocks=[W.TransformBlock(idx, idx, b0, np.zeros(5), L)])
    ds = DatasetSpec(n_bins=2, norm=1.0)
    model = ModelSpec(osc_model=OSC_EQ1, n_params=7, idx_osc=(-1,) * 6, fixed_osc=(0,) * 6, datasets=[ds],
                      prior_blocks=[W.PriorBlock(idx, b0, np.linalg.inv(V))])
    o = oracle_mod.Oracle(model)
    u = rng.normal(size=(8, 7))
    theta = oracle_mod.transform(sp, 7, u)
    nll = o.nll_from_mu(theta, np.tile([4.0, 6.0], (8, 1)), np.array([4.0, 6.0]))
    assert np.allclose(nll, 0.5 * (u[:, idx] ** 2).sum(axis=1), rtol=1e-10)


def test_blocks_apply_in_order(oracle_mod):
    sp = W.TransformSpec(n_u=1, copy_src=np.array([0, 0], np.int32), copy_const=np.zeros(2), blocks=[
        W.TransformBlock(np.array([1], np.int32), np.array([0], np.int32), np.array([1.0]), np.array([0.0]), np.array([[2.0]])),
        W.TransformBlock(np.array([1], np.int32), np.array([0], np.int32), np.array([5.0]), np.array([0.0]), np.array([[3.0]]))])
    assert np.array_equal(oracle_mod.transform(sp, 2, np.array([[2.0]])), [[2.0, 11.0]])


def test_flux_rebinning_41_to_38_conserves_area(oracle_mod):
    """41 flux parameters on uniform 0.25 MeV bins from 1 to 11.25 MeV, "transformed back to the
    original binning".  The piecewise-constant, area-conserving version of that map is a 38 x 41 block of the
    transformation layer: f_b = sum_j overlap(b, j) F_j / width_b (the analysis bins above 11.25 MeV keep 1).
    Pin: the integral of the flux correction over any union of analysis bins equals the integral of the 41-bin
    step function over the same range (R6 edges)."""
    edges = W.dc_edges()
    fine = 1.0 + 0.25 * np.arange(42)
    M = np.zeros((38, 41))
    off = np.zeros(38)
    for b in range(38):
        lo, hi = edges[b], edges[b + 1]
        for j in range(41):
            M[b, j] = max(0.0, min(hi, fine[j + 1]) - max(lo, fine[j])) / (hi - lo)
        off[b] = 1.0 - M[b].sum()                      # the part of the bin above 11.25 MeV keeps the nominal 1
    sp = W.TransformSpec(n_u=41, copy_src=np.full(38, -1, np.int32), copy_const=np.zeros(38),
                         blocks=[W.TransformBlock(np.arange(38, dtype=np.int32), np.arange(41, dtype=np.int32),
                                                  off, np.zeros(41), M)])
    rng = np.random.default_rng(9)
    F = 1.0 + 0.02 * rng.normal(size=(6, 41))
    f = oracle_mod.transform(sp, 38, F)
    widths = np.diff(edges)
    for p in range(6):
        # whole range 1-20 MeV, and 1-8 MeV where analysis and fine bins coincide
        assert (f[p] * widths).sum() == pytest.approx((F[p] * 0.25).sum() + (20.0 - 11.25), rel=1e-13)
        assert np.allclose(f[p, :28], F[p, :28], rtol=1e-14)
        assert f[p, -1] == 1.0                         # 18-20 MeV: beyond the flux parametrisation
    assert np.array_equal(oracle_mod.transform(sp, 38, np.ones((1, 41))), np.ones((1, 38)))
