"""Pins of the oracle's bin-level steps (PAPER.md:177 signal steps 2-3, :129 flux model; R27, R28).
The paper gives no formula for "smoothed using a second-degree polynomial function ... integrated over the original
binning"; these tests pin the reading taken against what mathematics fixes for it: identity, conservation of area,
exactness on quadratics, the one-bin shift, exact rationals on a toy, and the flux model's agreement with the
piecewise-constant 38 x 41 block where no energy correction acts."""
from fractions import Fraction

import numpy as np
import pytest

import workloads
from workloads.spec import DatasetSpec, FluxModel, ModelSpec, OSC_EQ1


def _edges_nonuniform():
    return np.array([1.0, 1.25, 1.5, 2.0, 2.25, 3.25, 3.5, 4.0, 6.0])


def test_inverse_of_the_energy_scale(oracle_mod):
    for a0, a1, a2 in ((0.0, 1.0, 0.0), (0.02, 0.99, 0.0), (0.03, 1.01, 1e-3), (-0.02, 0.98, -2e-3)):
        for t in (0.5, 1.0, 3.7, 9.0, 20.0):
            x = oracle_mod.escale_inverse(a0, a1, a2, t)
            assert a0 + a1 * x + a2 * x * x == pytest.approx(t, rel=1e-14)
    assert oracle_mod.escale_inverse(0.0, 1.0, 0.0, 3.5) == 3.5


def test_identity_map_returns_the_input(oracle_mod):
    e = _edges_nonuniform()
    h = np.array([3.0, 7.0, 2.0, 9.0, 4.0, 1.0, 0.5, 6.0])
    out = oracle_mod.rebin_quadratic(e, h, e)
    assert np.allclose(out, h, rtol=1e-14, atol=1e-14)          # the parabola of bin b integrates to H_b over bin b


def test_area_is_conserved_inside_the_range(oracle_mod):
    e = _edges_nonuniform()
    rng = np.random.default_rng(1)
    h = rng.uniform(0.0, 10.0, 8)
    h[0] = h[-1] = 0.0
    for a in ((0.01, 1.0, 0.0), (0.0, 1.002, 0.0), (0.005, 0.999, 2e-4)):
        x = np.array([oracle_mod.escale_inverse(*a, t) for t in e])
        # widen the first and last target so that they catch everything the map moves across the ends
        x[0], x[-1] = min(x[0], e[0]), max(x[-1], e[-1])
        out = oracle_mod.rebin_quadratic(e, h, x)
        assert out.sum() == pytest.approx(h.sum(), rel=1e-13)


def test_quadratic_density_is_reproduced_exactly(oracle_mod):
    """a spectrum that IS the bin integrals of one parabola: every local parabola is that parabola"""
    e = _edges_nonuniform()
    Q = lambda t: 2.0 * t - 0.3 * t ** 2 / 2 + 0.05 * t ** 3 / 3           # antiderivative of 2 - 0.3 t + 0.05 t^2
    h = Q(e[1:]) - Q(e[:-1])
    x = np.array([1.1, 1.7, 2.05, 2.9, 3.3, 5.5])
    out = oracle_mod.rebin_quadratic(e, h, x)
    assert np.allclose(out, Q(x[1:]) - Q(x[:-1]), rtol=1e-12)


def test_shift_by_one_bin_width_shifts_the_histogram(oracle_mod):
    """uniform bins, E' = E + width: the pre-image of bin c is exactly bin c-1, so H'_c = H_(c-1) whatever the
    contents -- the per-event map would move every event by one bin as well"""
    e = 1.0 + 0.25 * np.arange(13)
    rng = np.random.default_rng(2)
    h = rng.uniform(0.0, 50.0, 12)
    x = np.array([oracle_mod.escale_inverse(0.25, 1.0, 0.0, t) for t in e])
    assert np.array_equal(x[1:], e[:-1])
    out = oracle_mod.rebin_quadratic(e, h, x)
    assert out[0] == 0.0 and np.allclose(out[1:], h[:-1], rtol=1e-13)


def test_four_bin_toy_in_exact_rationals(oracle_mod):
    """brute force with fractions: cubic through the cumulative points of each triple, integrated over the overlaps"""
    e = [Fraction(0), Fraction(1), Fraction(3), Fraction(4), Fraction(6)]
    h = [Fraction(2), Fraction(5), Fraction(1), Fraction(4)]
    x = [Fraction(1, 2), Fraction(3, 2), Fraction(7, 2), Fraction(5)]

    def cum(t0, E):
        X, Y = e[t0:t0 + 4], h[t0:t0 + 3]
        f01, f12, f23 = Y[0] / (X[1] - X[0]), Y[1] / (X[2] - X[1]), Y[2] / (X[3] - X[2])
        f012, f123 = (f12 - f01) / (X[2] - X[0]), (f23 - f12) / (X[3] - X[1])
        f0123 = (f123 - f012) / (X[3] - X[0])
        return f01 * (E - X[0]) + f012 * (E - X[0]) * (E - X[1]) + f0123 * (E - X[0]) * (E - X[1]) * (E - X[2])

    want = []
    for c in range(3):
        s = Fraction(0)
        for b in range(4):
            lo, hi = max(x[c], e[b]), min(x[c + 1], e[b + 1])
            if lo < hi:
                t0 = min(max(b - 1, 0), 1)
                s += cum(t0, hi) - cum(t0, lo)
        want.append(float(s))
    got = oracle_mod.rebin_quadratic([float(v) for v in e], [float(v) for v in h], [float(v) for v in x])
    assert np.allclose(got, want, rtol=1e-14)
    # the cubic through four cumulative points reproduces the three bin contents: a triple checks itself
    assert cum(0, e[3]) == sum(h[:3]) and cum(1, e[4]) - cum(1, e[1]) == sum(h[1:])


def test_one_and_two_bin_spectra(oracle_mod):
    assert np.allclose(oracle_mod.rebin_quadratic([0.0, 2.0], [6.0], [0.5, 1.0, 2.0]), [1.5, 3.0])
    out = oracle_mod.rebin_quadratic([0.0, 1.0, 3.0], [2.0, 2.0], [0.0, 1.0, 3.0])
    assert np.allclose(out, [2.0, 2.0], rtol=1e-14)


def _flux_dataset():
    edges = workloads.dc_edges()
    ds = DatasetSpec(n_bins=38, idx_a=(41, 42, 43), flux_model=FluxModel(idx_par=np.arange(41, dtype=np.int32)))
    model = ModelSpec(osc_model=OSC_EQ1, n_params=44, idx_osc=(-1,) * 6, fixed_osc=(0.1, 2.5e-3, 0.85, 7.5e-5, 0, 0),
                      datasets=[ds])
    ev = workloads.reactor_events(np.random.default_rng(0), 10, [1000.0], [1.0], 0.08, edges)
    return model, [ev], edges


def test_flux_model_without_energy_correction_is_the_area_conserving_block(oracle_mod):
    """at the identity energy scale the spline's average over an analysis bin is the average of the
    fine bins it covers (area conservation), i.e. the piecewise-constant 38 x 41 block pinned in
    test_oracle_transform.py; above 11.25 MeV the scale stays 1."""
    model, evs, edges = _flux_dataset()
    orc = oracle_mod.Oracle(model, evs)
    rng = np.random.default_rng(4)
    F = 1.0 + 0.03 * rng.normal(size=41)
    theta = np.r_[F, 0.0, 1.0, 0.0]
    f = orc.flux_scales(0, theta)
    fine = 1.0 + 0.25 * np.arange(42)
    want = np.ones(38)
    for b in range(38):
        lo, hi = edges[b], edges[b + 1]
        ov = np.clip(np.minimum(hi, fine[1:]) - np.maximum(lo, fine[:-1]), 0.0, None)
        want[b] = (ov * F).sum() / (hi - lo) + (1.0 - ov.sum() / (hi - lo))
    assert np.allclose(f, want, rtol=1e-13)
    assert np.array_equal(orc.flux_scales(0, np.r_[np.ones(41), 0.01, 0.99, 1e-3]), np.ones(38)) or \
        np.allclose(orc.flux_scales(0, np.r_[np.ones(41), 0.01, 0.99, 1e-3]), 1.0, rtol=1e-14)


def test_flux_model_follows_the_energy_scale(oracle_mod):
    """a linear flux tilt phi(E) = 1 + s (E - 5) inside the fine grid: the spline reproduces a linear function exactly,
    so the scale of bin b is phi at the centre of the bin's pre-image"""
    model, evs, edges = _flux_dataset()
    orc = oracle_mod.Oracle(model, evs)
    fine_c = 1.125 + 0.25 * np.arange(41)
    F = 1.0 + 0.02 * (fine_c - 5.0)
    a = (0.03, 0.99, 0.0)
    f = orc.flux_scales(0, np.r_[F, a])
    x = np.array([oracle_mod.escale_inverse(*a, t) for t in edges])
    inside = (x[:-1] >= 1.0) & (x[1:] <= 11.25)
    centre = 0.5 * (x[1:] + x[:-1])
    assert np.allclose(f[inside], 1.0 + 0.02 * (centre[inside] - 5.0), rtol=1e-13)


def test_bin_level_mode_end_to_end_properties(oracle_mod):
    """energy_correction = 1 on a small workload: identity scale == per-event mode exactly; a shift by one bin width
    moves the spectrum by one bin in both modes; the likelihood is assembled as step 2 then step 3"""
    wl = workloads.make_tiny(seed=9, n_events=400, n_points=3)
    edges = 1.0 + 0.5 * np.arange(8)
    wl.events[0].edges = edges
    wl.events[0].e_vis = np.float32(1.0) + np.float32(0.5) * (np.arange(400, dtype=np.float32) % 7) + np.float32(0.25)
    wl.params[:, 6:9] = (0.0, 1.0, 0.0)
    wl.params[1] = wl.params[0]
    wl.params[1, 6] = 0.5                                  # the same point, one bin width up
    per_event = oracle_mod.Oracle(wl.model, wl.events)
    wl.model.energy_correction = 1
    binned = oracle_mod.Oracle(wl.model, wl.events)
    h_e, h_b = per_event.spectra(wl.params), binned.spectra(wl.params)
    assert np.allclose(h_b[0], h_e[0], rtol=1e-13) and np.allclose(h_b[2], h_e[2], rtol=1e-13)
    assert np.allclose(h_b[1], h_e[1], rtol=1e-12)          # events sit mid-bin: both modes shift them by one bin
    assert np.array_equal(binned.spectra_raw(wl.params)[1], binned.spectra_raw(wl.params)[0])
    assert h_b[1][0] == 0.0 and np.allclose(h_b[1][1:], h_b[0][:-1], rtol=1e-13)
    data = np.arange(7, dtype=np.float64) + 3.0
    mu = binned.expectation(wl.params, binned.spectra_raw(wl.params))
    assert np.allclose(binned.nll(wl.params, data), binned.nll_from_mu(wl.params, mu, data), rtol=1e-15)
    assert np.allclose(binned.nll(wl.params, data)[[0, 2]], per_event.nll(wl.params, data)[[0, 2]], rtol=1e-12)
