"""Pins for oracle step O3: per-event weight, energy-scale map, binning, per-bin sums.

PAPER.md:177 (signal step 1), :141 (polynomial response), :183 (bins independent);
DESIGN.md R7 (half-open bins), R8 (per-event E', Horner with fma).
Expected values come from numpy histograms, exact rationals and mpmath — never from the oracle.
"""
from fractions import Fraction

import mpmath as mp
import numpy as np
import pytest

import workloads as W
from workloads.spec import (OSC_EQ1, OSC_FULL3, OSC_STERILE4, DatasetEvents, DatasetSpec, ModelSpec)
from helpers import K, angles, escale_exact, hist_right, pee_eq1_mp


def _one_dataset_model(osc=OSC_EQ1, n_bins=7, with_a=True):
    return ModelSpec(osc_model=osc, n_params=9, idx_osc=(0, 1, 2, 3, 4, 5), fixed_osc=(0,) * 6,
                     datasets=[DatasetSpec(n_bins=n_bins, idx_a=(6, 7, 8) if with_a else (-1, -1, -1))])


def _theta(s13=0.1, mee=2.5e-3, s12=0.85, m21=7.5e-5, s14=0.0, m41=0.0, a=(0.0, 1.0, 0.0)):
    return np.array([s13, mee, s12, m21, s14, m41, *a])


def _events(seed, n=5000, edges=None, weights="uniform"):
    rng = np.random.Generator(np.random.PCG64(seed))
    edges = W.dc_edges() if edges is None else edges
    return W.reactor_events(rng, n, [355.0, 469.0, 1050.0], [0.3, 0.3, 0.4], 0.08, edges, weights=weights)


def test_unoscillated_is_plain_weighted_histogram(oracle_mod):
    """north_star pin: all mixings 0 => H == weighted histogram of E' (numpy searchsorted+bincount)."""
    ev = _events(1)
    o = oracle_mod.Oracle(_one_dataset_model(n_bins=38), [ev])
    a = (0.013, 0.991, 0.0007)
    h = o.spectra(_theta(s13=0.0, s12=0.0, a=a))[0]
    ep = np.array([escale_exact(a[0], a[1], a[2], float(v)) for v in ev.e_vis])
    want = hist_right(ep, ev.w, ev.edges)
    assert np.allclose(h, want, rtol=1e-13, atol=0)
    assert h.sum() > 0.9 * ev.w.sum()


def test_identity_energy_scale_is_histogram_of_evis(oracle_mod):
    ev = _events(2)
    for with_a in (True, False):
        o = oracle_mod.Oracle(_one_dataset_model(n_bins=38, with_a=with_a), [ev])
        h = o.spectra(_theta(s13=0.0, s12=0.0))[0]
        assert np.allclose(h, hist_right(ev.e_vis.astype(np.float64), ev.w, ev.edges), rtol=1e-13)


def test_exact_one_bin_shift(oracle_mod):
    """a0 = one bin width on a uniform 0.25 grid shifts the histogram by exactly one bin."""
    edges = 1.0 + 0.25 * np.arange(41)
    ev = _events(3, edges=edges)
    o = oracle_mod.Oracle(_one_dataset_model(n_bins=40), [ev])
    h0 = o.spectra(_theta(s13=0.0, s12=0.0))[0]
    h1 = o.spectra(_theta(s13=0.0, s12=0.0, a=(0.25, 1.0, 0.0)))[0]
    assert np.array_equal(h1[1:], h0[:-1])
    # what fell below edges[0] before now sits in bin 0; the old top bin fell off the end
    below = ev.w[(ev.e_vis >= 0.75) & (ev.e_vis < 1.0)].astype(np.float64).sum()
    assert h1[0] == pytest.approx(below, rel=1e-13)


def test_edge_conventions(oracle_mod):
    """Event exactly on an edge goes to the upper bin; last edge exclusive; below first dropped; NaN dropped."""
    edges = np.array([1.0, 1.5, 2.25, 3.0])
    e_vis = np.array([1.0, 1.5, 2.25, 3.0, 0.999999, np.nextafter(np.float32(3.0), np.float32(0)),
                      np.nextafter(np.float32(1.5), np.float32(0)), np.nan], dtype=np.float32)
    n = len(e_vis)
    ev = DatasetEvents(e_nu=np.full(n, 3.0, np.float32), e_vis=e_vis,
                       w=np.arange(1, n + 1, dtype=np.float32), core=np.zeros(n, np.int32),
                       L_m=np.array([1000.0]), edges=edges)
    o = oracle_mod.Oracle(_one_dataset_model(n_bins=3), [ev])
    h = o.spectra(_theta(s13=0.0, s12=0.0))[0]
    #   w:      1->bin0  2->bin1  3->bin2  4 dropped  5 dropped  6->bin2  7->bin0  8 dropped
    assert np.array_equal(h, np.array([1.0 + 7.0, 2.0, 3.0 + 6.0]))
    bins = o.event_bins(_theta(s13=0.0, s12=0.0))[0]
    assert bins.tolist() == [0, 1, 2, -1, -1, 2, 0, -1]
    assert oracle_mod.bin_index(edges, 1.0) == 0 and oracle_mod.bin_index(edges, 3.0) == -1
    assert oracle_mod.bin_index(edges, float("nan")) == -1
    assert oracle_mod.bin_index(edges, float("inf")) == -1 and oracle_mod.bin_index(edges, -1.0) == -1


def test_escale_is_horner_fma(oracle_mod):
    """E' = fma(fma(a2,v,a1),v,a0) bit-for-bit (exact rationals); differs from the unfused form somewhere."""
    rng = np.random.default_rng(0)
    differs = 0
    for _ in range(3000):
        a0, a1, a2 = rng.normal(0, 0.02), rng.normal(1, 0.01), rng.normal(0, 0.001)
        v = float(np.float32(rng.uniform(0.5, 12)))
        got = oracle_mod.escale(a0, a1, a2, v)
        assert got == escale_exact(a0, a1, a2, v)
        differs += got != (a0 + a1 * v + a2 * v * v)
    assert differs > 100        # the pin would be vacuous if fused and unfused always agreed


def test_bin_index_matches_searchsorted(oracle_mod):
    edges = W.dc_edges()
    rng = np.random.default_rng(1)
    vals = np.concatenate([rng.uniform(0, 21, 3000), edges, np.nextafter(edges, 0), np.nextafter(edges, 30)])
    for v in vals:
        want = int(np.searchsorted(edges, v, side="right") - 1)
        if not (edges[0] <= v < edges[-1]):
            want = -1
        assert oracle_mod.bin_index(edges, float(v)) == want


def test_monochromatic_source_separates(oracle_mod):
    """north_star pin: one E_nu, one L  =>  H = H_unosc * (1 - A1 S1 - A2 S2), S_k scalar."""
    ev = _events(4, n=3000)
    ev.e_nu[:] = np.float32(3.7)
    ev.core[:] = 2
    o = oracle_mod.Oracle(_one_dataset_model(n_bins=38), [ev])
    th = _theta(s13=0.12, s12=0.8)
    h = o.spectra(th)[0]
    h0 = o.spectra(_theta(s13=0.0, s12=0.0))[0]
    p = pee_eq1_mp(0.12, 2.5e-3, 0.8, 7.5e-5, 1050.0, float(np.float32(3.7)))
    assert np.allclose(h, h0 * float(p), rtol=1e-13)
    assert 0.85 < float(p) < 0.99


def test_affine_in_amplitudes(oracle_mod):
    """For fixed dm2 and energy scale H is affine in (A1, A2): three evaluations predict a fourth.
    STERILE4 with s13 = s12 = 0 isolates the amplitude s14 exactly (cos^4 factors multiply zeros)."""
    ev = _events(5, n=4000)
    o = oracle_mod.Oracle(_one_dataset_model(osc=OSC_STERILE4, n_bins=38), [ev])
    f = lambda s14: o.spectra(_theta(s13=0.0, s12=0.0, s14=s14, m41=0.8))[0]
    h0, h1, h2 = f(0.0), f(0.1), f(0.25)
    assert np.allclose(h2, h0 + 2.5 * (h1 - h0), rtol=1e-12)
    assert np.all(h1 <= h0) and np.any(h1 < 0.97 * h0)


def test_sum_over_bins_is_sum_of_weights_times_p(oracle_mod):
    ev = _events(6, n=2000)
    o = oracle_mod.Oracle(_one_dataset_model(n_bins=38), [ev])
    th = _theta()
    h = o.spectra(th)[0]
    A, m = o.terms(th)
    tot = mp.mpf(0)
    for i in range(ev.n):
        v = float(ev.e_vis[i])
        if ev.edges[0] <= v < ev.edges[-1]:
            tot += mp.mpf(float(ev.w[i])) * pee_eq1_mp(0.1, 2.5e-3, 0.85, 7.5e-5, ev.L_m[ev.core[i]], float(ev.e_nu[i]))
    assert abs(h.sum() - float(tot)) / float(tot) < 1e-13


@pytest.mark.parametrize("osc", [OSC_EQ1, OSC_FULL3, OSC_STERILE4])
def test_brute_force_tiny(oracle_mod, osc):
    """<= 100 events: every bin against mpmath (50 digits) + exact-rational E' and binning."""
    wl = W.make_tiny(seed=40 + osc, osc_model=osc, n_events=100, n_points=4, n_datasets=2)
    o = oracle_mod.Oracle(wl.model, wl.events)
    h = o.spectra(wl.params)
    for p in range(wl.n_points):
        th = wl.params[p]
        s13, mee, s12, m21, s14, m41 = [mp.mpf(float(x)) for x in th[:6]]
        t13, t12, t14 = angles(s13), angles(s12), angles(s14)
        off = 0
        for d, ev in enumerate(wl.events):
            a0, a1, a2 = [float(th[j]) for j in wl.model.datasets[d].idx_a]
            want = [mp.mpf(0)] * ev.n_bins
            for i in range(ev.n):
                x = mp.mpf(float(ev.L_m[ev.core[i]])) / mp.mpf(float(ev.e_nu[i]))
                sq = lambda dm: mp.sin(K * dm * x) ** 2
                if osc == OSC_EQ1:
                    P = 1 - s13 * sq(mee) - mp.cos(t13) ** 4 * s12 * sq(m21)
                elif osc == OSC_FULL3:
                    m31 = mee + mp.sin(t12) ** 2 * m21
                    m32 = mee - mp.cos(t12) ** 2 * m21
                    P = (1 - mp.cos(t13) ** 4 * s12 * sq(m21)
                         - s13 * (mp.cos(t12) ** 2 * sq(m31) + mp.sin(t12) ** 2 * sq(m32)))
                else:
                    P = (1 - mp.cos(t14) ** 4 * s13 * sq(mee) - s14 * sq(m41)
                         - mp.cos(t13) ** 4 * s12 * sq(m21))
                ep = escale_exact(a0, a1, a2, float(ev.e_vis[i]))
                if not (ev.edges[0] <= ep < ev.edges[-1]):
                    continue
                b = int(np.searchsorted(ev.edges, ep, side="right") - 1)
                want[b] += mp.mpf(float(ev.w[i])) * P
            got = h[p, off:off + ev.n_bins]
            for b in range(ev.n_bins):
                if want[b] == 0:
                    assert got[b] == 0.0
                else:
                    # FULL3 tiny input has a 52.5 km core: phase ~ 40 rad, fp64 phase rounding ~ 1e-14
                    assert abs(got[b] - float(want[b])) <= 2e-13 * float(want[b]), (p, d, b)
            off += ev.n_bins


def test_additivity_and_permutation(oracle_mod):
    """bins (and events) are independent — splitting the event list sums to the whole;
    any event order gives the same sums to 1e-12 (compensated summation)."""
    ev = _events(7, n=6000)
    model = _one_dataset_model(n_bins=38)
    th = _theta(a=(0.01, 1.004, -0.0003))
    h = oracle_mod.Oracle(model, [ev]).spectra(th)[0]

    def sub(idx):
        return DatasetEvents(e_nu=ev.e_nu[idx], e_vis=ev.e_vis[idx], w=ev.w[idx], core=ev.core[idx],
                             L_m=ev.L_m, edges=ev.edges)
    idx = np.arange(ev.n)
    ha = oracle_mod.Oracle(model, [sub(idx[:2500])]).spectra(th)[0]
    hb = oracle_mod.Oracle(model, [sub(idx[2500:])]).spectra(th)[0]
    assert np.allclose(ha + hb, h, rtol=1e-13)
    perm = np.random.default_rng(0).permutation(ev.n)
    hp = oracle_mod.Oracle(model, [sub(perm)]).spectra(th)[0]
    assert np.allclose(hp, h, rtol=1e-12)
    # sorted by (core, e_vis) -- the order the CUDA event store uses (R14)
    order = np.lexsort((ev.e_vis, ev.core))
    hs = oracle_mod.Oracle(model, [sub(order)]).spectra(th)[0]
    assert np.allclose(hs, h, rtol=1e-12)


def test_null_weight_and_core_defaults(oracle_mod):
    """w = NULL => 1, core = NULL => 0 (include/phylino.h mirrors this)."""
    ev = _events(8, n=500, weights="one")
    ev0 = DatasetEvents(e_nu=ev.e_nu, e_vis=ev.e_vis, w=None, core=None, L_m=ev.L_m[:1], edges=ev.edges)
    ev1 = DatasetEvents(e_nu=ev.e_nu, e_vis=ev.e_vis, w=np.ones(500, np.float32),
                        core=np.zeros(500, np.int32), L_m=ev.L_m[:1], edges=ev.edges)
    model = _one_dataset_model(n_bins=38)
    h0 = oracle_mod.Oracle(model, [ev0]).spectra(_theta())[0]
    h1 = oracle_mod.Oracle(model, [ev1]).spectra(_theta())[0]
    assert np.array_equal(h0, h1)


def test_threads_do_not_change_bits(oracle_mod):
    wl = W.make_config(2, scale=0.002, n_points=9)
    o = oracle_mod.Oracle(wl.model, wl.events)
    assert np.array_equal(o.spectra(wl.params, n_threads=1), o.spectra(wl.params, n_threads=0))
