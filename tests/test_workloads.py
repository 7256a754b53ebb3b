"""The seeded input recipe (BASELINE.json `configs`): shapes, sizes and distributions of the
five synthetic workloads, and that the generators are deterministic and hold no arithmetic of the method."""
import inspect

import numpy as np
import pytest

import workloads
from workloads import generate, spec


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_deterministic_and_shaped_like_the_config(k):
    a = workloads.make_config(k, scale=0.001)
    b = workloads.make_config(k, scale=0.001)
    assert np.array_equal(a.params, b.params)
    for ea, eb in zip(a.events, b.events):
        assert np.array_equal(ea.e_nu, eb.e_nu) and np.array_equal(ea.e_vis, eb.e_vis) and np.array_equal(ea.core, eb.core)
    m = a.model
    want = {1: (1, 1, 7, [40], 0), 2: (2, 64, 10, [38, 38], 0), 3: (3, 603, 301, [38] * 3, 0),
            4: (1, 128, 4, [410], 1), 5: (2, 4096, 6, [38, 38], 2)}[k]
    assert (len(a.events), a.n_points, m.n_params, [d.n_bins for d in m.datasets], m.osc_model) == want
    for e in a.events:
        assert e.e_nu.dtype == np.float32 and e.e_vis.dtype == np.float32 and e.w.dtype == np.float32
        assert e.e_nu.min() >= 1.8 and e.e_nu.max() < 10.0           # "support 1.8-10 MeV"
        assert np.all(e.w == 1.0)                                     # "MC weight 1"
        assert np.all(np.diff(e.edges) > 0)


def test_full_sizes_and_structure():
    n = {k: workloads.make_config(k, scale=1e-4) for k in (2, 3, 4, 5)}
    # config 3: central differences -- every point differs from the first in at most one parameter
    p = n[3].params
    assert p.shape == (603, 301)
    assert ((p[1:] != p[0]).sum(axis=1) == 1).all()
    # config 5: 64 x 64 grid in (sin^2 2theta14, dm2_41), log-spaced inside the stated ranges
    q = n[5].params
    s14, m41 = np.unique(q[:, 4]), np.unique(q[:, 5])
    assert len(s14) == 64 and len(m41) == 64
    assert s14[0] == pytest.approx(1e-3) and s14[-1] == pytest.approx(0.3)
    assert m41[0] == pytest.approx(1e-2) and m41[-1] == pytest.approx(10.0)
    assert np.allclose(np.diff(np.log(s14)), np.log(s14[1] / s14[0]))
    # config 4: 11 cores, 9 near ones 52.0-52.8 km, 215 and 265 km
    L = n[4].events[0].L_m
    assert len(L) == 11 and L[0] == 52_000.0 and L[8] == 52_800.0 and list(L[9:]) == [215_000.0, 265_000.0]
    assert n[4].events[0].edges[0] == pytest.approx(0.8) and n[4].events[0].edges[-1] == pytest.approx(9.0)
    # config 2: two cores per detector at the stated baselines
    assert list(n[2].events[0].L_m) == [355.0, 469.0] and list(n[2].events[1].L_m) == [998.0, 1115.0]


def test_reactor_spectrum_shape():
    """gamma-like, peak near 3.8 MeV; E_vis = E_nu - 0.782 smeared by 0.08 sqrt(E)."""
    rng = np.random.Generator(np.random.PCG64(5))
    ev = workloads.reactor_events(rng, 200_000, [1050.0], [1.0], 0.08, workloads.dc_edges())
    hist, edges = np.histogram(ev.e_nu, bins=np.arange(1.8, 10.01, 0.2))
    assert abs(edges[np.argmax(hist)] + 0.1 - 3.8) <= 0.3
    d = ev.e_vis.astype(np.float64) - (ev.e_nu.astype(np.float64) - 0.782)
    assert abs(d.mean()) < 2e-3
    assert d.std() == pytest.approx(0.08 * np.sqrt(np.mean(ev.e_nu.astype(np.float64) - 0.782)), rel=0.05)


def test_generators_hold_no_arithmetic_of_the_method():
    """workloads/ serves both the oracle and the CUDA path, so it may not compute what they compute."""
    src = inspect.getsource(generate) + inspect.getsource(spec)
    for word in ("sin(", "cos(", "1.267", "searchsorted", "digitize", "histogram(", "lgamma", "log("):
        assert word not in src, word
    for mod in ("import oracle", "from oracle", "paper_2502_15253_b200", "ctypes"):
        assert mod not in src, mod
