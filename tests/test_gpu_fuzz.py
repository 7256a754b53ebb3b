"""-m gpu: seeded random sweep of small workloads against the oracle.

Random event counts (including 0 and counts that leave ragged batches and units), 1-3 datasets, 1-70 points
(all lane mappings: sub-streams for <= 16 points, full groups, ragged last group), unit or random weights,
the three oscillation models (FULL3 in both mass orderings), random work cuts, the three schedules,
dense / host / cached entry points, and in a third of the cases prior blocks over parameters and over random
polynomial functions of them.  Same bars as everywhere:
bit-exact bins, per-bin relative error <= 1e-7, |dNLL| <= 1e-6.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

import os
N_CASES = int(os.environ.get("PHYLINO_FUZZ_CASES", "48"))     # more cases for an occasional deeper sweep


def _case(i):
    rng = np.random.default_rng(10_000 + i)
    osc = int(rng.integers(0, 3))
    n_ds = int(rng.integers(1, 4))
    n_ev = int(rng.choice([0, 1, 3, 4, 5, 63, 64, 65, 255, 257, 1000, 2049, 3001, 8191, 20000]))
    n_pt = int(rng.choice([1, 2, 3, 5, 8, 15, 16, 17, 31, 32, 33, 47, 64, 70]))
    ordering = -1 if (osc == 1 and rng.random() < 0.5) else +1      # FULL3: both mass orderings
    wl = workloads.make_tiny(seed=20_000 + i, osc_model=osc, n_events=n_ev, n_points=n_pt, n_datasets=n_ds,
                             ordering=ordering)
    if rng.random() < 0.5:                        # the unit-weight paths
        for e in wl.events:
            e.w[:] = 1.0
    if rng.random() < 0.3:                        # repeated points: something for the cache to find
        wl.params[n_pt // 2:] = wl.params[: n_pt - n_pt // 2]
        wl.params[n_pt // 2:, 0] *= 0.97
    if rng.random() < 0.33:                       # constraints on functions of the parameters, mixed with raw ones
        NP = wl.model.n_params
        fns = []
        for _ in range(int(rng.integers(1, 4))):
            terms = []
            for _ in range(int(rng.integers(0, 4))):
                k = int(rng.integers(0, 4))
                terms.append((float(rng.normal()), rng.integers(0, NP, k).astype(np.int32),
                              rng.integers(-2, 4, k).astype(np.int32)))
            fns.append(workloads.FunctionSpec(terms=terms, offset=float(rng.normal())))
        wl.model.functions = fns
        n = int(rng.integers(1, len(fns) + 3))
        idx = np.concatenate([NP + rng.permutation(len(fns))[: min(n, len(fns))],
                              rng.integers(0, NP, max(0, n - len(fns)))]).astype(np.int32)
        A = rng.normal(size=(len(idx), len(idx)))
        wl.model.prior_blocks = [workloads.PriorBlock(idx, rng.normal(size=len(idx)), A @ A.T + np.eye(len(idx)))]
    tuning = (int(rng.choice([0, 16, 64, 128, 256])), int(rng.choice([0, 1, 2])), int(rng.choice([0, 0, 8, 148, 1000])))
    return wl, tuning, bool(rng.random() < 0.5), int(rng.choice([0, 0, 1, 2]))


@pytest.mark.parametrize("i", range(N_CASES))
def test_random_small_workload(gpu, oracle_mod, i):
    import torch
    wl, tuning, cache, schedule = _case(i)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    data = np.arange(orc.total_bins, dtype=np.float64) * 2.0 + 1.0
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        ph.set_tuning(*tuning)
        ph.set_schedule(schedule)                 # library's choice / always tickets / small-batch kernel up to 16 points
        dp = torch.as_tensor(wl.params, device="cuda")
        h = ph.spectra(dp).cpu().numpy()
        nll = ph.nll(dp, torch.as_tensor(data, device="cuda")).cpu().numpy()
        bins = ph.event_bins(dp).cpu().numpy() if wl.n_events else None
        ph.set_caching(cache)
        nll_h = ph.nll_host(wl.params, data)
    h_o, nll_o = orc.spectra(wl.params), orc.nll(wl.params, data)
    if bins is not None:
        assert np.array_equal(bins, orc.event_bins(wl.params))
    nz = h_o != 0
    assert np.array_equal(h[~nz], h_o[~nz])
    if nz.any():
        assert (np.abs(h - h_o)[nz] / np.abs(h_o[nz])).max() <= 1e-7
    fin = np.isfinite(nll_o)
    assert np.array_equal(np.isfinite(nll), fin) and np.array_equal(np.isfinite(nll_h), fin)
    if fin.any():
        # DESIGN.md R31: the 1e-6 bar is for likelihoods of the paper's size (up to ~1e6); a random constraint on
        # theta^-2 of a 1e-5-sized parameter makes the NLL 1e10, where ONE ulp is 2e-6: beyond 1e6 the bar scales with
        # the value (1e-12 relative)
        tol = 1e-6 * np.maximum(1.0, np.abs(nll_o[fin]) / 1e6)
        assert np.all(np.abs(nll[fin] - nll_o[fin]) <= tol)
        assert np.all(np.abs(nll_h[fin] - nll_o[fin]) <= tol)
