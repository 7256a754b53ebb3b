"""Seeded generators for the five BASELINE.json configs and for tiny brute-force inputs.

Random numbers: numpy `Generator(PCG64(seed))`; every array both sides see is produced
here once and handed to the oracle and to the CUDA path unchanged.  Nothing in this
file evaluates an oscillation probability, an energy-scale map, a bin index or a
likelihood; `poisson_counts` takes the expectation as an argument.

Recipes (restated in DESIGN.md):
  E_nu  = 1.8 + Gamma(shape 5, scale 0.5 MeV), redrawn if >= 10   (mode 3.8 MeV, support 1.8-10;
          BASELINE.json config 1 "gamma-like, peak 3.8 MeV")
  E_vis = (E_nu - 0.782) + r * sqrt(E_nu - 0.782) * z,  z ~ N(0,1), r = 0.08 (DC) / 0.03 (JUNO-like)
  both stored as float32; MC weight 1 (configs) or U(0.5,1.5) (tiny inputs).
"""
from __future__ import annotations

import numpy as np

from .spec import (BkgSpec, DatasetEvents, DatasetSpec, ModelSpec, Workload,
                   OSC_EQ1, OSC_FULL3, OSC_STERILE4)

CONFIG_NAMES = {
    1: "dc_fd_single",       # BASELINE.json configs[0]
    2: "dc_fd_nd_batch64",   # configs[1]  (the bench workload)
    3: "dc_gradient_603",    # configs[2]
    4: "juno_like_128",      # configs[3]
    5: "sterile_grid_4096",  # configs[4]
}
DEFAULT_SEEDS = {1: 1001, 2: 1002, 3: 1003, 4: 1004, 5: 1005}

# nominal oscillation point (BASELINE.json config 1) and the "around nominal" widths
THETA0 = dict(s13=0.1, mee=2.5e-3, s12=0.85, m21=7.5e-5)
SIGMA0 = dict(s13=0.01, mee=5e-5, s12=0.02, m21=2e-6)
A_SIGMA = (0.02, 0.01, 0.001)       # energy-scale a0,a1,a2 widths (BASELINE.json config 2)


def dc_edges() -> np.ndarray:
    """38 synthetic Double-Chooz-like bins on 1-20 MeV with widths that are multiples of 0.25 MeV.

    The paper gives only "1 MeV to 20 MeV with custom bin sizes ... 38 energy bins"
     and that 0.25 MeV is the greatest common divisor of the widths
    (41 uniform bins span 1-11.25 MeV).  These edges satisfy that and are
    NOT claimed to be the experiment's: 28 x 0.25 (1-8), 4 x 0.5 (8-10), 2 x 1 (10-12), 4 x 2 (12-20).
    """
    e = [1.0 + 0.25 * i for i in range(28)]
    e += [8.0 + 0.5 * i for i in range(4)]
    e += [10.0 + 1.0 * i for i in range(2)]
    e += [12.0 + 2.0 * i for i in range(5)]
    e = np.asarray(e, dtype=np.float64)
    assert e.shape[0] == 39 and e[-1] == 20.0
    return e


def reactor_events(rng: np.random.Generator, n: int, L_m, core_prob, resolution: float,
                   edges: np.ndarray, weights: str = "one") -> DatasetEvents:
    """Draw n MC events with a reactor-like E_nu shape and Gaussian energy smearing."""
    L_m = np.asarray(L_m, dtype=np.float64)
    e_nu = 1.8 + rng.gamma(5.0, 0.5, size=n)
    bad = e_nu >= 10.0
    while bad.any():
        e_nu[bad] = 1.8 + rng.gamma(5.0, 0.5, size=int(bad.sum()))
        bad = e_nu >= 10.0
    e_dep = e_nu - 0.782
    e_vis = e_dep + resolution * np.sqrt(e_dep) * rng.standard_normal(n)
    core_prob = np.asarray(core_prob, dtype=np.float64)
    core = rng.choice(len(L_m), size=n, p=core_prob / core_prob.sum()).astype(np.int32)
    if weights == "one":
        w = np.ones(n, dtype=np.float32)
    else:
        w = rng.uniform(0.5, 1.5, size=n).astype(np.float32)
    return DatasetEvents(e_nu=e_nu.astype(np.float32), e_vis=e_vis.astype(np.float32), w=w,
                         core=core, L_m=L_m, edges=np.asarray(edges, dtype=np.float64))


def poisson_counts(mu: np.ndarray, seed: int) -> np.ndarray:
    """Pseudo-data n ~ Poisson(mu) as float64 counts; `mu` comes from the caller."""
    rng = np.random.Generator(np.random.PCG64(seed))
    mu = np.asarray(mu, dtype=np.float64)
    return rng.poisson(np.clip(mu, 0.0, None)).astype(np.float64)


# ----------------------------------------------------------------------------------------------
# background templates (synthetic; PAPER.md:131-137 names the three kinds, not their shapes)
# ----------------------------------------------------------------------------------------------
def _template(edges: np.ndarray, kind: str, total: float) -> np.ndarray:
    c = 0.5 * (edges[1:] + edges[:-1])
    wdt = edges[1:] - edges[:-1]
    if kind == "accidental":
        s = np.exp(-c / 1.5)
    elif kind == "li9":
        s = c * c * np.exp(-c / 2.0)
    elif kind == "fastn":
        s = np.ones_like(c)
    else:
        raise ValueError(kind)
    s = s * wdt
    return total * s / s.sum()


def _flat_bkg(edges: np.ndarray, signal_total: float) -> BkgSpec:
    """Fixed (parameter-free) flat background at 1 % of the signal: keeps mu > 0 in bins the MC
    leaves empty for some energy-scale points, as the data-driven backgrounds do in the paper's
    background-dominated bins."""
    return BkgSpec(tmpl=_template(edges, "fastn", 0.01 * signal_total))


def _n(n_full: int, scale: float) -> int:
    return max(1, int(round(n_full * scale)))


# ----------------------------------------------------------------------------------------------
# configs
# ----------------------------------------------------------------------------------------------
def _config1(rng, scale, n_points):
    edges = 0.5 + np.arange(41, dtype=np.float64) * (19.5 / 40.0)
    ev = reactor_events(rng, _n(100_000, scale), [1050.0], [1.0], 0.08, edges)
    # theta = (s13, mee, s12, m21, a0, a1, a2)
    theta0 = np.array([THETA0["s13"], THETA0["mee"], THETA0["s12"], THETA0["m21"], 0.0, 1.0, 0.0])
    prior_mean = theta0.copy()
    prior_sigma = np.array([0.0, SIGMA0["mee"], SIGMA0["s12"], SIGMA0["m21"], *A_SIGMA])
    model = ModelSpec(osc_model=OSC_EQ1, n_params=7, idx_osc=(0, 1, 2, 3, -1, -1),
                      fixed_osc=(0, 0, 0, 0, 0.0, 0.0),
                      datasets=[DatasetSpec(n_bins=40, idx_a=(4, 5, 6), norm=1.0,
                                            bkg=[_flat_bkg(edges, 1.0 * ev.n)])],
                      prior_mean=prior_mean, prior_sigma=prior_sigma)
    P = 1 if n_points is None else n_points
    params = np.tile(theta0, (P, 1))
    if P > 1:
        params[1:] += rng.standard_normal((P - 1, 7)) * np.where(prior_sigma > 0, prior_sigma, SIGMA0["s13"])
    return model, [ev], params, theta0


def _dc_two_detector_events(rng, scale):
    edges = dc_edges()
    nd = reactor_events(rng, _n(1_000_000, scale), [355.0, 469.0], [0.5, 0.5], 0.08, edges)
    fd = reactor_events(rng, _n(1_000_000, scale), [998.0, 1115.0], [0.5, 0.5], 0.08, edges)
    return [nd, fd]


def _config2(rng, scale, n_points):
    evs = _dc_two_detector_events(rng, scale)
    # theta = (s13, mee, s12, m21, aND0..2, aFD0..2)
    theta0 = np.array([THETA0["s13"], THETA0["mee"], THETA0["s12"], THETA0["m21"],
                       0.0, 1.0, 0.0, 0.0, 1.0, 0.0])
    sig = np.array([SIGMA0["s13"], SIGMA0["mee"], SIGMA0["s12"], SIGMA0["m21"], *A_SIGMA, *A_SIGMA])
    prior_sigma = sig.copy()
    prior_sigma[0] = 0.0           # sin^2 2theta13 is left unconstrained
    model = ModelSpec(osc_model=OSC_EQ1, n_params=10, idx_osc=(0, 1, 2, 3, -1, -1),
                      fixed_osc=(0, 0, 0, 0, 0.0, 0.0),
                      datasets=[DatasetSpec(n_bins=38, idx_a=(4, 5, 6), norm=0.4,
                                            bkg=[_flat_bkg(evs[0].edges, 0.4 * evs[0].n)]),
                                DatasetSpec(n_bins=38, idx_a=(7, 8, 9), norm=0.1,
                                            bkg=[_flat_bkg(evs[1].edges, 0.1 * evs[1].n)])],
                      prior_mean=theta0.copy(), prior_sigma=prior_sigma)
    P = 64 if n_points is None else n_points
    params = theta0[None, :] + rng.standard_normal((P, 10)) * sig[None, :]
    return model, evs, params, theta0


def _config3(rng, scale, n_points):
    edges = dc_edges()
    B = 38
    n_ev = _n(2_000_000, scale)
    evs = [reactor_events(rng, n_ev, [998.0, 1115.0], [0.5, 0.5], 0.08, edges),   # FD-I
           reactor_events(rng, n_ev, [998.0, 1115.0], [0.5, 0.5], 0.08, edges),   # FD-II
           reactor_events(rng, n_ev, [355.0, 469.0], [0.5, 0.5], 0.08, edges)]    # ND
    norms = (0.02, 0.05, 0.2)
    # parameter layout (301): 4 osc | 9 energy-scale | 114 flux | 3 signal norms | 9 bkg rates |
    #                         114 accidental shape | 38 shared Li shape | 10 shared fast-n shape groups
    o_a, o_flux, o_norm, o_rate = 4, 13, 127, 130
    o_acc, o_li, o_fn = 139, 253, 291
    NPAR = 301
    mean = np.zeros(NPAR)
    sigma = np.zeros(NPAR)
    mean[0:4] = [THETA0["s13"], THETA0["mee"], THETA0["s12"], THETA0["m21"]]
    sigma[0:4] = [0.0, SIGMA0["mee"], SIGMA0["s12"], SIGMA0["m21"]]       # s13 free
    for d in range(3):
        mean[o_a + 3 * d: o_a + 3 * d + 3] = (0.0, 1.0, 0.0)
        sigma[o_a + 3 * d: o_a + 3 * d + 3] = A_SIGMA
    mean[o_flux:o_flux + 3 * B] = 1.0
    sigma[o_flux:o_flux + 3 * B] = 0.02
    mean[o_norm:o_norm + 3] = 1.0
    sigma[o_norm:o_norm + 3] = 0.01
    mean[o_rate:o_rate + 9] = 1.0
    # per dataset (accidental, Li, fast-n): accidental constrained,
    # Li rate free, fast-n loosely constrained
    sigma[o_rate:o_rate + 9] = np.tile([0.01, 0.0, 0.1], 3)
    mean[o_acc:o_acc + 3 * B] = 1.0
    sigma[o_acc:o_acc + 3 * B] = 0.02
    mean[o_li:o_li + B] = 1.0
    sigma[o_li:o_li + B] = 0.05
    mean[o_fn:o_fn + 10] = 1.0
    sigma[o_fn:o_fn + 10] = 0.1
    fn_group = (np.arange(B) * 10 // B).astype(np.int32)

    dsets = []
    for d in range(3):
        sig_total = norms[d] * n_ev
        bk = [BkgSpec(tmpl=_template(edges, "accidental", 0.01 * sig_total), idx_rate=o_rate + 3 * d + 0,
                      idx_shape=(o_acc + B * d + np.arange(B)).astype(np.int32)),
              BkgSpec(tmpl=_template(edges, "li9", 0.02 * sig_total), idx_rate=o_rate + 3 * d + 1,
                      idx_shape=(o_li + np.arange(B)).astype(np.int32)),
              BkgSpec(tmpl=_template(edges, "fastn", 0.01 * sig_total), idx_rate=o_rate + 3 * d + 2,
                      idx_shape=(o_fn + fn_group).astype(np.int32))]
        dsets.append(DatasetSpec(n_bins=B, idx_a=(o_a + 3 * d, o_a + 3 * d + 1, o_a + 3 * d + 2),
                                 idx_signorm=o_norm + d, norm=norms[d],
                                 idx_flux=(o_flux + B * d + np.arange(B)).astype(np.int32), bkg=bk))
    model = ModelSpec(osc_model=OSC_EQ1, n_params=NPAR, idx_osc=(0, 1, 2, 3, -1, -1),
                      fixed_osc=(0, 0, 0, 0, 0.0, 0.0), datasets=dsets,
                      prior_mean=mean, prior_sigma=sigma)
    # expansion point: nuisances drawn once around their prior centres (pulls are non-zero)
    draw_sigma = np.where(sigma > 0, sigma, 0.0)
    draw_sigma[0] = SIGMA0["s13"]
    theta0 = mean + rng.standard_normal(NPAR) * draw_sigma
    # central-difference batch {theta0} U {theta0 +- h_j e_j}: 2*301 + 1 = 603 points
    h = np.where(sigma > 0, 0.01 * sigma, 1e-3)
    params = np.tile(theta0, (2 * NPAR + 1, 1))
    for j in range(NPAR):
        params[1 + 2 * j, j] += h[j]
        params[2 + 2 * j, j] -= h[j]
    if n_points is not None:
        # keep the centre and the first (n_points-1) shifted points: oscillation and energy-scale first
        params = params[:n_points]
    return model, evs, params, theta0


def _config4(rng, scale, n_points, ordering=+1):
    edges = 0.8 + np.arange(411, dtype=np.float64) * 0.02
    L = [52_000.0 + 100.0 * i for i in range(9)] + [215_000.0, 265_000.0]
    prob = [0.1] * 9 + [0.05, 0.05]
    ev = reactor_events(rng, _n(10_000_000, scale), L, prob, 0.03, edges)
    theta0 = np.array([THETA0["s13"], THETA0["mee"], THETA0["s12"], THETA0["m21"]])
    sig = np.array([SIGMA0["s13"], SIGMA0["mee"], SIGMA0["s12"], SIGMA0["m21"]])
    model = ModelSpec(osc_model=OSC_FULL3, ordering=ordering, n_params=4, idx_osc=(0, 1, 2, 3, -1, -1),
                      fixed_osc=(0, 0, 0, 0, 0.0, 0.0),
                      datasets=[DatasetSpec(n_bins=410, norm=0.05)],
                      prior_mean=theta0.copy(), prior_sigma=np.zeros(4))   # no systematics
    P = 128 if n_points is None else n_points
    params = theta0[None, :] + rng.standard_normal((P, 4)) * sig[None, :]
    return model, [ev], params, theta0


def _config5(rng, scale, n_points):
    evs = _dc_two_detector_events(rng, scale)
    theta0 = np.array([THETA0["s13"], THETA0["mee"], THETA0["s12"], THETA0["m21"], 0.0, 1.0])
    model = ModelSpec(osc_model=OSC_STERILE4, n_params=6, idx_osc=(0, 1, 2, 3, 4, 5),
                      fixed_osc=(0, 0, 0, 0, 0.0, 0.0),
                      datasets=[DatasetSpec(n_bins=38, norm=0.4, bkg=[_flat_bkg(evs[0].edges, 0.4 * evs[0].n)]),
                                DatasetSpec(n_bins=38, norm=0.1, bkg=[_flat_bkg(evs[1].edges, 0.1 * evs[1].n)])],
                      prior_mean=theta0.copy(),
                      prior_sigma=np.array([0.0, SIGMA0["mee"], SIGMA0["s12"], SIGMA0["m21"], 0.0, 0.0]))
    g = 64
    s14 = np.logspace(np.log10(1e-3), np.log10(0.3), g)
    m41 = np.logspace(-2.0, 1.0, g)
    S, M = np.meshgrid(s14, m41, indexing="ij")
    params = np.tile(theta0, (g * g, 1))
    params[:, 4] = S.ravel()
    params[:, 5] = M.ravel()
    if n_points is not None:
        sel = np.linspace(0, g * g - 1, n_points).round().astype(int)
        params = params[sel]
    return model, evs, params, theta0


_BUILDERS = {1: _config1, 2: _config2, 3: _config3, 4: _config4, 5: _config5}


def make_config(k: int, seed: int | None = None, scale: float = 1.0,
                n_points: int | None = None, ordering: int = +1) -> Workload:
    """BASELINE.json config k (1-based).  `scale` shrinks the event counts and `n_points`
    truncates the batch, for parity cases the oracle finishes in seconds.  `ordering` = -1 turns
    config 4 (the only one with the full 3-flavour P_ee) to the inverted mass ordering;
    the same events and points, BASELINE.json's config 4 itself is the normal ordering."""
    seed = DEFAULT_SEEDS[k] if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    if k == 4:
        model, evs, params, theta0 = _config4(rng, scale, n_points, ordering)
    else:
        if ordering != +1:
            raise ValueError("only config 4 (FULL3) has a mass ordering")
        model, evs, params, theta0 = _BUILDERS[k](rng, scale, n_points)
    return Workload(name=CONFIG_NAMES[k], model=model, events=evs,
                    params=np.ascontiguousarray(params, dtype=np.float64),
                    theta0=np.asarray(theta0, dtype=np.float64), seed=seed,
                    note=f"config {k}, scale {scale}, points {params.shape[0]}")


def make_tiny(seed: int, osc_model: int = OSC_EQ1, n_events: int = 100, n_points: int = 5,
              n_datasets: int = 1, ordering: int = +1) -> Workload:
    """<= 100 events per dataset, U(0.5,1.5) weights, 3 cores, 7 non-uniform bins: brute-force size."""
    rng = np.random.Generator(np.random.PCG64(seed))
    edges = np.array([1.0, 1.5, 2.25, 3.0, 3.5, 4.75, 6.0, 9.0])
    L = [400.0, 1050.0, 52_500.0] if osc_model == OSC_FULL3 else [355.0, 469.0, 1050.0]
    evs = [reactor_events(rng, n_events, L, [0.3, 0.3, 0.4], 0.08, edges, weights="uniform")
           for _ in range(n_datasets)]
    n_osc = 6
    npar = n_osc + 3 * n_datasets + 1 + 7     # osc | a per dataset | one rate | 7 shared shape params
    theta0 = np.zeros(npar)
    theta0[:6] = [THETA0["s13"], THETA0["mee"], THETA0["s12"], THETA0["m21"], 0.05, 0.5]
    sig = np.zeros(npar)
    sig[:6] = [SIGMA0["s13"], SIGMA0["mee"], SIGMA0["s12"], SIGMA0["m21"], 0.01, 0.05]
    dsets = []
    o_rate = n_osc + 3 * n_datasets
    o_shape = o_rate + 1
    theta0[o_rate] = 1.0
    sig[o_rate] = 0.1
    theta0[o_shape:o_shape + 7] = 1.0
    sig[o_shape:o_shape + 7] = 0.05
    for d in range(n_datasets):
        o = n_osc + 3 * d
        theta0[o:o + 3] = (0.0, 1.0, 0.0)
        sig[o:o + 3] = A_SIGMA
        bk = [BkgSpec(tmpl=_template(edges, "li9", 3.0), idx_rate=o_rate,
                      idx_shape=(o_shape + np.arange(7)).astype(np.int32)),
              BkgSpec(tmpl=_template(edges, "fastn", 1.0))]
        dsets.append(DatasetSpec(n_bins=7, idx_a=(o, o + 1, o + 2), norm=0.7 + 0.1 * d, bkg=bk))
    prior_sigma = sig.copy()
    prior_sigma[0] = 0.0
    model = ModelSpec(osc_model=osc_model, n_params=npar, idx_osc=(0, 1, 2, 3, 4, 5),
                      fixed_osc=(0,) * 6, datasets=dsets, ordering=ordering, prior_mean=theta0.copy(),
                      prior_sigma=prior_sigma)
    params = theta0[None, :] + rng.standard_normal((n_points, npar)) * sig[None, :]
    params[0] = theta0
    return Workload(name=f"tiny_{osc_model}", model=model, events=evs,
                    params=np.ascontiguousarray(params), theta0=theta0, seed=seed,
                    note="tiny brute-force input")
