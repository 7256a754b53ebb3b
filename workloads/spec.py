"""Plain data containers describing a fit model and its inputs (no arithmetic).

Names follow the paper: datasets d, bins i, parameter
vector theta, signal/background contributions.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

# oscillation models (BASELINE.json configs 1-3 / 4 / 5)
OSC_EQ1 = 0        # PAPER.md:34 Eq. 1 (two terms)
OSC_FULL3 = 1      # exact 3-flavour vacuum P_ee with dm31, dm32 (config 4; Eq. 2 inverted)
OSC_STERILE4 = 2   # 3+1 extension (formula from BASELINE.json config 5)

# slots of the six oscillation parameters in idx_osc / fixed_osc
S13, MEE, S12, M21, S14, M41 = range(6)   # sin^2 2theta13, dm2_ee, sin^2 2theta12, dm2_21, sin^2 2theta14, dm2_41


@dataclass
class BkgSpec:
    """One background contribution of one dataset: rate * shape_i * template_i."""
    tmpl: np.ndarray                       # float64 [n_bins] expected counts at rate = shape = 1
    idx_rate: int = -1                     # index into theta, -1 => 1
    idx_shape: Optional[np.ndarray] = None  # int32 [n_bins] indices into theta (-1 => 1), None => all 1


@dataclass
class FluxModel:
    """Reactor-flux nuisance model of one dataset on a uniform fine grid (41 parameters on 0.25-MeV bins
    from 1 to 11.25 MeV): theta[idx_par[j]] is the average flux correction on [lo + j width, lo + (j+1) width)."""
    idx_par: np.ndarray       # int32 [n] indices into theta
    lo: float = 1.0
    width: float = 0.25


@dataclass
class DatasetSpec:
    """How theta acts on one dataset's signal spectrum and backgrounds."""
    n_bins: int
    idx_a: tuple = (-1, -1, -1)            # energy-scale a0,a1,a2; -1 => (0,1,0)
    idx_signorm: int = -1                  # detection-efficiency-like multiplier; -1 => 1
    norm: float = 1.0                      # constant MC -> data normalisation
    idx_flux: Optional[np.ndarray] = None  # int32 [n_bins] per-bin flux scale; None => all 1
    bkg: List[BkgSpec] = field(default_factory=list)
    flux_model: Optional[FluxModel] = None  # replaces idx_flux: fine-grid parameters -> per-bin scales (R28)


@dataclass
class DatasetEvents:
    """MC event list of one dataset in the caller's (unsorted) order."""
    e_nu: np.ndarray      # float32 [n] true neutrino energy, MeV
    e_vis: np.ndarray     # float32 [n] reconstructed (visible) energy, MeV
    w: np.ndarray         # float32 [n] MC weight
    core: np.ndarray      # int32 [n] reactor-core index (two reactors => two baselines)
    L_m: np.ndarray       # float64 [n_cores] baseline per core, metres
    edges: np.ndarray     # float64 [n_bins+1] strictly ascending reco-energy bin edges, MeV

    @property
    def n(self) -> int:
        return int(self.e_nu.shape[0])

    @property
    def n_bins(self) -> int:
        return int(self.edges.shape[0] - 1)


@dataclass
class PriorBlock:
    """One correlated Gaussian constraint (Eq. 9 third factor): parameters idx with
    central values mean and INVERSE covariance inv_cov (row-major [n, n], symmetric)."""
    idx: np.ndarray           # int32 [n] indices into theta
    mean: np.ndarray          # float64 [n]
    inv_cov: np.ndarray       # float64 [n, n]


@dataclass
class FunctionSpec:
    """A constrained quantity that is a function of the fitted parameters (R29):
    b(theta) = offset + sum over terms of coef * prod_i theta[idx_i] ** power_i, integer powers.  A PriorBlock
    refers to function f of the model through the index n_params + f."""
    terms: list               # [(coef, idx int32 [k], power int32 [k]), ...]
    offset: float = 0.0


@dataclass
class TransformBlock:
    """theta[idx_out] = offset + matrix (u[idx_in] - centre): one block of the transformation layer between the
    minimiser's parameters u and the model parameters theta (the 9 <- 7 energy-response map of
    PAPER.md:141 is a 9 x 7 block, a Cholesky factor of a covariance a square one)."""
    idx_out: np.ndarray       # int32 [n_out] indices into theta
    idx_in: np.ndarray        # int32 [n_in] indices into u
    offset: np.ndarray        # float64 [n_out]
    centre: np.ndarray        # float64 [n_in]
    matrix: np.ndarray        # float64 [n_out, n_in]


@dataclass
class TransformSpec:
    n_u: int                  # length of the minimiser's parameter vector
    copy_src: np.ndarray      # int32 [n_params]: theta_j = u[copy_src[j]], or copy_const[j] where copy_src[j] < 0
    copy_const: np.ndarray    # float64 [n_params]
    blocks: List[TransformBlock] = field(default_factory=list)


@dataclass
class ModelSpec:
    osc_model: int
    n_params: int
    idx_osc: tuple                          # 6 indices into theta, -1 => use fixed_osc
    fixed_osc: tuple                        # 6 fixed values
    datasets: List[DatasetSpec]
    ordering: int = +1                      # +1 normal, -1 inverted (FULL3 only)
    prior_mean: Optional[np.ndarray] = None   # float64 [n_params]
    prior_sigma: Optional[np.ndarray] = None  # float64 [n_params]; <= 0 or inf => unconstrained
    prior_blocks: List[PriorBlock] = field(default_factory=list)
    functions: List[FunctionSpec] = field(default_factory=list)   # constrained functions of theta
    energy_correction: int = 0              # 0: per event before binning (north_star); 1: on the bins (PAPER.md:177 step 3)

    @property
    def total_bins(self) -> int:
        return sum(d.n_bins for d in self.datasets)


@dataclass
class Workload:
    name: str
    model: ModelSpec
    events: List[DatasetEvents]
    params: np.ndarray        # float64 [P, n_params] batch of parameter points
    theta0: np.ndarray        # float64 [n_params] the point pseudo-data is drawn at
    seed: int
    note: str = ""

    @property
    def n_points(self) -> int:
        return int(self.params.shape[0])

    @property
    def n_events(self) -> int:
        return sum(e.n for e in self.events)
