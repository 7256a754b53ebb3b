"""B200-native hot path of PhyLiNO's forward-folding likelihood fit (arXiv 2502.15253):
oscillation-weighted MC event spectra batched over parameter points, and the binned Poisson
negative log-likelihood with Gaussian priors.

The product is the C-ABI library `libphylino.so` (include/phylino.h, csrc/).  This package is a
thin ctypes binding with the same entry-point names; every step of the path runs in the CUDA
kernels.  There is no CPU fallback: importing works without a GPU (so the ABI can be inspected),
creating a context does not.
"""
from .binding import (  # noqa: F401
    Phylino,
    PhylinoError,
    abi_symbols,
    lib_path,
    load_library,
    variable_metric_step_static,
)
