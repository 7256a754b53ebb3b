"""Seeded synthetic inputs shaped like the paper's Double Chooz and JUNO-like workloads.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2502_15253_b200/`).  It holds none of the method's arithmetic: no survival
probability, no energy-scale map, no binning, no likelihood.  It only draws random
event lists, lays out parameter vectors and index maps, and draws Poisson counts from
an expectation that the caller hands in.

The paper's own inputs (Double Chooz MC + data; the JUNO-like rescaling,
PAPER.md:228) are not public; the recipes here take their shapes, sizes and value
distributions from PAPER.md (§3.2–3.3, §4.1, §4.3) and BASELINE.json `configs` and stand
in for them.  The recipes are restated in DESIGN.md §"Input recipe".
"""
from .spec import (BkgSpec, DatasetSpec, DatasetEvents, FluxModel, FunctionSpec, ModelSpec, PriorBlock, TransformBlock,  # noqa: F401
                   TransformSpec, Workload)
from .generate import (  # noqa: F401
    CONFIG_NAMES,
    THETA0,
    dc_edges,
    make_config,
    make_tiny,
    poisson_counts,
    reactor_events,
)
