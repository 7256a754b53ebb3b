"""Writes the stored expected values under tests/golden/ -- calls ONLY oracle/ and workloads/.

    python tests/golden/make_golden.py

The paper prints no numeric spectrum or likelihood value, so these fixtures are not the
paper's: they are the CPU oracle's results on seeded tiny inputs (<= 100 events per dataset, the brute-force
size), frozen so that (i) a later change of the oracle's arithmetic shows up as a diff that its commit message
has to justify, and (ii) the CUDA path is compared with numbers that no run of the CUDA path produced.
One file per oscillation model; every value as a C99 hex float (exact).
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
import workloads  # noqa: E402

# name -> (osc_model, seed, mass ordering); full3_inv: PAPER.md:226 (section 4.3), the inverted-ordering branch
CASES = {"eq1": (0, 611, +1), "full3": (1, 612, +1), "sterile4": (2, 613, +1), "full3_inv": (1, 614, -1)}


def case_inputs(name):
    osc, seed, ordering = CASES[name]
    wl = workloads.make_tiny(seed=seed, osc_model=osc, n_events=100, n_points=5, n_datasets=2, ordering=ordering)
    data = np.arange(wl.model.total_bins, dtype=np.float64) * 3.0 + 2.0
    return wl, data


def main():
    oracle.build()
    for name in CASES:
        wl, data = case_inputs(name)
        orc = oracle.Oracle(wl.model, wl.events)
        hist = orc.spectra(wl.params)
        nll = orc.nll(wl.params, data)
        path = os.path.join(HERE, f"tiny_{name}.txt")
        with open(path, "w") as f:
            f.write(f"# oracle results, workloads.make_tiny(seed={CASES[name][1]}, osc_model={CASES[name][0]}, "
                    f"n_events=100, n_points=5, n_datasets=2"
                    + (f", ordering={CASES[name][2]}" if CASES[name][2] != 1 else "") + "); data[i] = 3 i + 2\n")
            f.write("# written by tests/golden/make_golden.py (oracle only); P_ee: PAPER.md:34 Eq. 1 / DESIGN.md R2, R15;\n")
            f.write("# NLL: PAPER.md:67-83 Eq. 3-6, :119-125 Eq. 9.  Rows: 'hist p' then total_bins values; 'nll' then P values\n")
            for p in range(hist.shape[0]):
                f.write(f"hist {p} " + " ".join(float(x).hex() for x in hist[p]) + "\n")
            f.write("nll " + " ".join(float(x).hex() for x in nll) + "\n")
        print(path)


if __name__ == "__main__":
    main()
