"""Stored oracle results (tests/golden/, written by tests/golden/make_golden.py from the oracle alone).

not gpu: the oracle as it stands still reproduces them (to 1e-12 relative; a change of its arithmetic must come with
regenerated fixtures and a commit message naming the passage that justifies it).
gpu: the CUDA path meets the parity bars against the stored numbers.
"""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
_spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
make_golden = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(make_golden)


def _read(name):
    hist, nll = [], None
    for line in open(os.path.join(HERE, "golden", f"tiny_{name}.txt")):
        if line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "hist":
            hist.append([float.fromhex(x) for x in tok[2:]])
        elif tok[0] == "nll":
            nll = [float.fromhex(x) for x in tok[1:]]
    return np.array(hist), np.array(nll)


@pytest.mark.parametrize("name", sorted(make_golden.CASES))
def test_oracle_reproduces_golden(oracle_mod, name):
    wl, data = make_golden.case_inputs(name)
    orc = oracle_mod.Oracle(wl.model, wl.events)
    hist, nll = _read(name)
    # 1e-12: room for another libm build only; on this image the match is exact
    assert np.allclose(orc.spectra(wl.params), hist, rtol=1e-12, atol=0.0)
    assert np.allclose(orc.nll(wl.params, data), nll, rtol=1e-12, atol=0.0)


@pytest.mark.gpu
@pytest.mark.parametrize("name", sorted(make_golden.CASES))
def test_gpu_matches_golden(gpu, name):
    import torch
    wl, data = make_golden.case_inputs(name)
    hist, nll = _read(name)
    with gpu.Phylino() as ph:
        ph.load_workload(wl)
        dp = torch.as_tensor(wl.params, device="cuda")
        h = ph.spectra(dp).cpu().numpy()
        v = ph.nll(dp, torch.as_tensor(data, device="cuda")).cpu().numpy()
    nz = hist != 0
    assert np.array_equal(h[~nz], hist[~nz])
    assert (np.abs(h - hist)[nz] / np.abs(hist[nz])).max() <= 1e-7
    assert np.abs(v - nll).max() <= 1e-6
