"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/phylino.h declares, and refuses to create a context without a CUDA device (no fallback).
No compute call is made here."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "phylino.h")


def _declared():
    src = open(HEADER).read()
    return sorted(set(re.findall(r"PHYLINO_API\s+[\w\s\*]+?\b(phylino_\w+)\s*\(", src)))


def test_header_declares_the_boundary():
    names = _declared()
    for must in ("phylino_create", "phylino_destroy", "phylino_set_model", "phylino_load_events",
                 "phylino_spectra", "phylino_nll", "phylino_last_error"):
        assert must in names
    assert len(names) >= 12


def test_library_exports_every_declared_symbol(phylino_lib):
    lib = phylino_lib.load_library()
    declared = _declared()
    assert sorted(phylino_lib.abi_symbols) == declared
    out = subprocess.run(["nm", "-D", "--defined-only", phylino_lib.lib_path()], capture_output=True,
                         text=True, check=True).stdout
    exported = set(re.findall(r"\sT\s+(\w+)", out))
    for name in declared:
        assert name in exported, name
        assert getattr(lib, name) is not None
    # nothing but the ABI is exported
    assert exported == set(declared)


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "phylino.h"\nint main(void){ phylino_model_desc m; (void)m; return PHYLINO_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_no_cpu_fallback(phylino_lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    lib = phylino_lib.load_library()
    ctx = C.c_void_p()
    assert lib.phylino_create(0, None, C.byref(ctx)) == 5          # PHYLINO_ERR_CUDA
    assert not ctx
    with pytest.raises(phylino_lib.PhylinoError):
        phylino_lib.Phylino()


def test_null_context_is_rejected(phylino_lib):
    lib = phylino_lib.load_library()
    assert lib.phylino_total_bins(None) == 0
    assert lib.phylino_total_events(None) == 0
    assert lib.phylino_launch_count(None) == 0
    assert lib.phylino_last_error(None) == b""
    assert lib.phylino_set_tuning(None, 512, 0, 0) == 1               # PHYLINO_ERR_ARG
    assert lib.phylino_set_caching(None, 1) == 1
    assert lib.phylino_launch_floor(None, 1, None) == 1
    assert lib.phylino_set_transform(None, 0, None, None, 0, None) == 1
    assert lib.phylino_param_width(None) == 0
    assert lib.phylino_nll_ensemble(None, 1, None, 1, None, None) == 1
    assert lib.phylino_set_prior_blocks(None, 0, None) == 1
    assert lib.phylino_spectra(None, 1, None, None) == 1
    lib.phylino_destroy(None)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2502_15253_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text, (f, "product path must not touch the test oracle")
    assert "oracle" not in open(HEADER).read()
