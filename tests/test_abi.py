"""CPU-side checks of the boundary: the shared library builds/loads and exports every symbol include/dlr.h
declares; host-side logic that needs no GPU (configuration validation, workspace sizing, error strings)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2110_13481_b200 import build, dlr
    build.build()
    return dlr.lib()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "dlr.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(dlr_[a-z_0-9]+)\s*\(", hdr))
    assert {"dlr_create", "dlr_set_initial", "dlr_step", "dlr_moments", "dlr_destroy"} <= names
    for n in names:
        assert hasattr(lib, n), n


def test_config_validation_and_workspace_size(lib):
    from paper_2110_13481_b200 import dlr, inputs
    # about six factor-sized arrays (X, X1, V, KL, Q1, W) plus the field and the r x r work
    for idx, lo, hi in ((1, 1e5, 1e7), (3, 1.2e8, 5e8), (5, 1.5e10, 4e10)):
        nbytes = dlr.dlr_workspace_bytes(dlr.config_from_inputs(inputs.make_config(idx)))
        assert lo < nbytes < hi
    bad = dlr.make_config(8, 8, 0.0, 1.0, -1.0, 1.0, 5)
    bad.order = 3
    with pytest.raises(dlr.DlrError):
        dlr.dlr_workspace_bytes(bad)
    for n, r in ((4, 5), (512, 5), (24, 5), (8, 6)):
        with pytest.raises(dlr.DlrError) as e:
            dlr.dlr_workspace_bytes(dlr.make_config(n, n, 0.0, 1.0, -1.0, 1.0, r))
        assert e.value.code == -2
    assert lib.dlr_strerror(-5).decode().startswith("initial factors")


def test_product_path_fails_loudly_without_gpu(lib):
    import torch
    from paper_2110_13481_b200 import dlr, inputs
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        dlr.Dlr(dlr.config_from_inputs(inputs.make_config(1)))
