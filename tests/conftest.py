import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    # The built libraries are git-ignored: (re)build them in-tree before any test imports the binding.
    # nvcc cross-compiles sm_100a without a GPU; the oracle is plain C (gcc).
    from paper_2606_06302_b200 import build as _build
    _build.build(force=False)
    from oracle import tangram_oracle as _oracle
    _oracle.build_c()


def pytest_collection_modifyitems(config, items):
    # GPU tests are selected with `-m gpu`; if they are collected on a box without a device
    # (plain `pytest tests/`), skip them instead of failing on the missing driver.
    try:
        import torch
        has = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has = False
    if has:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
