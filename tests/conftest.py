import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_sessionstart(session):
    """FORGE_TEST_PROFILING_LIB=1 runs the whole suite against libforge_b200_prof.so (the -DFORGE_PROFILING build), so
    that a candidate instantiation selected with FORGE_CFG=<n> can be put through the parity tests before it is
    promoted to the product dispatch table.  Unset (the default and what the driver runs): the product library."""
    if os.environ.get("FORGE_TEST_PROFILING_LIB") == "1":
        from paper_2606_22932_b200 import binding
        binding.use_profiling_library(True)
