import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: longer statistical test")
    # a fresh checkout has no binaries: build the CUDA library (nvcc cross-compiles without a GPU) and the oracle
    # once if they are missing; an existing build is left alone (rebuild with __graft_entry__.build())
    from paper_2405_05700_b200 import build as pp_build
    if not os.path.exists(pp_build.LIB):
        pp_build.build(force=True)
    from oracle import oracle as O
    O.build()


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) on a GPU box without the extension; on a CPU box they are
    deselected by ``-m "not gpu"``.  If someone runs the whole suite on a CPU box, skip them."""
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
