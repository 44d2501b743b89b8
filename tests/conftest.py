import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (run with -m gpu on the GPU box)")
    config.addinivalue_line("markers", "slow: long-running parity case (full-size config)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(autouse=True)
def _captured_graphs_released(request):
    """Tests that capture a step into a CUDA graph drop the graph when they return.  The library pins a captured plan and
    its workspace until it is told the graphs are gone (include/dmuon.h, "CUDA graphs"): tell it after every GPU test."""
    yield
    if "gpu" in request.node.keywords:
        import gc
        gc.collect()
        import paper_2606_27153_b200 as dm
        dm.set_option("graphs_destroyed", 1)
