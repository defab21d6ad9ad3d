import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: takes more than a few seconds on CPU")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


@pytest.fixture(autouse=True)
def _default_library_options():
    """the library's process-wide test switches (gimbal_set_option) are back at their defaults after every test"""
    yield
    try:
        import paper_2606_15177_b200 as g
        if os.path.exists(g.lib_path()):
            for opt, val in ((g.OPT_CTA_GROUP, 0), (g.OPT_FUSE_GATE, 1), (g.OPT_SCORE_GENERIC, 0), (g.OPT_CHECK_SCORES_ALL, 0), (g.OPT_HIST_AGG, 1), (g.OPT_SCORE_TMA, 1), (g.OPT_EPI_PARTS, 0), (g.OPT_PDL, 1), (g.OPT_FUSE_UPDATE, 1)):
                g.set_option(opt, val)
    except Exception:
        pass
