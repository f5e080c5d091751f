import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


def pytest_collection_modifyitems(config, items):
    """GPU tests are skipped (not failed) on a machine without a device, so a bare `pytest tests`
    on the CPU box stays green; `-m gpu` on a GPU box runs them."""
    try:
        import torch
        have_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        have_gpu = False
    if have_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture
def solver_path(request):
    """Which of the two drivers of the CG iteration a test runs on (helpers.both_solvers parametrizes it):
    "launches" = two launches per iteration, as a CUDA graph or plainly (what large lattices get);
    "persistent" = the whole solve in one cooperative kernel (what lattices that live in L2 get by default)."""
    import paper_1801_01473_b200 as lq
    mode = getattr(request, "param", "auto")
    saved = dict(lq.Lattice.default_options)
    if mode == "launches":
        lq.Lattice.default_options[lq.LQCD_OPT_PERSISTENT] = 0
    elif mode == "persistent":
        lq.Lattice.default_options[lq.LQCD_OPT_PERSISTENT] = 1
    yield mode
    lq.Lattice.default_options.clear()
    lq.Lattice.default_options.update(saved)
