import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
    config.addinivalue_line("markers", "sanitizer: the small-lattice subset of the gpu tests that is run under "
                                       "compute-sanitizer (README; profiles/sanitizer_r03.md)")


# `compute-sanitizer --tool memcheck|racecheck|synccheck --target-processes all python -m pytest tests -m sanitizer`:
# between them these tests launch every kernel variant of the library -- dslash_kernel EPI 0/2/4/5 x full / two-row
# links x U(1) phases x whole lattice / slab interior / slab border x scalar step inside the sweep or not, in double and
# single precision; the persistent cooperative kernel; the block sweeps cg_flush_kernel<4/8/16/32> and the ticket that
# closes a block; the mixed-precision kernels; both slab transports on one rank and two ranks over peer memory (with
# and without the kernel-signal fall-back); lqcd_mdagm_static -- on lattices small enough for a tool that slows every
# kernel down 10-100x.
_SANITIZER_TESTS = {
    "test_dslash_doe_then_deo", "test_mshift_cg_small", "test_rational_apply_small", "test_dslash_with_u1_phases",
    "test_mshift_cg_with_u1_phases", "test_dslash_f32", "test_mshift_cg_f32", "test_mixed_solver_matches_oracle",
    "test_one_rank_slab_operators_and_cg", "test_slab_with_u1_phases", "test_peer_memory_kernel_signal_fallback",
    "test_two_ranks_share_the_gpu_over_peer_memory", "test_stop_in_the_middle_of_a_block",
    "test_static_matches_mdagm_on_two_calls_in_a_row",
}
_SANITIZER_MAX_SITES = 2000


def _in_sanitizer_subset(item) -> bool:
    if getattr(item, "originalname", item.name) not in _SANITIZER_TESTS:
        return False
    params = getattr(getattr(item, "callspec", None), "params", {})
    L = params.get("L")
    sites = L[0] * L[1] * L[2] * L[3] if L is not None else 0
    if sites > _SANITIZER_MAX_SITES:
        return False
    mode = params.get("mode")
    if mode is not None and mode not in ("graph", "recon12"):
        return False
    if sites > 300 and mode == "recon12":                       # whole solves: the ragged 4x6x8x10 lattice once per driver
        return False
    if "n_iter" in params and params["n_iter"] != 17:          # one stop position inside a block is enough here
        return False
    return True


def pytest_collection_modifyitems(config, items):
    """GPU tests are skipped (not failed) on a machine without a device, so a bare `pytest tests`
    on the CPU box stays green; `-m gpu` on a GPU box runs them."""
    for item in items:
        if _in_sanitizer_subset(item):
            item.add_marker(pytest.mark.sanitizer)
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
