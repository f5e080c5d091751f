"""Block-deferred shift updates (LQCD_OPT_SHIFT_BLOCK = m): the x_i, p_i of the
systems (for m >= 2 the base system's x_0 too) are updated once per block of m iterations from the m residuals
of the block.

What must hold, and is checked against the CPU oracle (which follows SURVEY.md §8(c2) iteration by iteration
and knows nothing about blocks):
  * the base recurrence (r, p, a, beta, zeta_i, freezing, stopping) is untouched by m: iteration counts, freeze
    schedule and the final residual are IDENTICAL for every m, bit for bit;
  * every x_i agrees with the oracle to the usual bar (1e-8; 1e-11 at a fixed iteration count), whatever m, also
    when the stop / MAX_ITER / a freeze falls in the middle of a block, when m exceeds the iteration count, in
    rational-sum mode, with plain launches instead of the graph, and in single precision.
"""
from __future__ import annotations

import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle
from helpers import both_solvers, make_inputs, oracle_parity_vector, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu

TOL_CG = 1e-8       # BASELINE north_star: CG solutions within 1e-8 relative L2 of the oracle's


def cuda(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def rational_coefficients(n):
    """alpha_i of mixed sign and size (seeded; not a particular rational approximation)."""
    rng = np.random.default_rng(7)
    return 0.37, list(rng.uniform(0.05, 1.5, n) * rng.choice([-1.0, 1.0], n))

BLOCKS = [1, 2, 3, 4, 5, 8, 11, 16, 23, 32]


@pytest.fixture(scope="module")
def lq():
    import paper_1801_01473_b200 as lq
    lq.load_library()
    return lq


def solve(lq, lat, b, shifts, tol, m, use_graph=True, max_iter=None):
    lat.set_option(lq.LQCD_OPT_SHIFT_BLOCK, m)
    lat.set_option(lq.LQCD_OPT_USE_GRAPH, 1 if use_graph else 0)
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 100000 if max_iter is None else max_iter)
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg(b, shifts, tol, raise_on_noconv=False)
    torch.cuda.synchronize()
    return x, info


def test_option_range(lq):
    lat = lq.Lattice((4, 4, 4, 4))
    assert lat.get_option(lq.LQCD_OPT_SHIFT_BLOCK) == 16          # chosen by the library: a lattice that lives in L2
    big = lq.Lattice((32, 32, 32, 32))
    assert big.get_option(lq.LQCD_OPT_SHIFT_BLOCK) == 32          # ... and one that does not
    big.close()
    for bad in (33, 2.5, -1):
        assert lq.lqcd_set_option(lat.ctx, lq.LQCD_OPT_SHIFT_BLOCK, bad) == lq.LQCD_EINVAL
    lat.set_option(lq.LQCD_OPT_SHIFT_BLOCK, 5)
    lat.set_option(lq.LQCD_OPT_CHECK_EVERY, 7)
    assert lat.get_option(lq.LQCD_OPT_CHECK_EVERY) == 10          # rounded up to whole blocks
    lat.close()


@both_solvers
@pytest.mark.parametrize("L,mass,shifts", [
    ((4, 4, 4, 4), 0.05, [1e-3, 1e-2, 1e-1, 1.0]),
    ((4, 6, 8, 10), 0.02, [1e-2, 1e-3, 1e-1, 1.0, 0.5]),
    ((8, 8, 8, 8), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
])
def test_every_block_length_gives_the_same_solve(lq, L, mass, shifts, solver_path):
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, 1e-10)
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    b = cuda(b_soa)
    # the persistent solver handles blocks up to 16 (longer ones go to the launch path, whose sums run over another grid)
    blocks = [m for m in BLOCKS if m <= 16] if solver_path == "persistent" else BLOCKS
    runs = {m: solve(lq, lat, b, shifts, 1e-10, m, use_graph=(m != 3)) for m in blocks}
    x1, i1 = runs[1]
    for m, (x, info) in runs.items():
        assert info["status"] == 0
        assert info["iters"] == i1["iters"] and info["freeze_iter"] == i1["freeze_iter"], (m, info, i1)
        assert info["rel_res"] == i1["rel_res"]
        # (for m >= 2 the base system's x_0 is block-deferred like the shifted ones: equal up to rounding, below)
        for i in range(len(shifts)):
            assert rel_l2(x[i].cpu().numpy(), x1[i].cpu().numpy()) <= 1e-12, (m, i)
            assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= TOL_CG, (m, i)
    lat.close()


@both_solvers
@pytest.mark.parametrize("n_iter", [1, 2, 7, 8, 9, 15, 16, 17, 23, 40])
def test_stop_in_the_middle_of_a_block(lq, n_iter, solver_path):
    """MAX_ITER = n_iter with tol tiny: both sides do exactly n_iter iterations; for m = 8 and 16 the stop falls
    at every position of a block (including its first and last iteration); some shifts freeze on the way."""
    L, mass = (8, 8, 8, 8), 0.0075
    shifts = gen.shifts_geometric(1e-5, 1.0, 16)
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, 1e-30, max_iter=n_iter)
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    b = cuda(b_soa)
    for m in ((1, 5, 8, 16) if solver_path == "persistent" else (1, 5, 8, 16, 32)):     # the persistent kernel: m <= 16
        x, info = solve(lq, lat, b, shifts, 1e-30, m, max_iter=n_iter)
        assert info["status"] == lq.LQCD_ENOCONV and info["iters"] == n_iter == info_ref["iters"]
        for i in range(16):
            assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= 1e-11, (m, i)
    lat.close()


@both_solvers
def test_freeze_in_the_middle_of_a_block(lq, solver_path):
    """Loose tolerance: the large shifts freeze after a handful of iterations, i.e. inside the first blocks;
    their x_i must stop moving exactly there (the oracle's do)."""
    L, mass = (8, 8, 8, 8), 0.05
    shifts = [1e-3, 0.3, 1.0, 3.0, 10.0]
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, 1e-6)
    assert len(set(info_ref["freeze_iter"])) == len(shifts) and min(info_ref["freeze_iter"]) < 16
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    b = cuda(b_soa)
    x1, _ = solve(lq, lat, b, shifts, 1e-6, 1)
    for m in (4, 8, 16):
        x, info = solve(lq, lat, b, shifts, 1e-6, m)
        assert info["iters"] == info_ref["iters"] and info["freeze_iter"] == info_ref["freeze_iter"]
        for i in range(len(shifts)):
            # same iterations on all sides: against the per-iteration update (m = 1) only the rounding of the
            # regrouped sums differs; against the oracle the usual bar (two CG runs drift apart by more than
            # one rounding over ~100 iterations, whatever m)
            assert rel_l2(x[i].cpu().numpy(), x1[i].cpu().numpy()) <= 1e-12, (m, i)
            assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= TOL_CG, (m, i)
    lat.close()


@both_solvers
@pytest.mark.parametrize("m", [1, 4, 7, 16, 32])
def test_rational_sum_with_blocks(lq, m, solver_path):
    if solver_path == "persistent" and m > 16:
        pytest.skip("the persistent kernel handles blocks of up to 16 iterations (test_persistent_option_is_strict)")
    L, mass = (8, 8, 8, 8), 0.01
    shifts = [1e-4 * 10 ** (i / 2) for i in range(8)]
    a0, al = rational_coefficients(len(shifts))
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    y_ref, info_ref = oracle.rational_apply(L, U.numpy(), mass, b_aos, a0, al, shifts, 1e-10)
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    lat.set_option(lq.LQCD_OPT_SHIFT_BLOCK, m)
    b = cuda(b_soa)
    with torch.cuda.stream(torch.cuda.Stream()):
        y, info = lat.rational_apply(b, a0, al, shifts, 1e-10)
        x, info_x = lat.mshift_cg(b, shifts, 1e-10)
    torch.cuda.synchronize()
    assert info["iters"] == info_x["iters"] and info["freeze_iter"] == info_x["freeze_iter"]
    assert rel_l2(soa_gpu_to_aos(y), y_ref) <= TOL_CG
    y_sum = a0 * b + sum(al[i] * x[i] for i in range(len(shifts)))
    assert rel_l2(y.cpu().numpy(), y_sum.cpu().numpy()) <= 1e-11
    # fixed count, stop inside a block
    y_ref2, _ = oracle.rational_apply(L, U.numpy(), mass, b_aos, a0, al, shifts, 1e-30, max_iter=21)
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 21)
    with torch.cuda.stream(torch.cuda.Stream()):
        y2, info2 = lat.rational_apply(b, a0, al, shifts, 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    assert info2["iters"] == 21 and rel_l2(soa_gpu_to_aos(y2), y_ref2) <= 1e-11
    lat.close()


@both_solvers
def test_single_precision_with_blocks(lq, solver_path):
    L, mass, shifts = (8, 8, 8, 8), 0.05, [1e-3, 1e-2, 1e-1, 1.0]
    U, f = make_inputs(L)
    U32 = U.float().double()
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    b32 = torch.as_tensor(b_soa).float()
    b_aos32 = oracle.soa_to_aos(b32.double().numpy())
    x_ref, info_ref = oracle.mshift_cg(L, U32.numpy(), mass, b_aos32, shifts, 1e-30, max_iter=20)
    lat = lq.Lattice(L, mass=mass, precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(U.cuda())
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 20)
    res = {}
    blocks = (1, 8, 16) if solver_path == "persistent" else (1, 8, 16, 32)
    for m in blocks:
        lat.set_option(lq.LQCD_OPT_SHIFT_BLOCK, m)
        with torch.cuda.stream(torch.cuda.Stream()):
            x, info = lat.mshift_cg(b32.cuda(), shifts, 1e-30, raise_on_noconv=False)
        torch.cuda.synchronize()
        assert info["iters"] == 20
        res[m] = info
        for i in range(len(shifts)):
            # 20 iterations x (24 + few) eps32 per iteration, as in test_gpu_f32.py
            assert rel_l2(oracle.soa_to_aos(x[i].double().cpu().numpy()), x_ref[i]) <= 2e-5, (m, i)
    assert len({res[m]["rel_res"] for m in blocks}) == 1
    lat.close()


def test_persistent_option_is_strict(lq):
    """LQCD_OPT_PERSISTENT = 1 means the persistent kernel or an error, never a silent change of driver; -1 and 0 say
    through LQCD_STAT_SOLVER_PATH which driver ran."""
    L, mass, shifts = (8, 8, 8, 8), 0.05, [0.01, 0.1]
    U, f = make_inputs(L)
    b = cuda(oracle_parity_vector(L, f.numpy(), 0)[0])
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    with torch.cuda.stream(torch.cuda.Stream()):
        lat.set_option(lq.LQCD_OPT_PERSISTENT, 1)
        lat.set_option(lq.LQCD_OPT_SHIFT_BLOCK, 32)
        with pytest.raises(lq.LqcdError) as e:
            lat.mshift_cg(b, shifts, 1e-10)
        assert e.value.code == lq.LQCD_EINVAL and "SHIFT_BLOCK" in str(e.value)
        lat.set_option(lq.LQCD_OPT_SHIFT_BLOCK, 16)
        x2, info2 = lat.mshift_cg(b, shifts, 1e-10)
        assert info2["solver_path"] == 2
        lat.set_option(lq.LQCD_OPT_PERSISTENT, 0)
        x1, info1 = lat.mshift_cg(b, shifts, 1e-10)
        assert info1["solver_path"] == 1 and info1["graph_replays"] >= 1
        lat.set_option(lq.LQCD_OPT_USE_GRAPH, 0)
        x0, info0 = lat.mshift_cg(b, shifts, 1e-10)
        assert info0["solver_path"] == 0 and info0["graph_replays"] == 0
    torch.cuda.synchronize()
    assert info0["iters"] == info1["iters"] and abs(info2["iters"] - info1["iters"]) <= 1
    for i in range(len(shifts)):
        assert rel_l2(x0[i].cpu().numpy(), x1[i].cpu().numpy()) <= 1e-12
        assert rel_l2(x2[i].cpu().numpy(), x1[i].cpu().numpy()) <= 1e-10
    lat.close()
