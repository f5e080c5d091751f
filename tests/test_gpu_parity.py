"""GPU parity: the CUDA library (through its C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; derivation in DESIGN.md "Tolerances"):
  * one Dslash application: relative L2 <= 1e-12 (expected ~1e-16: 8x9 complex FMAs per output);
  * CG solutions: relative L2 <= 1e-8 per shift, iteration count within +-1 of the oracle's.
"""
import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle
from helpers import both_solvers, make_inputs, oracle_parity_vector, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu

TOL_D = 1e-12
TOL_CG = 1e-8


@pytest.fixture(scope="module")
def lq():
    import paper_1801_01473_b200 as lq
    lq.load_library()
    return lq


def cuda(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


DSLASH_LATTICES = [(4, 4, 4, 4), (4, 6, 8, 10), (2, 2, 2, 2), (2, 4, 2, 6), (6, 2, 4, 2), (8, 8, 8, 6),
                   (10, 6, 4, 14), (16, 16, 16, 16), (24, 12, 8, 6)]


def test_pack_unpack_match_oracle_layout(lq):
    L = (4, 6, 8, 10)
    _, f = make_inputs(L)
    lat = lq.Lattice(L)
    fg = f.cuda()
    for p in (0, 1):
        soa, aos = oracle_parity_vector(L, f.numpy(), p)
        v = lat.pack(fg, p)
        assert np.array_equal(v.cpu().numpy(), soa)
        back = lat.unpack(v, p).cpu().numpy()
        assert np.array_equal(back, oracle.scatter(L, p, aos))
    lat.close()


@pytest.mark.parametrize("L", DSLASH_LATTICES)
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("antiperiodic", [True, False])
def test_dslash_doe_then_deo(lq, L, recon, antiperiodic):
    """BASELINE config 1 (4^4) and the asymmetric / ragged / L=2 cases: t = D_oe b, u = D_eo t."""
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    t_ref = oracle.doe(L, U.numpy(), b_aos, antiperiodic)
    u_ref = oracle.deo(L, U.numpy(), t_ref, antiperiodic)

    lat = lq.Lattice(L, antiperiodic=antiperiodic, recon=recon)
    lat.set_gauge(U.cuda())
    b = cuda(b_soa)
    t = lat.doe(b)
    u = lat.deo(t)
    torch.cuda.synchronize()
    assert rel_l2(soa_gpu_to_aos(t), t_ref) <= TOL_D
    assert rel_l2(soa_gpu_to_aos(u), u_ref) <= TOL_D
    # D_eo alone on an independent odd vector
    o_soa, o_aos = oracle_parity_vector(L, f.numpy(), 1)
    w = lat.deo(cuda(o_soa))
    assert rel_l2(soa_gpu_to_aos(w), oracle.deo(L, U.numpy(), o_aos, antiperiodic)) <= TOL_D
    # Eq. 2 operator in two launches
    lat.set_option(lq.LQCD_OPT_MASS, 0.37)
    a = lat.mdagm(b, 0.11)
    assert rel_l2(soa_gpu_to_aos(a), oracle.mdagm(L, U.numpy(), 0.37, 0.11, b_aos, antiperiodic)) <= TOL_D
    lat.close()


def test_dslash_host_entry_points(lq):
    L = (4, 6, 8, 10)
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L)
    lat.set_gauge(U)                                   # CPU tensor -> lqcd_set_gauge_host
    b = torch.as_tensor(b_soa).pin_memory()
    t = lat.doe(b)                                     # CPU tensors -> lqcd_doe_host
    assert t.device.type == "cpu"
    t_ref = oracle.doe(L, U.numpy(), b_aos)
    assert rel_l2(oracle.soa_to_aos(t.numpy()), t_ref) <= TOL_D
    u = lat.deo(t)
    assert rel_l2(oracle.soa_to_aos(u.numpy()), oracle.deo(L, U.numpy(), t_ref)) <= TOL_D
    lat.close()


def oracle_iteration_band(L, U, mass, b_aos, shifts, tol, n_ref, trials):
    """[lo, hi] spanned by the oracle's own iteration count under rounding-level perturbations: the other
    summation order of the scalar products, and the source moved by at most one ulp per component.
    (R9: beyond a few hundred iterations the CG residual history is sensitive to the last bit,
    so "the same count +-1" can only be asked relative to this band.)"""
    counts = [n_ref, oracle.mshift_cg(L, U, mass, b_aos, shifts, tol, sum_order=1)[1]["iters"]]
    rng = np.random.default_rng(1234)
    for _ in range(trials):
        bp = b_aos * (1.0 + rng.integers(-1, 2, size=b_aos.shape) * 2.0 ** -52)
        counts.append(oracle.mshift_cg(L, U, mass, bp, shifts, tol)[1]["iters"])
    return min(counts), max(counts)


_ORACLE_SOLVES = {}      # run_cg_both(keep_oracle=True): the oracle's solve of a long case, shared by its parametrizations


def run_cg_both(lq, L, mass, shifts, tol, recon=18, use_graph=True, stream=None, max_iter=None, host=False,
                check_every=None, band_trials=3, keep_oracle=False):
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    kw = {} if max_iter is None else dict(max_iter=max_iter)
    key = (tuple(L), mass, tuple(shifts), tol, max_iter, band_trials)
    if keep_oracle and key in _ORACLE_SOLVES:
        x_ref, info_ref = _ORACLE_SOLVES[key]
    else:
        x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, tol, **kw)
        if max_iter is None and info_ref["iters"] > 300:
            info_ref["band"] = oracle_iteration_band(L, U.numpy(), mass, b_aos, shifts, tol, info_ref["iters"], band_trials)
        else:
            info_ref["band"] = (info_ref["iters"], info_ref["iters"])
        if keep_oracle:
            _ORACLE_SOLVES[key] = (x_ref, info_ref)
    lat = lq.Lattice(L, mass=mass, recon=recon)
    lat.set_option(lq.LQCD_OPT_USE_GRAPH, 1 if use_graph else 0)
    if max_iter is not None:
        lat.set_option(lq.LQCD_OPT_MAX_ITER, max_iter)
    if check_every is not None:
        lat.set_option(lq.LQCD_OPT_CHECK_EVERY, check_every)

    def go():
        lat.set_gauge(U.cuda())
        b = torch.as_tensor(b_soa).pin_memory() if host else cuda(b_soa)
        return lat.mshift_cg(b, shifts, tol, raise_on_noconv=False)

    if stream is not None:
        with torch.cuda.stream(stream):
            x, info = go()
        stream.synchronize()
    else:
        x, info = go()
    torch.cuda.synchronize()
    launches = lat.launches
    lat.close()
    return x, info, x_ref, info_ref, launches


def check_cg(x, info, x_ref, info_ref, shifts):
    """iteration count within +-1 of the oracle's (of the oracle's rounding band for long solves), every
    solution within 1e-8, freeze schedule within the same slack."""
    lo, hi = info_ref.get("band", (info_ref["iters"], info_ref["iters"]))
    assert lo - 1 <= info["iters"] <= hi + 1, (info["iters"], info_ref["iters"], (lo, hi))
    slack = 1 + (hi - lo)
    for i in range(len(shifts)):
        err = rel_l2(soa_gpu_to_aos(x[i]), x_ref[i])
        assert err <= TOL_CG, (i, shifts[i], err)
        assert abs(info["freeze_iter"][i] - info_ref["freeze_iter"][i]) <= slack + 1, (i, info["freeze_iter"], info_ref["freeze_iter"])


@pytest.mark.parametrize("L,mass,shifts", [
    ((4, 4, 4, 4), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
    ((2, 2, 2, 2), 0.05, [0.3, 0.0, 2.0, 1e-3]),
    ((4, 6, 8, 10), 0.02, [1e-2, 1e-3, 1e-1, 1.0, 0.5]),
    ((8, 8, 8, 8), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
])
@pytest.mark.parametrize("mode", ["graph", "plain", "legacy_stream", "recon12", "host"])
@both_solvers
def test_mshift_cg_small(lq, L, mass, shifts, mode, solver_path):
    if solver_path == "persistent" and mode == "plain":
        pytest.skip("graph or plain launches: a property of the launch path only")
    s = None if mode == "legacy_stream" else torch.cuda.Stream()
    x, info, x_ref, info_ref, launches = run_cg_both(
        lq, L, mass, shifts, 1e-10, recon=12 if mode == "recon12" else 18, use_graph=(mode != "plain"),
        stream=s, host=(mode == "host"))
    assert info["status"] == 0 and info_ref["status"] == 0
    assert info["rel_res"] <= 1e-10
    assert info["base_shift"] == int(np.argmin(shifts))
    check_cg(x, info, x_ref, info_ref, shifts)
    if solver_path == "launches":
        assert launches >= 2 * info["iters"] + 2      # two launches per iteration (K1, K2 of cg.cuh) + init + sweeps
        assert info["solver_path"] == (1 if mode in ("graph", "recon12", "host") else 0)
    else:
        assert launches <= 8                          # links, pack, |b|^2 + ONE kernel for all iterations
        assert info["solver_path"] == 2


@both_solvers
@pytest.mark.parametrize("recon", [18, 12])
def test_mshift_cg_config2_16x4(lq, solver_path, recon):
    """BASELINE config 2: 16^4, m = 0.01, 8 shifts 1e-4*10^(i/2), tol 1e-10 -- full solve on both sides, with full
    and with two-row links (16^4 with two-row links is the case the library itself gives to the persistent kernel)."""
    cfg = gen.CONFIGS["config2_16^4"]
    x, info, x_ref, info_ref, _ = run_cg_both(lq, cfg["L"], cfg["mass"], cfg["shifts"], cfg["tol"], recon=recon,
                                              stream=torch.cuda.Stream(), band_trials=1, keep_oracle=True)
    assert info["status"] == 0 and info_ref["status"] == 0
    assert info["solver_path"] == (2 if solver_path == "persistent" else 1)      # the driver asked for is the one that ran
    print("config 2: GPU iterations", info["iters"], "oracle", info_ref["iters"], "oracle band", info_ref["band"],
          "freeze", info["freeze_iter"], info_ref["freeze_iter"])
    check_cg(x, info, x_ref, info_ref, cfg["shifts"])
    # true residual of every GPU solution, computed by the oracle operator (one application per shift)
    L = cfg["L"]
    U, f = make_inputs(L)
    _, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    bn = np.linalg.norm(b_aos)
    for i, sigma in enumerate(cfg["shifts"]):
        xi = soa_gpu_to_aos(x[i])
        res = b_aos - oracle.mdagm(L, U.numpy(), cfg["mass"], sigma, xi)
        assert np.linalg.norm(res) / bn <= 3 * cfg["tol"], (i, np.linalg.norm(res) / bn)


@both_solvers
def test_mshift_cg_fixed_iteration_count(lq, solver_path):
    """The protocol used at the large configs (R9): both sides run exactly n iterations."""
    L, mass = (8, 8, 8, 8), 0.0075
    shifts = gen.shifts_geometric(1e-5, 1.0, 16)
    x, info, x_ref, info_ref, _ = run_cg_both(lq, L, mass, shifts, 1e-30, max_iter=40, stream=torch.cuda.Stream())
    assert info["status"] == lq.LQCD_ENOCONV and info_ref["status"] == 1
    assert info["iters"] == 40 == info_ref["iters"]
    for i in range(16):
        assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= 1e-11
    assert abs(info["rel_res"] - info_ref["rel_res"]) <= 1e-9 * info_ref["rel_res"]


@pytest.mark.parametrize("L,n_it", [((20, 20, 20, 20), 40), ((24, 24, 24, 24), 20)])
@pytest.mark.parametrize("solver_path", ["launches"], indirect=True)
def test_mshift_cg_fixed_count_around_the_small_lattice_bound(lq, L, n_it, solver_path):
    """20^4 (625 blocks, more than one wave of them): the scalar steps ride in the sweeps (dslash_kernel FS = 1);
    24^4 (1296 blocks): the one-block kernels.  Both sides run exactly n iterations, across a block boundary of the
    deferred updates at 20^4 (m = 32 there, 40 iterations)."""
    mass = 0.01
    shifts = gen.shifts_geometric(1e-4, 1.0, 6)
    x, info, x_ref, info_ref, _ = run_cg_both(lq, L, mass, shifts, 1e-30, max_iter=n_it, stream=torch.cuda.Stream())
    assert info["iters"] == n_it == info_ref["iters"]
    for i in range(len(shifts)):
        assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= 1e-11
    assert abs(info["rel_res"] - info_ref["rel_res"]) <= 1e-9 * info_ref["rel_res"]


@pytest.mark.parametrize("check_every", [1, 3, 64])
@pytest.mark.parametrize("solver_path", ["launches"], indirect=True)      # the host polls only on the launch path
def test_mshift_cg_check_every_does_not_change_the_result(lq, check_every, solver_path):
    L, mass, shifts = (4, 4, 4, 4), 0.05, [1e-3, 1e-1]
    x, info, x_ref, info_ref, _ = run_cg_both(lq, L, mass, shifts, 1e-10, stream=torch.cuda.Stream(),
                                              check_every=check_every)
    check_cg(x, info, x_ref, info_ref, shifts)


@both_solvers
def test_mshift_cg_is_bit_reproducible(lq, solver_path):
    L, mass, shifts = (8, 8, 8, 8), 0.02, [1e-3, 1e-2, 1e-1]
    U, f = make_inputs(L)
    b_soa, _ = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    b = cuda(b_soa)
    with torch.cuda.stream(torch.cuda.Stream()):
        x1, i1 = lat.mshift_cg(b, shifts, 1e-10)
        x2, i2 = lat.mshift_cg(b, shifts, 1e-10)
    torch.cuda.synchronize()
    assert i1["iters"] == i2["iters"] and i1["freeze_iter"] == i2["freeze_iter"]
    assert torch.equal(x1, x2)
    lat.close()


@both_solvers
def test_edge_cases_and_errors(lq, solver_path):
    L = (4, 4, 4, 4)
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    # bad extents
    assert not lq.lqcd_create(3, 4, 4, 4) and "even" in lq.lqcd_last_error(None)
    assert not lq.lqcd_create(4, 4, 0, 4)
    lat = lq.Lattice(L, mass=0.1)
    b = cuda(b_soa)
    out = torch.empty_like(b)
    # no gauge yet
    assert lq.lqcd_doe(lat.ctx, out.data_ptr(), b.data_ptr()) == lq.LQCD_ENOGAUGE
    assert lq.lqcd_mshift_cg(lat.ctx, b.data_ptr(), [0.1], 1e-8, [out.data_ptr()]) == lq.LQCD_ENOGAUGE
    lat.set_gauge(U.cuda())
    # argument errors
    assert lq.lqcd_doe(lat.ctx, b.data_ptr(), b.data_ptr()) == lq.LQCD_EINVAL
    assert lq.lqcd_doe(lat.ctx, None, b.data_ptr()) == lq.LQCD_EINVAL
    assert lq.lqcd_mshift_cg(lat.ctx, b.data_ptr(), [-0.1], 1e-8, [out.data_ptr()]) == lq.LQCD_EINVAL
    assert lq.lqcd_mshift_cg(lat.ctx, b.data_ptr(), [0.1], 0.0, [out.data_ptr()]) == lq.LQCD_EINVAL
    assert lq.lqcd_mshift_cg(lat.ctx, b.data_ptr(), [0.1, 0.2], 1e-8, [out.data_ptr(), out.data_ptr()]) == lq.LQCD_EINVAL
    assert lq.lqcd_set_option(lat.ctx, lq.LQCD_OPT_RECON, 10) == lq.LQCD_EINVAL
    assert lq.lqcd_set_option(lat.ctx, 99, 1) == lq.LQCD_EINVAL
    # zero source -> zero solutions, zero iterations
    x, info = lat.mshift_cg(torch.zeros_like(b), [0.0, 1.0], 1e-10)
    assert info["iters"] == 0 and info["status"] == 0 and not x.any()
    # single shift, and the iteration cap
    x, info = lat.mshift_cg(b, [0.25], 1e-12)
    xr, ir = oracle.mshift_cg(L, U.numpy(), 0.1, b_aos, [0.25], 1e-12)
    assert abs(info["iters"] - ir["iters"]) <= 1 and rel_l2(soa_gpu_to_aos(x[0]), xr[0]) <= TOL_CG
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 3)
    x, info = lat.mshift_cg(b, [0.0], 1e-12, raise_on_noconv=False)
    assert info["status"] == lq.LQCD_ENOCONV and info["iters"] == 3
    xr, ir = oracle.mshift_cg(L, U.numpy(), 0.1, b_aos, [0.0], 1e-12, max_iter=3)
    assert rel_l2(soa_gpu_to_aos(x[0]), xr[0]) <= 1e-12
    # links that are not SU(3) are refused in 12-real mode, accepted in 18-real mode
    bad = U.clone()
    bad[2, 17, 2, 1, 0] += 1e-6
    lat.set_option(lq.LQCD_OPT_RECON, 12)
    assert lq.lqcd_set_gauge(lat.ctx, bad.cuda().data_ptr()) == lq.LQCD_ENOTSU3
    assert lq.lqcd_doe(lat.ctx, out.data_ptr(), b.data_ptr()) == lq.LQCD_ENOGAUGE      # nothing stored after a refusal
    lat.set_option(lq.LQCD_OPT_RECON, 18)
    lat.set_gauge(bad.cuda())
    t = lat.doe(b)
    assert rel_l2(soa_gpu_to_aos(t), oracle.doe(L, bad.numpy(), b_aos)) <= TOL_D
    lat.close()


@both_solvers
def test_caller_workspace(lq, solver_path):
    L, mass, shifts = (4, 6, 8, 10), 0.05, [1e-2, 1e-1, 1.0]
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, mass=mass)
    need = lq.lqcd_workspace_bytes(lat.ctx, len(shifts))
    assert need > 4 * lat.V * 144
    small = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    assert lq.lqcd_set_workspace(lat.ctx, small.data_ptr(), small.numel()) == 0
    assert lq.lqcd_set_gauge(lat.ctx, U.cuda().data_ptr()) == lq.LQCD_ENOMEM
    lat.close()
    lat = lq.Lattice(L, mass=mass)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    assert lq.lqcd_set_workspace(lat.ctx, ws.data_ptr(), ws.numel()) == 0
    lat.set_gauge(U.cuda())
    x, info = lat.mshift_cg(cuda(b_soa), shifts, 1e-10)
    xr, ir = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, 1e-10)
    ir["band"] = oracle_iteration_band(L, U.numpy(), mass, b_aos, shifts, 1e-10, ir["iters"], 3)
    check_cg(x, info, xr, ir, shifts)
    lat.close()
    # an arena of exactly the documented size also serves the host entry points and the mixed-precision solver
    # (their staging copies are allocated outside it); both link precisions are named BEFORE the query
    lat = lq.Lattice(L, mass=mass, precisions=lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32)
    need2 = lq.lqcd_workspace_bytes(lat.ctx, len(shifts))
    assert need2 > need
    ws = torch.empty(need2, dtype=torch.uint8, device="cuda")
    assert lq.lqcd_set_workspace(lat.ctx, ws.data_ptr(), ws.numel()) == 0
    lat.set_gauge(U.cuda())
    xh, ih = lat.mshift_cg(torch.as_tensor(b_soa).pin_memory(), shifts, 1e-10)
    assert torch.equal(xh, x.cpu()) and ih["iters"] == info["iters"]
    xm, im = lat.mshift_cg_mixed(cuda(b_soa), shifts, 1e-10)
    for i in range(len(shifts)):
        assert rel_l2(soa_gpu_to_aos(xm[i]), xr[i]) <= TOL_CG
    lat.close()


# ---- rational function of the Eq. 2 operator, accumulated during the solve ------
RATIONAL_CASES = [
    ((4, 4, 4, 4), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
    ((2, 2, 2, 2), 0.05, [0.3, 0.0, 2.0, 1e-3]),
    ((4, 6, 8, 10), 0.02, [1e-2, 1e-3, 1e-1, 1.0, 0.5]),
    ((8, 8, 8, 8), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
]


def rational_coefficients(n):
    """alpha_i of mixed sign and size (seeded; not a particular rational approximation)."""
    rng = np.random.default_rng(7)
    return 0.37, list(rng.uniform(0.05, 1.5, n) * rng.choice([-1.0, 1.0], n))


@pytest.mark.parametrize("L,mass,shifts", RATIONAL_CASES)
@pytest.mark.parametrize("mode", ["graph", "plain", "recon12", "host"])
@both_solvers
def test_rational_apply_small(lq, L, mass, shifts, mode, solver_path):
    if solver_path == "persistent" and mode == "plain":
        pytest.skip("graph or plain launches: a property of the launch path only")
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    a0, al = rational_coefficients(len(shifts))
    y_ref, info_ref = oracle.rational_apply(L, U.numpy(), mass, b_aos, a0, al, shifts, 1e-10)
    lat = lq.Lattice(L, mass=mass, recon=12 if mode == "recon12" else 18)
    lat.set_option(lq.LQCD_OPT_USE_GRAPH, 0 if mode == "plain" else 1)
    with torch.cuda.stream(torch.cuda.Stream()):
        lat.set_gauge(U.cuda())
        b = torch.as_tensor(b_soa).pin_memory() if mode == "host" else cuda(b_soa)
        y, info = lat.rational_apply(b, a0, al, shifts, 1e-10)
        # the same solve with the x_i stored: the fused sum must be the sum of those x_i
        x, info_x = lat.mshift_cg(cuda(b_soa), shifts, 1e-10)
    torch.cuda.synchronize()
    assert info["status"] == 0 and info["rel_res"] <= 1e-10
    assert info["iters"] == info_x["iters"] and info["freeze_iter"] == info_x["freeze_iter"]
    lo, hi = (info_ref["iters"],) * 2
    if info_ref["iters"] > 300:
        lo, hi = oracle_iteration_band(L, U.numpy(), mass, b_aos, shifts, 1e-10, info_ref["iters"], 2)
    assert lo - 1 <= info["iters"] <= hi + 1
    assert rel_l2(soa_gpu_to_aos(y), y_ref) <= TOL_CG
    y_sum = a0 * cuda(b_soa) + sum(al[i] * x[i] for i in range(len(shifts)))
    assert rel_l2(y.cpu().numpy(), y_sum.cpu().numpy()) <= 1e-11
    lat.close()


@both_solvers
def test_rational_apply_fixed_iteration_count_and_errors(lq, solver_path):
    L, mass = (8, 8, 8, 8), 0.0075
    shifts = gen.shifts_geometric(1e-5, 1.0, 16)
    a0, al = rational_coefficients(16)
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    y_ref, info_ref = oracle.rational_apply(L, U.numpy(), mass, b_aos, a0, al, shifts, 1e-30, max_iter=40)
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U.cuda())
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 40)
    b = cuda(b_soa)
    with torch.cuda.stream(torch.cuda.Stream()):
        y, info = lat.rational_apply(b, a0, al, shifts, 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    assert info["status"] == lq.LQCD_ENOCONV and info["iters"] == 40 == info_ref["iters"]
    assert rel_l2(soa_gpu_to_aos(y), y_ref) <= 1e-11
    # zero source, argument errors
    y0, info0 = lat.rational_apply(torch.zeros_like(b), a0, al, shifts, 1e-10)
    assert info0["iters"] == 0 and not y0.any()
    out = torch.empty_like(b)
    assert lq.lqcd_rational_apply(lat.ctx, b.data_ptr(), 1.0, [1.0], [-1.0], 1e-8, out.data_ptr()) == lq.LQCD_EINVAL
    assert lq.lqcd_rational_apply(lat.ctx, b.data_ptr(), 1.0, [float("nan")], [1.0], 1e-8, out.data_ptr()) == lq.LQCD_EINVAL
    assert lq.lqcd_rational_apply(lat.ctx, b.data_ptr(), 1.0, [1.0], [1.0], 1e-8, b.data_ptr()) == lq.LQCD_EINVAL
    assert lq.lqcd_rational_apply(lat.ctx, b.data_ptr(), 1.0, [1.0], [1.0], 1e-8, None) == lq.LQCD_EINVAL
    lat.close()


# ---- full BASELINE sizes, in the launch configuration bench.py times ---------------------------------
@pytest.mark.parametrize("L", [(32, 32, 32, 32), (48, 48, 48, 48)])
@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_full_size(lq, L, recon):
    """Configs 3 and 4: the whole output field of D_oe then D_eo against the oracle (inputs drawn on the GPU,
    the same bytes copied to the host for the oracle)."""
    U, f = make_inputs(L, device="cuda")
    lat = lq.Lattice(L, recon=recon)
    lat.set_gauge(U)
    b = lat.pack(f, 0)
    t = lat.doe(b)
    u = lat.deo(t)
    torch.cuda.synchronize()
    Uh = U.cpu().numpy()
    del U
    b_aos = soa_gpu_to_aos(b)
    t_ref = oracle.doe(L, Uh, b_aos)
    assert rel_l2(soa_gpu_to_aos(t), t_ref) <= TOL_D
    u_ref = oracle.deo(L, Uh, t_ref)
    assert rel_l2(soa_gpu_to_aos(u), u_ref) <= TOL_D
    lat.close()


def large_config_protocol(lq, name, n_it, residual_shifts):
    """DESIGN.md R9 protocol for the configs whose full oracle solve would take hours: (1) exactly n_it
    iterations on both sides, every x_i compared; (2) the GPU's own full solve, checked through
    oracle-computed true residuals of some shifts.  Inputs are drawn on the GPU; the same bytes go to the
    oracle."""
    cfg = gen.CONFIGS[name]
    L, mass, shifts = cfg["L"], cfg["mass"], cfg["shifts"]
    U, f = make_inputs(L, device="cuda")
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U)
    b = lat.pack(f, 0)
    Uh = U.cpu().numpy()
    del U, f
    b_aos = soa_gpu_to_aos(b)
    lat.set_option(lq.LQCD_OPT_MAX_ITER, n_it)
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg(b, shifts, 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    x_ref, info_ref = oracle.mshift_cg(L, Uh, mass, b_aos, shifts, 1e-30, max_iter=n_it)
    assert info["iters"] == n_it == info_ref["iters"]
    for i in range(len(shifts)):
        assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= 1e-11, i
    assert abs(info["rel_res"] - info_ref["rel_res"]) <= 1e-9 * info_ref["rel_res"]
    del x_ref
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 100000)
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg(b, shifts, cfg["tol"])
    torch.cuda.synchronize()
    assert info["status"] == 0 and info["rel_res"] <= cfg["tol"]
    fr = info["freeze_iter"]
    assert all(fr[i] >= fr[i + 1] for i in range(len(fr) - 1)) and fr[0] == info["iters"]
    print(name, "GPU full solve:", info["iters"], "iterations,", info["solve_ms"] / info["iters"], "ms/iter, freeze", fr)
    bn = np.linalg.norm(b_aos)
    for i in residual_shifts:
        res = b_aos - oracle.mdagm(L, Uh, mass, shifts[i], soa_gpu_to_aos(x[i]))
        assert np.linalg.norm(res) / bn <= 3 * cfg["tol"], (i, np.linalg.norm(res) / bn)
    lat.close()


def test_mshift_cg_config4_48x4(lq):
    """BASELINE config 4: 48^4, 16 shifts 1e-5..1, m = 0.0075, tol 1e-10."""
    # shift blocks are 32 iterations long here: 68 = the first sweep (iteration 32), a middle one (64: all residuals of
    # the block, p_i read and stored -- the sweep a real solve runs a hundred times) and a short closing one (68)
    large_config_protocol(lq, "config4_48^4", n_it=68, residual_shifts=(0, 7, 15))


def test_mshift_cg_config5_64x4(lq):
    """BASELINE config 5: 64^4 (16.8M sites, 9.7 GB of links), 16 shifts, m = 0.005, tol 1e-10."""
    large_config_protocol(lq, "config5_64^4", n_it=34, residual_shifts=(0, 15))         # one whole block of 32 + 2
