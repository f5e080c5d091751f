"""GPU parity of the single-precision path ("double (or float)", L282
single-precision MD) against the fp64 CPU oracle.

Both sides see the SAME inputs: the source is rounded to float once, the library rounds the (double, exactly
SU(3)) links to float when it stores them, and the oracle gets those floats widened back to double, so every
difference is float arithmetic in the kernels (with 12-real storage also the third row rebuilt in float from
the rounded rows against the rounded third row: a few eps32, inside the same bound).

Tolerances (eps32 = 2^-24):
  * one Dslash application: an output component is a sum of 8x3 complex products of O(1) numbers, worst-case
    forward error 24 eps32 = 1.4e-6 relative; bound 2e-6 (observed 1.3e-7);
  * CG solutions: each of the n updates x_i += a_i p_i rounds x_i once (eps32 relative), the n roundings add
    up to at most n eps32; both sides stop at the same tol, a stop a few iterations apart moves x_i by O(tol):
    bound n eps32 + 10 tol (observed 2e-6 at n = 1349, i.e. ~ sqrt(n) eps32);
  * iteration count: within max(3, 3 %) of the oracle's (observed <= 2.3 %, 3 of 132): the float residual
    recurrence follows the double one until it nears the float noise floor, where it converges a little slower.
"""
import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle
from helpers import both_solvers, make_inputs, oracle_parity_vector, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu

EPS32 = 2.0 ** -24
TOL_D32 = 2e-6


@pytest.fixture(scope="module")
def lq():
    import paper_1801_01473_b200 as lq
    lq.load_library()
    return lq


def cuda(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


class F32Inputs:
    """U: the double links handed to lqcd_set_gauge; U32 / f: links and site field rounded to float and widened
    back, the exact values the float kernels compute with, handed to the oracle."""

    def __init__(self, L, device="cpu"):
        self.U, f = make_inputs(L, device=device)
        self.U32 = self.U.float().double()
        self.f = f.float().double()


def f32_inputs(L, device="cpu"):
    i = F32Inputs(L, device)
    return i.U, i.U32, i.f


def aos64(v):
    return soa_gpu_to_aos(v.double())


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (4, 6, 8, 10), (2, 2, 2, 2), (6, 2, 4, 2), (10, 6, 4, 14), (16, 16, 16, 16)])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("antiperiodic", [True, False])
def test_dslash_f32(lq, L, recon, antiperiodic):
    U, U32, f = f32_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, mass=0.37, antiperiodic=antiperiodic, recon=recon, precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(U.cuda())
    b = cuda(b_soa).float()
    t = lat.doe(b)
    u = lat.deo(t)
    a = lat.mdagm(b, 0.11)
    torch.cuda.synchronize()
    assert t.dtype == torch.float32
    assert rel_l2(aos64(t), oracle.doe(L, U32.numpy(), b_aos, antiperiodic)) <= TOL_D32
    assert rel_l2(aos64(u), oracle.deo(L, U32.numpy(), aos64(t), antiperiodic)) <= TOL_D32
    assert rel_l2(aos64(a), oracle.mdagm(L, U32.numpy(), 0.37, 0.11, b_aos, antiperiodic)) <= 2 * TOL_D32
    # only the float links are stored: the double entry points must refuse, not fall back
    bd = cuda(b_soa)
    assert lq.lqcd_doe(lat.ctx, torch.empty_like(bd).data_ptr(), bd.data_ptr()) == lq.LQCD_ENOGAUGE
    lat.close()


def test_f32_needs_f32_links_and_pack_unpack(lq):
    L = (4, 6, 8, 10)
    U, U32, f = f32_inputs(L)
    lat = lq.Lattice(L)                         # default: double links only
    lat.set_gauge(U.cuda())
    b = torch.zeros((3, lat.Vh, 2), dtype=torch.float32, device="cuda")
    out = torch.empty_like(b)
    assert lq.lqcd_doe_f32(lat.ctx, out.data_ptr(), b.data_ptr()) == lq.LQCD_ENOGAUGE
    assert lq.lqcd_mshift_cg_f32(lat.ctx, b.data_ptr(), [0.1], 1e-5, [out.data_ptr()]) == lq.LQCD_ENOGAUGE
    assert lq.lqcd_set_option(lat.ctx, lq.LQCD_OPT_LINK_PRECISIONS, 4) == lq.LQCD_EINVAL
    fg = f.cuda().float()
    for p in (0, 1):
        soa, aos = oracle_parity_vector(L, f.numpy(), p)
        v = lat.pack(fg, p)
        assert v.dtype == torch.float32 and np.array_equal(v.double().cpu().numpy(), soa)
        assert np.array_equal(lat.unpack(v, p).double().cpu().numpy(), oracle.scatter(L, p, aos))
    lat.close()


def test_dslash_f32_host_entry_points(lq):
    L = (4, 6, 8, 10)
    U, U32, f = f32_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, precisions=lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32)
    lat.set_gauge(U)                                   # CPU tensor -> lqcd_set_gauge_host, both precisions
    b = torch.as_tensor(b_soa).float().pin_memory()
    t = lat.doe(b)                                     # CPU float tensor -> lqcd_doe_f32_host
    assert t.device.type == "cpu" and t.dtype == torch.float32
    t_ref = oracle.doe(L, U32.numpy(), b_aos)
    assert rel_l2(oracle.soa_to_aos(t.double().numpy()), t_ref) <= TOL_D32
    td = lat.doe(torch.as_tensor(b_soa).pin_memory())  # the double copy serves the double entry points
    assert rel_l2(oracle.soa_to_aos(td.numpy()), oracle.doe(L, U.numpy(), b_aos)) <= 1e-12
    lat.close()


CG_CASES = [
    ((4, 4, 4, 4), 0.05, [1e-2, 1e-1, 1.0], 1e-5),
    ((2, 2, 2, 2), 0.05, [0.3, 0.0, 2.0, 1e-3], 1e-5),
    ((4, 6, 8, 10), 0.02, [1e-2, 1e-3, 1e-1, 1.0, 0.5], 1e-5),
    ((8, 8, 8, 8), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)], 1e-5),
    ((16, 16, 16, 16), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)], 1e-4),     # BASELINE config 2 inputs
]


def check_cg_f32(L, U, mass, b_aos, shifts, tol, x, info, x_ref, info_ref):
    n, n_ref = info["iters"], info_ref["iters"]
    dim = 3 * int(np.prod(L)) // 2
    if n_ref < dim:
        assert abs(n - n_ref) <= max(3, 0.03 * n_ref), (n, n_ref)
    else:
        # 2^4: the oracle needs more iterations than the matrix has rows (24), i.e. it is already past the
        # point where exact CG would have terminated and rounding alone decides the count; float takes longer
        assert n_ref <= n <= 2 * n_ref, (n, n_ref)
    bn = np.linalg.norm(b_aos)
    for i, sigma in enumerate(shifts):
        xi = aos64(x[i])
        err = rel_l2(xi, x_ref[i])
        assert err <= n * EPS32 + 10 * tol, (i, sigma, err)
        # true residual (oracle operator, double): stopping tolerance plus the drift of the float recurrence,
        # n roundings of size eps32 |A+sigma| |x_i| adding up like sqrt(n) <= 64
        res = np.linalg.norm(b_aos - oracle.mdagm(L, U, mass, sigma, xi)) / bn
        drift = 64 * EPS32 * (7.0 + sigma) * np.linalg.norm(xi) / bn
        assert res <= 3 * tol + drift, (i, sigma, res, drift)


@pytest.mark.parametrize("L,mass,shifts,tol", CG_CASES)
@pytest.mark.parametrize("mode", ["graph", "plain", "recon12", "host"])
@both_solvers
def test_mshift_cg_f32(lq, L, mass, shifts, tol, mode, solver_path):
    if solver_path == "persistent" and mode == "plain":
        pytest.skip("graph or plain launches: a property of the launch path only")
    if mode != "graph" and L[0] == 16:
        pytest.skip("the 16^4 case runs once")
    U, U32, f = f32_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    x_ref, info_ref = oracle.mshift_cg(L, U32.numpy(), mass, b_aos, shifts, tol)
    lat = lq.Lattice(L, mass=mass, recon=12 if mode == "recon12" else 18, precisions=lq.LQCD_PREC_F32)
    lat.set_option(lq.LQCD_OPT_USE_GRAPH, 0 if mode == "plain" else 1)
    with torch.cuda.stream(torch.cuda.Stream()):
        lat.set_gauge(U.cuda())
        b = torch.as_tensor(b_soa).float()
        b = b.pin_memory() if mode == "host" else b.cuda()
        x, info = lat.mshift_cg(b, shifts, tol)
    torch.cuda.synchronize()
    assert info["status"] == 0 and x.dtype == torch.float32
    assert info["base_shift"] == int(np.argmin(shifts))
    check_cg_f32(L, U32.numpy(), mass, b_aos, shifts, tol, x, info, x_ref, info_ref)
    lat.close()


@both_solvers
def test_mshift_cg_f32_fixed_iteration_count_and_rational(lq, solver_path):
    """Exactly 30 iterations on both sides (no stopping decision involved): x_i within 30 eps32-ish of the
    oracle; the fused rational sum equals the sum of the stored x_i."""
    L, mass = (8, 8, 8, 8), 0.0075
    shifts = gen.shifts_geometric(1e-5, 1.0, 16)
    U, U32, f = f32_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    x_ref, info_ref = oracle.mshift_cg(L, U32.numpy(), mass, b_aos, shifts, 1e-30, max_iter=30)
    lat = lq.Lattice(L, mass=mass, precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(U.cuda())
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 30)
    b = cuda(b_soa).float()
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg(b, shifts, 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    assert info["status"] == lq.LQCD_ENOCONV and info["iters"] == 30 == info_ref["iters"]
    for i in range(16):
        assert rel_l2(aos64(x[i]), x_ref[i]) <= 2e-5, i          # 30 iterations x (24 + few) eps32 per iteration
    assert abs(info["rel_res"] - info_ref["rel_res"]) <= 1e-4 * info_ref["rel_res"]
    rng = np.random.default_rng(7)
    al = list(rng.uniform(0.05, 1.5, 16) * rng.choice([-1.0, 1.0], 16))
    y_ref, _ = oracle.rational_apply(L, U32.numpy(), mass, b_aos, 0.37, al, shifts, 1e-30, max_iter=30)
    with torch.cuda.stream(torch.cuda.Stream()):
        y, info_y = lat.rational_apply(b, 0.37, al, shifts, 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    assert y.dtype == torch.float32 and info_y["iters"] == 30
    assert rel_l2(aos64(y), y_ref) <= 2e-5
    lat.close()


@pytest.mark.parametrize("L", [(32, 32, 32, 32), (48, 48, 48, 48)])
@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_f32_full_size(lq, L, recon):
    """BASELINE configs 3 and 4 in single precision, whole output field against the oracle."""
    U, U32, f = f32_inputs(L, device="cuda")
    lat = lq.Lattice(L, recon=recon, precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(U)
    b = lat.pack(f.float(), 0)
    t = lat.doe(b)
    u = lat.deo(t)
    torch.cuda.synchronize()
    Uh = U32.cpu().numpy()
    del U, U32
    t_ref = oracle.doe(L, Uh, aos64(b))
    assert rel_l2(aos64(t), t_ref) <= TOL_D32
    assert rel_l2(aos64(u), oracle.deo(L, Uh, aos64(t))) <= TOL_D32
    lat.close()
