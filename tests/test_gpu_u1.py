"""GPU parity for the general U(1) phase field u_mu(x) = exp(i theta_mu(x)):
lqcd_set_u1_phases + every operator / solver, against the oracle's *_u1 entry points on the same seeded inputs.

Tolerances: the U(1) factor adds one cos/sin (<= 2 ulp in CUDA's double sincos, correctly rounded to < 1 ulp in
glibc) and one complex multiply per hop to the 8x9 complex FMAs of the plain operator, so the forward error
stays at a few 1e-16 relative; the bound is the north_star's 1e-12 for one application.  Single precision:
bound from tests/test_gpu_f32.py's derivation (storage rounding 6e-8 per operand, 24-term sums) + sincosf
(<= 2 ulp) => 1e-6 relative L2.  CG: 1e-8 per shift as for the plain operator.
"""
import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle
from helpers import both_solvers, make_inputs, oracle_parity_vector, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu

TOL_D = 1e-12
TOL_D_F32 = 1e-6
TOL_CG = 1e-8


@pytest.fixture(scope="module")
def lq():
    import paper_1801_01473_b200 as lq
    lq.load_library()
    return lq


def cuda(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


LATTICES = [(4, 4, 4, 4), (4, 6, 8, 10), (2, 2, 2, 2), (6, 2, 4, 2), (10, 6, 4, 14), (16, 16, 16, 16)]


@pytest.mark.parametrize("L", LATTICES)
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("antiperiodic", [True, False])
def test_dslash_with_u1_phases(lq, L, recon, antiperiodic):
    U, f = make_inputs(L)
    th = gen.random_u1_phases(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    t_ref = oracle.doe(L, U.numpy(), b_aos, antiperiodic, theta=th.numpy())
    u_ref = oracle.deo(L, U.numpy(), t_ref, antiperiodic, theta=th.numpy())
    # the field must matter, otherwise this test pins nothing
    assert rel_l2(t_ref, oracle.doe(L, U.numpy(), b_aos, antiperiodic)) > 0.1

    lat = lq.Lattice(L, antiperiodic=antiperiodic, recon=recon)
    lat.set_u1_phases(th.cuda())                       # before the gauge field: the two are independent
    lat.set_gauge(U.cuda())
    b = cuda(b_soa)
    t = lat.doe(b)
    u = lat.deo(t)
    torch.cuda.synchronize()
    assert rel_l2(soa_gpu_to_aos(t), t_ref) <= TOL_D
    assert rel_l2(soa_gpu_to_aos(u), u_ref) <= TOL_D
    lat.set_option(lq.LQCD_OPT_MASS, 0.37)
    a = lat.mdagm(b, 0.11)
    a_ref = oracle.mdagm(L, U.numpy(), 0.37, 0.11, b_aos, antiperiodic, theta=th.numpy())
    assert rel_l2(soa_gpu_to_aos(a), a_ref) <= TOL_D
    # switching the field off restores the plain operator
    lat.set_u1_phases(None)
    t0 = lat.doe(b)
    assert rel_l2(soa_gpu_to_aos(t0), oracle.doe(L, U.numpy(), b_aos, antiperiodic)) <= TOL_D
    lat.close()


def test_u1_host_entry_point_and_large_angles(lq):
    """theta from host memory; angles far outside (-pi, pi) go through the same argument reduction."""
    L = (4, 6, 8, 10)
    U, f = make_inputs(L)
    th = gen.random_u1_phases(L) * 40.0                 # |theta| up to ~126
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L)
    lat.set_gauge(U.cuda())
    lat.set_u1_phases(th)                              # CPU tensor -> lqcd_set_u1_phases_host
    t = lat.doe(cuda(b_soa))
    assert rel_l2(soa_gpu_to_aos(t), oracle.doe(L, U.numpy(), b_aos, True, theta=th.numpy())) <= TOL_D
    lat.close()


def test_u1_pi_on_last_time_slice_equals_antiperiodic(lq):
    """PAPER.md:L159 "by which we handle antiperiodic boundary conditions": theta = pi on the t-links leaving
    t = Lt-1 with the periodic operator equals the built-in antiperiodic operator.  GPU against GPU, exact up to
    cos(pi) = -1, sin(pi) = 1.2e-16."""
    L = (4, 6, 4, 8)
    U, f = make_inputs(L)
    V = L[0] * L[1] * L[2] * L[3]
    th = torch.zeros((4, V), dtype=torch.float64)
    lex = torch.arange(V)
    t_of = lex // (L[0] * L[1] * L[2])
    th[3, t_of == L[3] - 1] = np.pi
    b_soa, _ = oracle_parity_vector(L, f.numpy(), 0)
    b = cuda(b_soa)
    lat_a = lq.Lattice(L, antiperiodic=True)
    lat_a.set_gauge(U.cuda())
    lat_p = lq.Lattice(L, antiperiodic=False)
    lat_p.set_gauge(U.cuda())
    lat_p.set_u1_phases(th.cuda())
    ta, tp = lat_a.doe(b), lat_p.doe(b)
    assert rel_l2(tp.cpu().numpy(), ta.cpu().numpy()) <= 1e-15
    lat_a.close()
    lat_p.close()


@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_f32_with_u1_phases(lq, recon):
    L = (4, 6, 8, 10)
    U, f = make_inputs(L)
    th = gen.random_u1_phases(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, recon=recon, precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(U.cuda())
    lat.set_u1_phases(th.cuda())
    b32 = cuda(b_soa).float()
    t = lat.doe(b32)
    t_ref = oracle.doe(L, U.numpy(), oracle.soa_to_aos(b32.double().cpu().numpy()), True, theta=th.numpy())
    assert rel_l2(soa_gpu_to_aos(t.double()), t_ref) <= TOL_D_F32
    # double entry points have no phases stored in this context: loud error, not a silent u = 1
    with pytest.raises(lq.LqcdError):
        lat.doe(cuda(b_soa))
    lat.close()


@pytest.mark.parametrize("use_graph", [True, False])
@both_solvers
def test_mshift_cg_with_u1_phases(lq, use_graph, solver_path):
    L, mass, tol = (8, 8, 8, 8), 0.05, 1e-10
    shifts = [1e-3, 1e-2, 1e-1, 1.0]
    U, f = make_inputs(L)
    th = gen.random_u1_phases(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, tol, theta=th.numpy())
    lat = lq.Lattice(L, mass=mass)
    lat.set_option(lq.LQCD_OPT_USE_GRAPH, 1 if use_graph else 0)
    lat.set_gauge(U.cuda())
    lat.set_u1_phases(th.cuda())
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg(cuda(b_soa), shifts, tol)
    torch.cuda.synchronize()
    assert info["status"] == 0
    assert abs(info["iters"] - info_ref["iters"]) <= 1, (info, info_ref)
    for i in range(len(shifts)):
        assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= TOL_CG
        # true residual of the GPU solution, computed by the oracle's operator
        r = b_aos - oracle.mdagm(L, U.numpy(), mass, shifts[i], soa_gpu_to_aos(x[i]), True, theta=th.numpy())
        assert np.linalg.norm(r) / np.linalg.norm(b_aos) <= 5 * tol
    # the graph is rebuilt when the field is switched off: same context, plain operator again
    lat.set_u1_phases(None)
    x_ref0, info_ref0 = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, tol)
    with torch.cuda.stream(torch.cuda.Stream()):
        x0, info0 = lat.mshift_cg(cuda(b_soa), shifts, tol)
    torch.cuda.synchronize()
    assert abs(info0["iters"] - info_ref0["iters"]) <= 1
    for i in range(len(shifts)):
        assert rel_l2(soa_gpu_to_aos(x0[i]), x_ref0[i]) <= TOL_CG
    lat.close()
