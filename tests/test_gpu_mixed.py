"""NEXT-2, second half: float CG with double-precision reliable updates (lqcd_mshift_cg_mixed)
against the double-precision oracle.  The method is a different route to the same solutions, so what is compared is
what is unique: x_i = (A + sigma_i)^-1 b within the north_star bar (relative L2 <= 1e-8), and the TRUE residual of
every system, computed by the oracle's operator in double, <= tol (the solver's own stopping rule, with 0.1 % slack
for the different summation order of the two norms)."""
import numpy as np
import pytest
import torch

import oracle
import paper_1801_01473_b200 as lq
from helpers import make_inputs, oracle_parity_vector, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu
BOTH = lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32


def _true_residuals(L, U, mass, b_aos, shifts, xs):
    nb = np.linalg.norm(b_aos)
    return [float(np.linalg.norm(b_aos - oracle.mdagm(L, U, mass, s, x)) / nb) for s, x in zip(shifts, xs)]


@pytest.mark.parametrize("L,mass,shifts,recon", [
    ((8, 8, 8, 8), 0.05, [0.0], 18),
    ((8, 8, 8, 8), 0.05, [1e-3, 1e-2, 1e-1, 1.0], 18),
    ((4, 6, 8, 10), 0.02, [0.5, 0.0, 0.03], 12),
    ((8, 8, 8, 16), 0.01, [1e-4, 1e-2], 18),
])
@pytest.mark.parametrize("graph", [True, False])
def test_mixed_solver_matches_oracle(L, mass, shifts, recon, graph):
    tol = 1e-10
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, mass=mass, recon=recon, precisions=BOTH)
    lat.set_option(lq.LQCD_OPT_USE_GRAPH, 1.0 if graph else 0.0)
    lat.set_gauge(U.cuda())
    b = torch.as_tensor(b_soa).cuda()
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg_mixed(b, shifts, tol)
        xd, info_d = lat.mshift_cg(b, shifts, tol)
    torch.cuda.synchronize()
    x_ref, _ = oracle.mshift_cg(L, U.numpy(), mass, b_aos, shifts, tol)
    xs = [soa_gpu_to_aos(x[i]) for i in range(len(shifts))]
    for i in range(len(shifts)):
        assert rel_l2(xs[i], x_ref[i]) <= 1e-8, (i, rel_l2(xs[i], x_ref[i]))
    res = _true_residuals(L, U.numpy(), mass, b_aos, shifts, xs)
    assert max(res) <= tol * 1.001, res
    assert info["rel_res"] <= tol and abs(info["rel_res"] - max(res)) <= 1e-3 * tol
    assert info["reliable_updates"] >= len(shifts)          # every system ends on a true residual
    assert info["iters"] >= info_d["iters"] // 2            # it did iterate (float iterations, all phases)
    lat.close()


def test_mixed_solver_edge_cases():
    L = (4, 4, 4, 4)
    U, f = make_inputs(L)
    b_soa, _ = oracle_parity_vector(L, f.numpy(), 0)
    b = torch.as_tensor(b_soa).cuda()
    # needs both link copies
    lat = lq.Lattice(L, mass=0.1)
    lat.set_gauge(U.cuda())
    x = lat.new_vector(1)
    assert lq.lqcd_mshift_cg_mixed(lat.ctx, b.data_ptr(), [0.0], 1e-10, [x[0].data_ptr()]) == lq.LQCD_ENOGAUGE
    lat.close()
    lat = lq.Lattice(L, mass=0.1, precisions=BOTH)
    lat.set_gauge(U.cuda())
    with torch.cuda.stream(torch.cuda.Stream()):
        # zero source
        x, info = lat.mshift_cg_mixed(torch.zeros_like(b), [0.0, 0.1], 1e-10)
        assert float(x.abs().max()) == 0.0 and info["iters"] == 0
        # a tolerance single precision reaches alone still ends on a true residual
        x, info = lat.mshift_cg_mixed(b, [0.0, 0.1], 1e-4)
        assert info["rel_res"] <= 1e-4          # checked on the true residual even when no replacement was needed
        # iteration cap
        lat.set_option(lq.LQCD_OPT_MAX_ITER, 3)
        x, info = lat.mshift_cg_mixed(b, [0.0], 1e-12, raise_on_noconv=False)
        assert info["status"] == lq.LQCD_ENOCONV
    torch.cuda.synchronize()
    assert lq.lqcd_mshift_cg_mixed(lat.ctx, b.data_ptr(), [-1.0], 1e-10, [x[0].data_ptr()]) == lq.LQCD_EINVAL
    assert lq.lqcd_mshift_cg_mixed(lat.ctx, b.data_ptr(), [0.0], 1e-10, [b.data_ptr()]) == lq.LQCD_EINVAL
    lat.close()
