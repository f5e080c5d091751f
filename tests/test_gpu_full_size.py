"""Parity of the widened rows AT THE SIZE bench.py times them (48^4; mixed precision at 32^4),
each against the CPU oracle on the same seeded inputs -- the small-lattice tests of these rows live in
test_gpu_u1.py, test_gpu_f32.py, test_gpu_parity.py (rational sum), test_gpu_slab.py, test_gpu_mixed.py:

  * NEXT-4  general U(1) phases: the whole output field of D_oe then D_eo, 18- and 12-real links;
  * NEXT-2  single precision: 20 iterations of the multi-shift CG at a fixed count against the fp64 oracle fed the
            float-rounded links and source; tolerance as in test_gpu_f32.py;
  * NEXT-1  rational sum accumulated in the solve, 20 iterations at a fixed count;
  * NEXT-3  one rank of the slab path (ring closed on itself, over NCCL and over peer memory): the operator
            bit-identical to the whole-lattice kernel and within 1e-12 of the oracle, 20 CG iterations at a fixed
            count against the oracle;
  * NEXT-2  mixed precision, one system at 32^4 to tol 1e-10: the TRUE residual recomputed by the oracle's operator.

The inputs are drawn once on the GPU (module fixture); the same bytes go to the oracle."""
import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle
from helpers import make_inputs, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu

TOL_D = 1e-12


@pytest.fixture(scope="module")
def lq():
    import paper_1801_01473_b200 as lq
    lq.load_library()
    return lq


class Big:
    """config 4 inputs: links and source on the GPU, and their host copies for the oracle"""

    def __init__(self, lq):
        self.cfg = gen.CONFIGS["config4_48^4"]
        self.L = self.cfg["L"]
        self.U, f = make_inputs(self.L, device="cuda")
        lat = lq.Lattice(self.L)
        self.b = lat.pack(f, 0)
        lat.close()
        del f
        self.Uh = self.U.cpu().numpy()
        self.b_aos = soa_gpu_to_aos(self.b)


@pytest.fixture(scope="module")
def big(lq):
    b = Big(lq)
    yield b
    del b.U, b.Uh
    torch.cuda.empty_cache()


@pytest.mark.parametrize("recon", [18, 12])
def test_u1_dslash_48(lq, big, recon):
    L = big.L
    th = gen.random_u1_phases(L, device="cuda")
    thh = th.cpu().numpy()
    lat = lq.Lattice(L, recon=recon)
    lat.set_gauge(big.U)
    lat.set_u1_phases(th)
    t = lat.doe(big.b)
    u = lat.deo(t)
    torch.cuda.synchronize()
    t_ref = oracle.doe(L, big.Uh, big.b_aos, theta=thh)
    assert rel_l2(soa_gpu_to_aos(t), t_ref) <= TOL_D
    # the field matters at this size too (otherwise nothing is pinned)
    assert rel_l2(t_ref, oracle.doe(L, big.Uh, big.b_aos)) > 0.1
    u_ref = oracle.deo(L, big.Uh, t_ref, theta=thh)
    assert rel_l2(soa_gpu_to_aos(u), u_ref) <= TOL_D
    lat.close()


def test_rational_apply_fixed_count_48(lq, big):
    L, cfg, n_it = big.L, big.cfg, 40        # a whole shift block of 32, then a short one
    rng = np.random.default_rng(7)
    n = len(cfg["shifts"])
    alpha = list(rng.uniform(0.05, 1.5, n) * rng.choice([-1.0, 1.0], n))
    lat = lq.Lattice(L, mass=cfg["mass"])
    lat.set_gauge(big.U)
    lat.set_option(lq.LQCD_OPT_MAX_ITER, n_it)
    with torch.cuda.stream(torch.cuda.Stream()):
        y, info = lat.rational_apply(big.b, 0.37, alpha, cfg["shifts"], 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    y_ref, info_ref = oracle.rational_apply(L, big.Uh, cfg["mass"], big.b_aos, 0.37, alpha, cfg["shifts"], 1e-30,
                                            max_iter=n_it)
    assert info["iters"] == n_it == info_ref["iters"]
    assert rel_l2(soa_gpu_to_aos(y), y_ref) <= 1e-11
    lat.close()


@pytest.mark.parametrize("comm", ["nccl", "p2p"])
def test_slab_one_rank_48(lq, big, comm):
    """One rank of the slab path at the size bench.py times it, over either transport: the operator bit-identical to
    the whole-lattice kernel and within 1e-12 of the oracle; 40 iterations of the fused CG iteration on the slab (p
    faces formed by their owner, interior + border launches, reductions through the transport) at a fixed count
    against the oracle, <= 1e-11 as on the whole lattice."""
    L, cfg, n_it = big.L, big.cfg, 40        # a whole shift block of 32, then a short one
    whole = lq.Lattice(L)
    whole.set_gauge(big.U)
    slab = lq.Lattice(L, mass=cfg["mass"], slab=(0, 1), comm=comm)
    slab.set_gauge(big.U)
    slab.set_option(lq.LQCD_OPT_MAX_ITER, n_it)
    with torch.cuda.stream(torch.cuda.Stream()):
        t0, t1 = whole.doe(big.b), slab.doe(big.b)
        u0, u1 = whole.deo(t0), slab.deo(t1)
        x, info = slab.mshift_cg(big.b, cfg["shifts"], 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    assert torch.equal(t0, t1) and torch.equal(u0, u1)
    whole.close()
    t_ref = oracle.doe(L, big.Uh, big.b_aos)
    assert rel_l2(soa_gpu_to_aos(t1), t_ref) <= TOL_D
    assert rel_l2(soa_gpu_to_aos(u1), oracle.deo(L, big.Uh, t_ref)) <= TOL_D
    del t0, t1, u0, u1
    x_ref, info_ref = _oracle_cg20(big)
    assert info["iters"] == n_it == info_ref["iters"]
    assert max(rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) for i in range(len(cfg["shifts"]))) <= 1e-11
    slab.close()


_CG20 = {}


def _oracle_cg20(big):
    """40 iterations of the oracle's multi-shift CG on config 4 at a fixed count (computed once per module)"""
    if "r" not in _CG20:
        cfg = big.cfg
        _CG20["r"] = oracle.mshift_cg(big.L, big.Uh, cfg["mass"], big.b_aos, cfg["shifts"], 1e-30, max_iter=40)
    return _CG20["r"]


def test_f32_cg_fixed_count_48(lq, big):
    """The oracle (fp64) sees the float-rounded links and source, so every difference is float arithmetic in the
    kernels: 40 iterations x (24 + few) eps32 per iteration, bound 2e-5 as at 8^4 (test_gpu_f32.py)."""
    L, cfg, n_it = big.L, big.cfg, 40        # a whole shift block of 32, then a short one
    lat = lq.Lattice(L, mass=cfg["mass"], precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(big.U)
    b32 = big.b.float()
    lat.set_option(lq.LQCD_OPT_MAX_ITER, n_it)
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg(b32, cfg["shifts"], 1e-30, raise_on_noconv=False)
    torch.cuda.synchronize()
    U32h = big.Uh.astype(np.float32).astype(np.float64)
    b_aos32 = soa_gpu_to_aos(b32.double())
    x_ref, info_ref = oracle.mshift_cg(L, U32h, cfg["mass"], b_aos32, cfg["shifts"], 1e-30, max_iter=n_it)
    del U32h
    assert info["iters"] == n_it == info_ref["iters"] and x.dtype == torch.float32
    for i in range(len(cfg["shifts"])):
        assert rel_l2(soa_gpu_to_aos(x[i].double()), x_ref[i]) <= 2e-5, i
    assert abs(info["rel_res"] - info_ref["rel_res"]) <= 1e-4 * info_ref["rel_res"]
    lat.close()


def test_mixed_one_system_32(lq):
    """lqcd_mshift_cg_mixed, one system at 32^4 (m = 0.01, sigma = 1e-4, ~2200 float iterations with reliable
    updates): the true residual b - (A + sigma) x recomputed by the oracle's double operator is <= tol."""
    L, mass, sigma, tol = (32, 32, 32, 32), 0.01, 1e-4, 1e-10
    U, f = make_inputs(L, device="cuda")
    lat = lq.Lattice(L, mass=mass, precisions=lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32)
    lat.set_gauge(U)
    b = lat.pack(f, 0)
    with torch.cuda.stream(torch.cuda.Stream()):
        x, info = lat.mshift_cg_mixed(b, [sigma], tol)
    torch.cuda.synchronize()
    assert info["status"] == 0 and info["reliable_updates"] >= 2 and info["iters"] > 1000
    b_aos, x_aos = soa_gpu_to_aos(b), soa_gpu_to_aos(x[0])
    res = np.linalg.norm(b_aos - oracle.mdagm(L, U.cpu().numpy(), mass, sigma, x_aos)) / np.linalg.norm(b_aos)
    assert res <= tol * 1.001, res
    assert abs(info["rel_res"] - res) <= 1e-3 * tol
    lat.close()
