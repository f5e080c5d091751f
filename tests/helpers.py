"""Shared test plumbing: inputs from lqcd_inputs, conversions through the ORACLE's layout helpers.
Nothing here is used by the product."""
import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle


def rel_l2(a, b) -> float:
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / (nb if nb > 0 else 1.0))


def make_inputs(L, seed_links=gen.SEED_LINKS, seed_src=gen.SEED_SOURCE, device="cpu"):
    """links (4,V,3,3,2) and a whole-lattice Gaussian site field (V,3,2), as torch tensors."""
    U = gen.random_su3_links(L, seed_links, device=device)
    f = gen.gaussian_field(L, seed_src, device=device)
    return U, f


def oracle_parity_vector(L, site_field_np, parity):
    """Oracle-side route from a site field to the boundary (vec3_soa) layout, and the AoS parity field."""
    aos = oracle.restrict(L, parity, site_field_np)
    return oracle.aos_to_soa(aos), aos


def soa_gpu_to_aos(v) -> np.ndarray:
    """GPU parity vector (3,Vh,2) -> oracle AoS parity field (Vh,3,2), via the oracle's own helper."""
    return oracle.soa_to_aos(v.detach().cpu().numpy())


# run a test once on each driver of the CG iteration (conftest.solver_path)
both_solvers = pytest.mark.parametrize("solver_path", ["launches", "persistent"], indirect=True)
