"""ctypes front end of the CPU oracle (oracle/lqcd_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and the cpu_baseline /
``--impl reference`` legs of bench.py.  The product (paper_1801_01473_b200) never imports this package
and this package never imports the product.

All fields are numpy float64 arrays holding (re, im) pairs:

* gauge field   (4, V, 3, 3, 2)   canonical layout, ``U[mu, lex]`` = link leaving ``lex`` along +mu
* parity field  (Vh, 3, 2)        array-of-structs over the sites of one parity, index ``lex >> 1``
* boundary      (3, Vh, 2)        the library's ``vec3_soa`` layout
"""
from __future__ import annotations

import ctypes
from typing import Sequence

import numpy as np

from .build import build as _build

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build())
        L = _lib
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_num_threads.argtypes = [ctypes.c_int]
        L.oracle_dslash.argtypes = [_ip, _dp, _dp, _dp, ctypes.c_int, ctypes.c_int]
        L.oracle_mdagm.argtypes = [_ip, _dp, ctypes.c_double, ctypes.c_double, _dp, _dp, ctypes.c_int]
        L.oracle_reconstruct_third_row.argtypes = [ctypes.c_int64, _dp]
        L.oracle_soa_to_aos.argtypes = [ctypes.c_int64, _dp, _dp]
        L.oracle_aos_to_soa.argtypes = [ctypes.c_int64, _dp, _dp]
        L.oracle_restrict.argtypes = [_ip, ctypes.c_int, _dp, _dp]
        L.oracle_scatter.argtypes = [_ip, ctypes.c_int, _dp, _dp]
        L.oracle_mshift_cg.argtypes = [_ip, _dp, ctypes.c_double, ctypes.c_int, _dp, _dp, ctypes.c_int,
                                       ctypes.c_double, ctypes.c_int, ctypes.c_int, _dp, _ip, _ip, _dp]
        L.oracle_mshift_cg.restype = ctypes.c_int
        L.oracle_dslash_u1.argtypes = [_ip, _dp, _dp, _dp, _dp, ctypes.c_int, ctypes.c_int]
        L.oracle_mdagm_u1.argtypes = [_ip, _dp, _dp, ctypes.c_double, ctypes.c_double, _dp, _dp, ctypes.c_int]
        L.oracle_mshift_cg_u1.argtypes = [_ip, _dp, _dp, ctypes.c_double, ctypes.c_int, _dp, _dp, ctypes.c_int,
                                          ctypes.c_double, ctypes.c_int, ctypes.c_int, _dp, _ip, _ip, _dp]
        L.oracle_mshift_cg_u1.restype = ctypes.c_int
        L.oracle_rational_apply.argtypes = [_ip, _dp, ctypes.c_double, ctypes.c_int, _dp, ctypes.c_double, _dp, _dp,
                                            ctypes.c_int, ctypes.c_double, ctypes.c_int, _dp, _ip, _dp]
        L.oracle_rational_apply.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_dp)


def _L(L: Sequence[int]):
    return (ctypes.c_int * 4)(*[int(v) for v in L])


def _vh(L):
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3]) // 2


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return lib().oracle_num_threads()


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def _theta(L, theta):
    """theta: None, or the U(1) phase field (4, V) in radians, u_mu(x) = exp(i theta_mu(x))."""
    if theta is None:
        return None
    theta = _c(theta)
    assert theta.shape == (4, 2 * _vh(L))
    return theta


def dslash(L, U, f_in, out_parity: int, antiperiodic: bool = True, theta=None) -> np.ndarray:
    """Parity field on `out_parity` = D applied to the parity field `f_in` on the other parity."""
    U, f_in, theta = _c(U), _c(f_in), _theta(L, theta)
    out = np.empty((_vh(L), 3, 2), dtype=np.float64)
    if theta is None:
        lib().oracle_dslash(_L(L), _p(U), _p(f_in), _p(out), int(out_parity), int(antiperiodic))
    else:
        lib().oracle_dslash_u1(_L(L), _p(U), _p(theta), _p(f_in), _p(out), int(out_parity), int(antiperiodic))
    return out


def doe(L, U, f_even, antiperiodic: bool = True, theta=None) -> np.ndarray:
    """D_oe: even -> odd."""
    return dslash(L, U, f_even, 1, antiperiodic, theta)


def deo(L, U, f_odd, antiperiodic: bool = True, theta=None) -> np.ndarray:
    """D_eo: odd -> even."""
    return dslash(L, U, f_odd, 0, antiperiodic, theta)


def mdagm(L, U, mass: float, sigma: float, f_even, antiperiodic: bool = True, theta=None) -> np.ndarray:
    """(m^2 + sigma) f - D_eo D_oe f   (Eq. 2)."""
    U, f_even, theta = _c(U), _c(f_even), _theta(L, theta)
    out = np.empty_like(f_even)
    if theta is None:
        lib().oracle_mdagm(_L(L), _p(U), float(mass), float(sigma), _p(f_even), _p(out), int(antiperiodic))
    else:
        lib().oracle_mdagm_u1(_L(L), _p(U), _p(theta), float(mass), float(sigma), _p(f_even), _p(out),
                              int(antiperiodic))
    return out


def reconstruct_third_row(U) -> np.ndarray:
    """Copy of U with every third row replaced by conj(r0 x r1)."""
    out = _c(U).copy()
    lib().oracle_reconstruct_third_row(out.size // 18, _p(out))
    return out


def soa_to_aos(v_soa) -> np.ndarray:
    v_soa = _c(v_soa)
    vh = v_soa.shape[1]
    out = np.empty((vh, 3, 2), dtype=np.float64)
    lib().oracle_soa_to_aos(vh, _p(v_soa), _p(out))
    return out


def aos_to_soa(f) -> np.ndarray:
    f = _c(f)
    vh = f.shape[0]
    out = np.empty((3, vh, 2), dtype=np.float64)
    lib().oracle_aos_to_soa(vh, _p(f), _p(out))
    return out


def restrict(L, parity: int, full) -> np.ndarray:
    """Whole-lattice field (V,3,2) -> parity field (Vh,3,2)."""
    full = _c(full)
    out = np.empty((_vh(L), 3, 2), dtype=np.float64)
    lib().oracle_restrict(_L(L), int(parity), _p(full), _p(out))
    return out


def scatter(L, parity: int, f, full=None) -> np.ndarray:
    """Parity field -> whole-lattice field (other parity zero unless `full` is given)."""
    f = _c(f)
    if full is None:
        full = np.zeros((2 * _vh(L), 3, 2), dtype=np.float64)
    lib().oracle_scatter(_L(L), int(parity), _p(f), _p(full))
    return full


def mshift_cg(L, U, mass: float, b_even, shifts, tol: float, max_iter: int = 100000,
              antiperiodic: bool = True, sum_order: int = 0, theta=None):
    """Multi-shift CG for (m^2 - D_eo D_oe + sigma_i) x_i = b.

    sum_order 0 (default) adds the per-slice partials of each scalar product in increasing t, 1 in
    decreasing t: the same algorithm under a rounding-level perturbation (R9).
    Returns (x, info): x is (nshift, Vh, 3, 2); info = dict(status, iters, freeze_iter, rel_res)."""
    U, b_even = _c(U), _c(b_even)
    sh = _c(np.asarray(shifts, dtype=np.float64))
    n = sh.shape[0]
    x = np.empty((n,) + b_even.shape, dtype=np.float64)
    iters = ctypes.c_int(0)
    freeze = (ctypes.c_int * n)()
    rel = ctypes.c_double(0.0)
    theta = _theta(L, theta)
    if theta is None:
        status = lib().oracle_mshift_cg(_L(L), _p(U), float(mass), int(antiperiodic), _p(b_even), _p(sh), n,
                                        float(tol), int(max_iter), int(sum_order), _p(x), ctypes.byref(iters),
                                        freeze, ctypes.byref(rel))
    else:
        status = lib().oracle_mshift_cg_u1(_L(L), _p(U), _p(theta), float(mass), int(antiperiodic), _p(b_even),
                                           _p(sh), n, float(tol), int(max_iter), int(sum_order), _p(x),
                                           ctypes.byref(iters), freeze, ctypes.byref(rel))
    return x, dict(status=status, iters=iters.value, freeze_iter=list(freeze), rel_res=rel.value)


def rational_apply(L, U, mass: float, b_even, alpha0: float, alpha, shifts, tol: float, max_iter: int = 100000,
                   antiperiodic: bool = True):
    """y = alpha0 b + sum_i alpha_i (m^2 - D_eo D_oe + sigma_i)^-1 b: the partial-fraction form of the RHMC's
    rational function of the Eq. 2 operator.  Returns (y, info)."""
    U, b_even = _c(U), _c(b_even)
    sh = _c(np.asarray(shifts, dtype=np.float64))
    al = _c(np.asarray(alpha, dtype=np.float64))
    assert sh.shape == al.shape and sh.ndim == 1
    y = np.empty_like(b_even)
    iters = ctypes.c_int(0)
    rel = ctypes.c_double(0.0)
    status = lib().oracle_rational_apply(_L(L), _p(U), float(mass), int(antiperiodic), _p(b_even), float(alpha0),
                                         _p(al), _p(sh), sh.shape[0], float(tol), int(max_iter), _p(y),
                                         ctypes.byref(iters), ctypes.byref(rel))
    return y, dict(status=status, iters=iters.value, rel_res=rel.value)
