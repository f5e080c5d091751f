"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

Each test is chosen so that a plausible mistake in oracle/lqcd_oracle.cpp fails it:

* P2 anti-hermiticity  D_oe^dagger = -D_eo: hop signs, backward-link index, dagger,
  boundary sign on both hops;
* P3 gauge covariance: links sit on the right sites / directions, U vs U^T, U vs U^dagger;
* P4 free-field closed form  D_eo D_oe e^{ipx} = -sum_mu sin^2(p_mu) e^{ipx}: the factor 1/2, the eta
  convention, the periodic wrap, and (with p_t = 2 pi (k_t + 1/2)/L_t) the antiperiodic boundary;
* P5 dense inversion with numpy.linalg for every shift: the whole multi-shift CG (recurrences,
  freezing, stopping rule), Eq. 2 of the paper;
* P1 third-row reconstruction r2 = conj(r0 x r1) against numpy.cross on unitary
  matrices that do not come from our generator;
* a second, link-centric dense assembly of D in numpy (different formulation, no shared code).
"""
import itertools

import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle


def c(a):
    """(…,2) float64 -> complex128 view."""
    a = np.ascontiguousarray(a)
    return a.view(np.complex128)[..., 0]


def r(a):
    """complex128 -> (…,2) float64."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64).reshape(a.shape + (2,))


def links(L, seed=gen.SEED_LINKS):
    return gen.random_su3_links(L, seed).numpy()


def coords(L):
    """x,y,z,t coordinate arrays in lex order, each shape (V,)."""
    Lx, Ly, Lz, Lt = L
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return x.ravel(), y.ravel(), z.ravel(), t.ravel()


def parity_mask(L, p):
    x, y, z, t = coords(L)
    return ((x + y + z + t) & 1) == p


def random_parity_field(L, seed):
    rng = np.random.default_rng(seed)
    vh = int(np.prod(L)) // 2
    return rng.standard_normal((vh, 3, 2))


def vdot(u, v):
    return np.vdot(c(u).ravel(), c(v).ravel())


LATTICES = [(2, 2, 2, 2), (4, 4, 2, 4), (4, 2, 4, 6), (2, 4, 6, 2), (4, 6, 4, 4)]


# ---------------------------------------------------------------------------------------------------
# layout helpers
# ---------------------------------------------------------------------------------------------------
def test_layout_helpers_match_their_definition():
    L = (4, 2, 6, 2)
    V = int(np.prod(L))
    full = np.random.default_rng(1).standard_normal((V, 3, 2))
    for p in (0, 1):
        m = parity_mask(L, p)
        f = oracle.restrict(L, p, full)
        # sites of one parity in increasing lex order are exactly index lex>>1 = 0,1,2,...
        lex = np.nonzero(m)[0]
        assert np.array_equal(lex >> 1, np.arange(V // 2))
        assert np.array_equal(f, full[m])
        back = oracle.scatter(L, p, f)
        assert np.array_equal(back[m], full[m]) and not back[~m].any()
        soa = oracle.aos_to_soa(f)
        assert soa.shape == (3, V // 2, 2)
        assert np.array_equal(soa, np.transpose(f, (1, 0, 2)))
        assert np.array_equal(oracle.soa_to_aos(soa), f)


# ---------------------------------------------------------------------------------------------------
# P1  link compression
# ---------------------------------------------------------------------------------------------------
def test_third_row_reconstruction_on_foreign_su3():
    rng = np.random.default_rng(7)
    n = 200
    a = rng.standard_normal((n, 3, 3)) + 1j * rng.standard_normal((n, 3, 3))
    q, _ = np.linalg.qr(a)
    q = q / np.linalg.det(q)[:, None, None] ** (1.0 / 3.0)          # det = 1, still unitary
    assert np.abs(np.linalg.det(q) - 1).max() < 1e-13
    rec = c(oracle.reconstruct_third_row(r(q)))
    assert np.array_equal(rec[:, :2], q[:, :2])
    assert np.abs(rec[:, 2] - np.conj(np.cross(q[:, 0], q[:, 1]))).max() < 1e-15
    assert np.abs(rec - q).max() < 1e-13                              # it *is* the third row


def test_third_row_reconstruction_on_generated_links():
    U = links((4, 4, 2, 2))
    assert np.abs(oracle.reconstruct_third_row(U) - U).max() < 1e-15


# ---------------------------------------------------------------------------------------------------
# P2  anti-hermiticity
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", LATTICES)
@pytest.mark.parametrize("antiperiodic", [True, False])
def test_antihermiticity(L, antiperiodic):
    U = links(L)
    chi = random_parity_field(L, 11)      # even
    psi = random_parity_field(L, 12)      # odd
    lhs = vdot(chi, oracle.deo(L, U, psi, antiperiodic))
    rhs = vdot(psi, oracle.doe(L, U, chi, antiperiodic))
    scale = np.sqrt(vdot(chi, chi).real * vdot(psi, psi).real)
    assert abs(lhs + np.conj(rhs)) < 1e-14 * scale
    assert abs(lhs) > 1e-3 * scale        # not trivially zero


# ---------------------------------------------------------------------------------------------------
# P3  gauge covariance
# ---------------------------------------------------------------------------------------------------
def gauge_transform(L, U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger, with x+mu by numpy.roll on the coordinate grid."""
    Lx, Ly, Lz, Lt = L
    Uc, gc = c(U), c(g)
    out = np.empty_like(Uc)
    grid = gc.reshape(Lt, Lz, Ly, Lx, 3, 3)
    for mu in range(4):
        g_fwd = np.roll(grid, -1, axis=3 - mu).reshape(-1, 3, 3)
        out[mu] = gc @ Uc[mu] @ np.conj(np.transpose(g_fwd, (0, 2, 1)))
    return r(out)


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 2, 4, 6), (4, 6, 4, 4)])
def test_gauge_covariance(L):
    U = links(L)
    g = gen.random_gauge_transform(L, seed=99).numpy()
    Ug = gauge_transform(L, U, g)
    assert np.abs(c(Ug) @ np.conj(np.transpose(c(Ug), (0, 1, 3, 2))) - np.eye(3)).max() < 1e-14
    for p_in in (0, 1):
        psi = random_parity_field(L, 20 + p_in)
        g_in = c(g)[parity_mask(L, p_in)]
        g_out = c(g)[parity_mask(L, 1 - p_in)]
        psi_g = r(np.einsum("nab,nb->na", g_in, c(psi)))
        lhs = c(oracle.dslash(L, Ug, psi_g, 1 - p_in))
        rhs = np.einsum("nab,nb->na", g_out, c(oracle.dslash(L, U, psi, 1 - p_in)))
        assert np.abs(lhs - rhs).max() < 1e-13
        assert np.abs(rhs).max() > 0.1


# ---------------------------------------------------------------------------------------------------
# P4  free-field closed form
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,k", [((4, 6, 4, 4), (1, 1, 1, 1)), ((4, 6, 4, 4), (1, 2, 0, 3)),
                                 ((8, 4, 6, 4), (3, 1, 2, 1)), ((2, 2, 2, 2), (0, 1, 0, 1)),
                                 ((6, 4, 2, 8), (1, 0, 1, 5))])
@pytest.mark.parametrize("antiperiodic", [False, True])
def test_free_field_plane_wave(L, k, antiperiodic):
    U = gen.unit_links(L).numpy()
    x, y, z, t = coords(L)
    p = [2 * np.pi * k[i] / L[i] for i in range(3)]
    p.append(2 * np.pi * (k[3] + (0.5 if antiperiodic else 0.0)) / L[3])
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    colour = np.array([0.3 - 0.2j, -1.1 + 0.5j, 0.7 + 0.9j])
    psi_e = r((phase[:, None] * colour[None, :])[parity_mask(L, 0)])
    out = c(oracle.deo(L, U, oracle.doe(L, U, psi_e, antiperiodic), antiperiodic))
    lam = -sum(np.sin(pm) ** 2 for pm in p)
    assert np.abs(out - lam * c(psi_e)).max() < 2e-14
    # and Eq. 2's operator: (m^2 + sigma - lam) psi
    m, sigma = 0.37, 0.11
    out2 = c(oracle.mdagm(L, U, m, sigma, psi_e, antiperiodic))
    assert np.abs(out2 - (m * m + sigma - lam) * c(psi_e)).max() < 2e-14


def test_free_field_eigenvalue_is_not_degenerate_case():
    # the plane waves used above really have sum sin^2 != 0 and different per direction
    L, k = (4, 6, 4, 4), (1, 1, 1, 1)
    s = [np.sin(2 * np.pi * k[i] / L[i]) ** 2 for i in range(4)]
    assert abs(sum(s) - 3.75) < 1e-12 and len({round(v, 6) for v in s}) == 2


# ---------------------------------------------------------------------------------------------------
# second, link-centric dense assembly of D (numpy), compared entry by entry
# ---------------------------------------------------------------------------------------------------
def dense_D_linkwise(L, U, antiperiodic):
    """Every link (x,mu) contributes +1/2 s U to row x / column x+mu and -1/2 s U^dagger to the
    transposed position, so the matrix is anti-Hermitian by construction."""
    Lx, Ly, Lz, Lt = L
    V = int(np.prod(L))
    Uc = c(U)
    x, y, z, t = coords(L)
    eta = [np.ones(V), (-1.0) ** x, (-1.0) ** (x + y), (-1.0) ** (x + y + z)]
    idx = np.arange(V).reshape(Lt, Lz, Ly, Lx)
    D = np.zeros((V, 3, V, 3), dtype=np.complex128)
    for mu in range(4):
        fwd = np.roll(idx, -1, axis=3 - mu).ravel()
        s = eta[mu].copy()
        if antiperiodic and mu == 3:
            s[t == Lt - 1] *= -1
        for n in range(V):
            D[n, :, fwd[n], :] += 0.5 * s[n] * Uc[mu, n]
            D[fwd[n], :, n, :] -= 0.5 * s[n] * Uc[mu, n].conj().T
    return D.reshape(3 * V, 3 * V)


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 2, 2, 4), (2, 4, 6, 2)])
@pytest.mark.parametrize("antiperiodic", [True, False])
def test_dense_linkwise_assembly_matches_oracle(L, antiperiodic):
    U = links(L, seed=5)
    V = int(np.prod(L))
    D = dense_D_linkwise(L, U, antiperiodic)
    assert np.abs(D + D.conj().T).max() == 0.0
    me, mo = parity_mask(L, 0), parity_mask(L, 1)
    me3, mo3 = np.repeat(me, 3), np.repeat(mo, 3)
    assert not D[np.ix_(me3, me3)].any() and not D[np.ix_(mo3, mo3)].any()     # D_ee = D_oo = 0
    D_oe = D[np.ix_(mo3, me3)]
    D_eo = D[np.ix_(me3, mo3)]
    rng = np.random.default_rng(3)
    for _ in range(2):
        fe = rng.standard_normal((V // 2, 3, 2))
        fo = rng.standard_normal((V // 2, 3, 2))
        assert np.abs(c(oracle.doe(L, U, fe, antiperiodic)).ravel() - D_oe @ c(fe).ravel()).max() < 1e-14
        assert np.abs(c(oracle.deo(L, U, fo, antiperiodic)).ravel() - D_eo @ c(fo).ravel()).max() < 1e-14


# ---------------------------------------------------------------------------------------------------
# P5  dense inversion for every shift, P6 CG invariants
# ---------------------------------------------------------------------------------------------------
def dense_A(L, U, mass, antiperiodic=True):
    """A = m^2 - D_eo D_oe as a dense matrix, column by column through the oracle operator."""
    n = int(np.prod(L)) // 2 * 3
    A = np.empty((n, n), dtype=np.complex128)
    e = np.zeros((n, 2))
    for j in range(n):
        e[:] = 0.0
        e[j, 0] = 1.0
        A[:, j] = c(oracle.mdagm(L, U, mass, 0.0, e.reshape(-1, 3, 2), antiperiodic)).ravel()
    return A


@pytest.mark.parametrize("L,mass,shifts", [
    ((2, 2, 2, 2), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
    ((2, 2, 2, 2), 0.05, [0.3, 0.0, 2.0, 1e-3]),                     # base shift is not the first one
    ((4, 2, 2, 4), 0.02, [1e-3, 1e-2, 1e-1, 1.0]),
    ((4, 4, 4, 4), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)]),
])
def test_mshift_cg_against_dense_solve(L, mass, shifts):
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    A = dense_A(L, U, mass)
    assert np.abs(A - A.conj().T).max() < 1e-14                      # Hermitian
    ev = np.linalg.eigvalsh(A)
    assert ev.min() >= mass * mass * (1 - 1e-9) and ev.max() < 7.5   # positive definite
    tol = 1e-10
    x, info = oracle.mshift_cg(L, U, mass, b, shifts, tol)
    assert info["status"] == 0 and info["rel_res"] <= tol
    bn = np.linalg.norm(c(b))
    for i, sigma in enumerate(shifts):
        ref = np.linalg.solve(A + sigma * np.eye(A.shape[0]), c(b).ravel())
        err = np.linalg.norm(c(x[i]).ravel() - ref) / np.linalg.norm(ref)
        cond = (ev.max() + sigma) / (ev.min() + sigma)
        assert err < 5 * tol * cond ** 0.5 and err < 1e-6, (i, err)
        true_res = np.linalg.norm(c(b).ravel() - (A + sigma * np.eye(A.shape[0])) @ c(x[i]).ravel()) / bn
        assert true_res < 3 * tol, (i, true_res)
    # freeze schedule: larger shifts converge no later than smaller ones; the smallest runs to the end
    order = np.argsort(shifts)
    fr = np.array(info["freeze_iter"])[order]
    assert np.all(np.diff(fr) <= 0) and fr[0] == info["iters"]


def dense_A_linkwise(L, U, mass, antiperiodic=True):
    """A = m^2 - D_eo D_oe from the link-centric numpy assembly of D: shares nothing with the oracle."""
    D = dense_D_linkwise(L, U, antiperiodic)
    me3, mo3 = np.repeat(parity_mask(L, 0), 3), np.repeat(parity_mask(L, 1), 3)
    D_oe, D_eo = D[np.ix_(mo3, me3)], D[np.ix_(me3, mo3)]
    return mass * mass * np.eye(D_oe.shape[1]) - D_eo @ D_oe


def textbook_cg(M, b, nit):
    """Plain CG (Hestenes-Stiefel) on one dense Hermitian system M x = b, zero initial guess, own loop and own
    dot products.  Returns the relative residual norms |r_n|/|b| and the iterates x_n for n = 0..nit."""
    x, res, p = np.zeros_like(b), b.copy(), b.copy()
    rr = np.vdot(res, res).real
    bb = rr
    norms, iterates = [1.0], [x.copy()]
    for _ in range(nit):
        Mp = M @ p
        a = rr / np.vdot(p, Mp).real
        x = x + a * p
        res = res - a * Mp
        rr_new = np.vdot(res, res).real
        p = res + (rr_new / rr) * p
        rr = rr_new
        norms.append(np.sqrt(rr / bb))
        iterates.append(x.copy())
    return np.array(norms), iterates


# (lattice, mass, shifts, slack): slack = allowed distance between the oracle's freeze iteration and the first
# iteration at which the independent CG's residual is below tol.  +-1 is rounding (the two programs add in a
# different order); the 600-iteration solve on 4^4 at m = 0.01 moves by 2 (R9).
STOP_CASES = [
    ((2, 2, 2, 2), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)], 1),
    ((2, 2, 2, 2), 0.05, [0.3, 0.0, 2.0, 1e-3], 1),
    ((4, 2, 2, 4), 0.02, [1e-3, 1e-2, 1e-1, 1.0], 1),
    ((4, 4, 4, 4), 0.1, [1e-2 * 10 ** (i / 2) for i in range(6)], 1),
    ((4, 4, 4, 4), 0.01, [1e-4 * 10 ** (i / 2) for i in range(8)], 2),
]


@pytest.mark.parametrize("L,mass,shifts,slack", STOP_CASES)
def test_stop_and_freeze_iterations_against_independent_cg_per_shift(L, mass, shifts, slack):
    """In exact arithmetic the multi-shift iterate of system i IS the CG iterate of (A + sigma_i) x = b, and its
    residual is zeta_i r (refs 32/33; R5).  So the rules R6/R7 say: shift i is frozen at
    the FIRST iteration n at which a plain CG on that system alone has |r_n| <= tol |b|, its solution is that
    CG's n-th iterate, and the solve stops when the smallest shift gets there.  Checked against a textbook CG in
    numpy on the dense matrix assembled link by link (no oracle code on that side).  This pins the freeze test
    (zeta_i^2 |r|^2 against tol^2 |b|^2), the stopping test and the reported counts from BOTH sides: freezing
    or stopping later than necessary fails as well as earlier ("stopping residuals")."""
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    bv = c(b).ravel()
    A = dense_A_linkwise(L, U, mass)
    tol = 1e-10
    x, info = oracle.mshift_cg(L, U, mass, b, shifts, tol)
    assert info["status"] == 0
    i0 = int(np.argmin(shifts))
    assert info["freeze_iter"][i0] == info["iters"] == max(info["freeze_iter"])
    for i, sigma in enumerate(shifts):
        M = A + sigma * np.eye(A.shape[0])
        fz = info["freeze_iter"][i]
        norms, iterates = textbook_cg(M, bv, fz + slack + 1)
        first = int(np.argmax(norms <= tol))
        assert norms[first] <= tol and abs(first - fz) <= slack, (i, sigma, first, fz)
        # not later than necessary: well before the freeze iteration the system had NOT converged ...
        assert norms[fz - slack - 1] > tol, (i, norms[fz - slack - 1])
        # ... and the frozen x_i is that CG's iterate of the same iteration, not a later (more accurate) one
        xi = c(x[i]).ravel()
        assert np.linalg.norm(xi - iterates[fz]) <= 1e-9 * np.linalg.norm(iterates[fz]), (i, sigma)
        true_res = np.linalg.norm(bv - M @ xi) / np.linalg.norm(bv)
        # zeta_i |r| at the freeze iteration = |r_n| of the system's own CG (the recurrences differ by rounding)
        band = norms[fz - slack:fz + slack + 1]
        assert 0.5 * band.min() <= true_res <= 2.0 * band.max() and true_res <= tol * 1.01, (i, true_res, band)
        if i == i0:      # the reported residual is that of the base system at the stop
            assert 0.5 * band.min() <= info["rel_res"] <= 2.0 * band.max() and info["rel_res"] <= tol


def test_mshift_cg_fixed_iteration_count_and_first_step():
    # after exactly one iteration x_i = a_0/(1 + delta_i a_0) b with a_0 = <b,b>/<b,B b>: the exact
    # first CG step of every shifted system (closed form, independent of the zeta recurrence code path)
    L, mass = (4, 4, 2, 2), 0.1
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    shifts = [0.05, 0.5, 5.0]
    x, info = oracle.mshift_cg(L, U, mass, b, shifts, 1e-30, max_iter=1)
    assert info["status"] == 1 and info["iters"] == 1
    Bb = oracle.mdagm(L, U, mass, shifts[0], b)
    a0 = vdot(b, b).real / vdot(b, Bb).real
    for i, s in enumerate(shifts):
        ai = a0 / (1 + (s - shifts[0]) * a0)
        assert np.abs(c(x[i]) - ai * c(b)).max() < 1e-14
    # and x after n iterations lies in the Krylov space and minimises: compare 5 iterations with dense CG
    # optimum: x_n = argmin over K_n of the A-norm error -> check Galerkin condition r_n _|_ K_n.
    nit = 5
    x, info = oracle.mshift_cg(L, U, mass, b, shifts, 1e-30, max_iter=nit)
    for i, s in enumerate(shifts):
        res = c(b) - c(oracle.mdagm(L, U, mass, s, x[i]))
        k = c(b)
        for _ in range(nit):
            assert abs(np.vdot(k.ravel(), res.ravel())) < 1e-10 * np.linalg.norm(k) * np.linalg.norm(c(b))
            k = c(oracle.mdagm(L, U, mass, s, r(k)))


def test_mshift_cg_zero_source_and_single_shift():
    L = (2, 2, 2, 2)
    U = links(L)
    b0 = np.zeros((8, 3, 2))
    x, info = oracle.mshift_cg(L, U, 0.1, b0, [0.0, 1.0], 1e-10)
    assert info["iters"] == 0 and info["status"] == 0 and not x.any()
    b = random_parity_field(L, 5)
    x, info = oracle.mshift_cg(L, U, 0.1, b, [0.25], 1e-12)
    assert info["status"] == 0
    res = c(b) - c(oracle.mdagm(L, U, 0.1, 0.25, x[0]))
    assert np.linalg.norm(res) < 3e-12 * np.linalg.norm(c(b))


def test_reductions_do_not_depend_on_thread_count():
    L = (4, 4, 4, 4)
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    shifts = [1e-3, 1e-1]
    n0 = oracle.num_threads()
    try:
        oracle.set_num_threads(1)
        x1, i1 = oracle.mshift_cg(L, U, 0.05, b, shifts, 1e-10)
        oracle.set_num_threads(max(2, n0))
        x2, i2 = oracle.mshift_cg(L, U, 0.05, b, shifts, 1e-10)
    finally:
        oracle.set_num_threads(n0)
    assert i1 == i2 and np.array_equal(x1, x2)


def test_iteration_count_moves_under_one_ulp_perturbations():
    """DESIGN.md R9: for solves of several hundred iterations the count at which |r| crosses tol*|b| is
    sensitive to the last bit of the input, while the solutions are not.  This is why the GPU parity
    tests compare iteration counts with the oracle's own band (+-1) rather than with a single number."""
    L, mass, shifts, tol = (4, 6, 8, 10), 0.02, [1e-2, 1e-3, 1e-1, 1.0, 0.5], 1e-10
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    x0, i0 = oracle.mshift_cg(L, U, mass, b, shifts, tol)
    counts = [i0["iters"], oracle.mshift_cg(L, U, mass, b, shifts, tol, sum_order=1)[1]["iters"]]
    rng = np.random.default_rng(0)
    for _ in range(4):
        bp = b * (1.0 + rng.integers(-1, 2, size=b.shape) * 2.0 ** -52)
        xp, ip = oracle.mshift_cg(L, U, mass, bp, shifts, tol)
        counts.append(ip["iters"])
        for i in range(len(shifts)):
            assert np.linalg.norm(xp[i] - x0[i]) <= 1e-9 * np.linalg.norm(x0[i])
    assert 0 <= max(counts) - min(counts) <= 6 and min(counts) > 700


# ---------------------------------------------------------------------------------------------------
# rational function of the Eq. 2 operator: y = alpha0 b + sum_i alpha_i (A+sigma_i)^-1 b
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,mass", [((2, 2, 2, 2), 0.05), ((4, 2, 2, 4), 0.02)])
def test_rational_apply_against_dense_function_of_the_matrix(L, mass):
    """r(x) = (x+c1)(x+c2)(x+c3) / ((x+s1)(x+s2)(x+s3)) has the partial fractions 1 + sum_i alpha_i/(x+s_i)
    with alpha_i = prod_j (c_j - s_i) / prod_{j != i} (s_j - s_i); r(A) b is computed independently from the
    eigen-decomposition of the dense A.  Pins alpha0, the pairing alpha_i <-> sigma_i and the signs."""
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    A = dense_A(L, U, mass)
    ev, W = np.linalg.eigh(A)
    cz = np.array([0.7, 0.03, 2.5])
    sp = np.array([0.2, 1.3, 0.004])                                 # base shift is the last one
    alpha = np.array([np.prod(cz - sp[i]) / np.prod(np.delete(sp, i) - sp[i]) for i in range(3)])
    rl = np.prod(ev[:, None] + cz[None, :], axis=1) / np.prod(ev[:, None] + sp[None, :], axis=1)
    ref = W @ (rl * (W.conj().T @ c(b).ravel()))
    y, info = oracle.rational_apply(L, U, mass, b, 1.0, alpha, sp, 1e-12)
    assert info["status"] == 0
    assert np.linalg.norm(c(y).ravel() - ref) <= 1e-9 * np.linalg.norm(ref)
    # alpha0 alone, and one pole alone against numpy.linalg.solve
    y0, _ = oracle.rational_apply(L, U, mass, b, -2.5, [0.0, 0.0], [0.1, 0.2], 1e-12)
    assert np.abs(c(y0) + 2.5 * c(b)).max() < 1e-14
    y1, _ = oracle.rational_apply(L, U, mass, b, 0.0, [3.0], [0.3], 1e-12)
    ref1 = 3.0 * np.linalg.solve(A + 0.3 * np.eye(A.shape[0]), c(b).ravel())
    assert np.linalg.norm(c(y1).ravel() - ref1) <= 1e-10 * np.linalg.norm(ref1)


def test_rational_apply_product_of_two_inverses():
    """1/((x+s1)(x+s2)) = [1/(x+s1) - 1/(x+s2)]/(s2-s1): applying (A+s2)(A+s1) to y must give b back."""
    L, mass, s1, s2 = (4, 4, 4, 4), 0.05, 0.01, 0.4
    U = links(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    y, info = oracle.rational_apply(L, U, mass, b, 0.0, [1 / (s2 - s1), -1 / (s2 - s1)], [s1, s2], 1e-12)
    assert info["status"] == 0
    back = oracle.mdagm(L, U, mass, s2, oracle.mdagm(L, U, mass, s1, y))
    assert np.linalg.norm(back - b) <= 1e-10 * np.linalg.norm(b)


# ---------------------------------------------------------------------------------------------------
# general U(1) field u_mu(x) = exp(i theta_mu(x)) on the links
# ---------------------------------------------------------------------------------------------------
def u1_phases(L, seed=11):
    return gen.random_u1_phases(L, seed).numpy()


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 2, 4, 6), (4, 6, 4, 4)])
@pytest.mark.parametrize("antiperiodic", [True, False])
def test_u1_antihermiticity(L, antiperiodic):
    """u is unitary, so D stays anti-Hermitian: the backward hop must carry conj(u) of the neighbour's link."""
    U, th = links(L), u1_phases(L)
    chi, psi = random_parity_field(L, 1), random_parity_field(L, 2)
    lhs = vdot(chi, oracle.deo(L, U, psi, antiperiodic, theta=th))
    rhs = -np.conj(vdot(psi, oracle.doe(L, U, chi, antiperiodic, theta=th)))
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # and the field does something
    assert np.abs(oracle.deo(L, U, psi, antiperiodic, theta=th) - oracle.deo(L, U, psi, antiperiodic)).max() > 0.1


@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 2, 4, 6)])
def test_u1_gauge_covariance(L):
    """theta'_mu(x) = theta_mu(x) + a(x) - a(x+mu)  =>  D[theta'] (e^{ia} psi) = e^{ia} D[theta] psi.
    Pins which site each theta belongs to and the direction of the phase on forward and backward hops."""
    Lx, Ly, Lz, Lt = L
    V = int(np.prod(L))
    U, th = links(L), u1_phases(L)
    a = np.random.default_rng(4).uniform(-np.pi, np.pi, V)
    a4 = a.reshape(Lt, Lz, Ly, Lx)
    th2 = np.stack([th[mu] + a - np.roll(a4, -1, axis=3 - mu).ravel() for mu in range(4)])
    for p_in in (0, 1):
        psi = random_parity_field(L, 5 + p_in)
        m_in, m_out = parity_mask(L, p_in), parity_mask(L, 1 - p_in)
        psi_g = r(np.exp(1j * a[m_in])[:, None] * c(psi))
        lhs = c(oracle.dslash(L, U, psi_g, 1 - p_in, True, theta=th2))
        rhs = np.exp(1j * a[m_out])[:, None] * c(oracle.dslash(L, U, psi, 1 - p_in, True, theta=th))
        assert np.abs(lhs - rhs).max() < 1e-13


@pytest.mark.parametrize("L,k", [((4, 6, 4, 4), (1, 2, 0, 3)), ((2, 4, 6, 8), (1, 0, 2, 5))])
def test_u1_constant_phase_shifts_the_momentum(L, k):
    """Unit links, periodic, theta_mu(x) = phi_mu: D_eo D_oe e^{ipx} = -sum_mu sin^2(p_mu + phi_mu) e^{ipx}
    (an imaginary chemical potential is a constant theta_t).  Pins the sign of theta."""
    U = gen.unit_links(L).numpy()
    V = int(np.prod(L))
    phi = np.array([0.3, -0.7, 1.1, 0.45])
    th = np.repeat(phi[:, None], V, axis=1)
    x = coords(L)
    p = [2 * np.pi * k[mu] / L[mu] for mu in range(4)]
    wave = np.exp(1j * sum(p[mu] * x[mu] for mu in range(4)))
    col = np.array([0.3 - 0.2j, 1.0, -0.5j])
    psi = r(wave[parity_mask(L, 0)][:, None] * col[None, :])
    out = c(oracle.deo(L, U, oracle.doe(L, U, psi, False, theta=th), False, theta=th))
    lam = -sum(np.sin(p[mu] + phi[mu]) ** 2 for mu in range(4))
    assert np.abs(out - lam * c(psi)).max() < 1e-13
    lam0 = -sum(np.sin(p[mu]) ** 2 for mu in range(4))
    assert abs(lam - lam0) > 0.05


def test_u1_phase_pi_on_the_last_time_links_is_the_antiperiodic_boundary():
    """"by which we handle antiperiodic boundary conditions": theta = pi on the links leaving
    t = Lt-1 with the periodic operator must equal the antiperiodic operator without theta."""
    L = (4, 2, 4, 6)
    U = links(L)
    V = int(np.prod(L))
    th = np.zeros((4, V))
    th[3, coords(L)[3] == L[3] - 1] = np.pi
    for p_in in (0, 1):
        psi = random_parity_field(L, 8 + p_in)
        a = oracle.dslash(L, U, psi, 1 - p_in, False, theta=th)
        b = oracle.dslash(L, U, psi, 1 - p_in, True)
        assert np.abs(a - b).max() < 1e-14


def test_u1_mshift_cg_against_dense_solve():
    L, mass, shifts = (4, 2, 2, 4), 0.05, [1e-2, 1e-1, 1.0]
    U, th = links(L), u1_phases(L)
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    n = int(np.prod(L)) // 2 * 3
    A = np.empty((n, n), dtype=np.complex128)
    e = np.zeros((n, 2))
    for j in range(n):
        e[:] = 0.0
        e[j, 0] = 1.0
        A[:, j] = c(oracle.mdagm(L, U, mass, 0.0, e.reshape(-1, 3, 2), True, theta=th)).ravel()
    assert np.abs(A - A.conj().T).max() < 1e-14 and np.linalg.eigvalsh(A).min() >= mass * mass * (1 - 1e-9)
    x, info = oracle.mshift_cg(L, U, mass, b, shifts, 1e-11, theta=th)
    assert info["status"] == 0
    for i, sigma in enumerate(shifts):
        ref = np.linalg.solve(A + sigma * np.eye(n), c(b).ravel())
        assert np.linalg.norm(c(x[i]).ravel() - ref) <= 1e-8 * np.linalg.norm(ref)
