"""Seeded synthetic inputs for the staggered Dslash / multi-shift CG path.

TEST / BENCH INFRASTRUCTURE ONLY.  This module holds *none* of the method's arithmetic (no Dirac
operator, no phases, no CG, no even/odd index maps): it only draws random numbers and shapes them into
the two kinds of input the path consumes, in the *canonical user layouts* of ``include/lqcd.h``:

* gauge links  ``links[mu, lex, row, col, {re,im}]``   float64, shape (4, V, 3, 3, 2)
* a site field ``field[lex, colour, {re,im}]``          float64, shape (V, 3, 2)
* (optional) U(1) link phases ``theta[mu, lex]``        float64, shape (4, V), radians

with ``lex = x + Lx*(y + Ly*(z + Lz*t))`` and ``mu = 0..3 = x,y,z,t``.  The same bytes are handed to the
CPU oracle (``oracle/``) and to the CUDA library through their public entry points; neither of them
imports the other and both import only this module ("Input recipe").

Recipe (BASELINE.json configs): every real number is a function of
``(seed, stream, counter)`` only -- a counter-based generator -- so the values do not depend on the
generation order, chunking, device or thread count:

* 64-bit mixer: two rounds of the splitmix64 finaliser over ``counter + seed*G1 + stream*G2``;
* uniform in (0,1): top 53 bits, ``(n + 0.5) * 2**-53``;
* complex Gaussian, re and im iid N(0,1): Box-Muller on the pair of uniforms (2c, 2c+1);
* SU(3) link: rows a0, a1 drawn as complex Gaussian 3-vectors; ``r0 = a0/|a0|``;
  ``a1 -= <r0,a1> r0`` with ``<u,v> = sum conj(u) v``; ``r1 = a1/|a1|``; ``r2 = conj(r0 x r1)``
  (BASELINE.json configs[0]: "Gram-Schmidt rows 1-2, row3=conj(r1 x r2)").

The paper measured on thermalised 32^3x48 / 32^3x64 production configurations that
are not available; these random links stand in for them (strong-coupling limit: same access pattern and
cost per application, worst-case conditioning for the CG).

Everything is written with torch ops so that the same code runs on the CPU (tests) and on the GPU
(full-size bench inputs, where the host would take minutes).  Transcendentals differ in the last ulp
between devices, so one call site must generate once and hand the *same bytes* to both sides.
"""
from __future__ import annotations

import math
from typing import Sequence

import torch

# Seeds of the BASELINE configs.
SEED_LINKS = 180101473
SEED_SOURCE = 180101474

_STREAM_LINKS = 1
_STREAM_FIELD = 2
_STREAM_GAUGE_XFORM = 3
_STREAM_U1 = 4

_MASK64 = (1 << 64) - 1


def _s64(u: int) -> int:
    """Two's-complement view of an unsigned 64-bit constant (torch has no uint64 arithmetic)."""
    u &= _MASK64
    return u - (1 << 64) if u >= (1 << 63) else u


_G1 = _s64(0x9E3779B97F4A7C15)
_G2 = _s64(0xD1B54A32D192ED03)
_M1 = _s64(0xBF58476D1CE4E5B9)
_M2 = _s64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of int64 lanes (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _fmix(x: torch.Tensor) -> torch.Tensor:
    x = x ^ _lsr(x, 30)
    x = x * _M1
    x = x ^ _lsr(x, 27)
    x = x * _M2
    x = x ^ _lsr(x, 31)
    return x


def mix64(seed: int, stream: int, counter: torch.Tensor) -> torch.Tensor:
    """64 pseudo-random bits per int64 counter (wrapping arithmetic mod 2**64)."""
    key = _s64(seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03)
    x = counter + key
    x = _fmix(x)
    x = _fmix(x + _G1)
    return x


def uniform01(seed: int, stream: int, counter: torch.Tensor) -> torch.Tensor:
    """float64 uniform in the open interval (0, 1)."""
    bits = _lsr(mix64(seed, stream, counter), 11)          # 53 bits, non-negative
    return (bits.to(torch.float64) + 0.5) * (2.0 ** -53)


def complex_gaussian(seed: int, stream: int, counter: torch.Tensor) -> torch.Tensor:
    """complex128, re and im iid N(0,1), one number per counter value."""
    u1 = uniform01(seed, stream, 2 * counter)
    u2 = uniform01(seed, stream, 2 * counter + 1)
    rad = torch.sqrt(-2.0 * torch.log(u1))
    ang = (2.0 * math.pi) * u2
    return torch.complex(rad * torch.cos(ang), rad * torch.sin(ang))


def volume(L: Sequence[int]) -> int:
    Lx, Ly, Lz, Lt = L
    return Lx * Ly * Lz * Lt


def _su3_from_rows(a0: torch.Tensor, a1: torch.Tensor) -> torch.Tensor:
    """(n,3),(n,3) complex -> (n,3,3) complex with orthonormal rows and det = 1."""
    r0 = a0 / torch.linalg.vector_norm(a0, dim=-1, keepdim=True)
    a1 = a1 - (r0.conj() * a1).sum(-1, keepdim=True) * r0
    r1 = a1 / torch.linalg.vector_norm(a1, dim=-1, keepdim=True)
    r2 = torch.stack(
        (
            r0[:, 1] * r1[:, 2] - r0[:, 2] * r1[:, 1],
            r0[:, 2] * r1[:, 0] - r0[:, 0] * r1[:, 2],
            r0[:, 0] * r1[:, 1] - r0[:, 1] * r1[:, 0],
        ),
        dim=-1,
    ).conj()
    return torch.stack((r0, r1, r2), dim=1)


def _random_su3(seed: int, stream: int, first: int, count: int, device) -> torch.Tensor:
    """`count` SU(3) matrices number first..first+count-1 of the given stream -> (count,3,3) complex."""
    idx = torch.arange(first, first + count, dtype=torch.int64, device=device)
    ctr = idx[:, None] * 6 + torch.arange(6, dtype=torch.int64, device=device)[None, :]
    a = complex_gaussian(seed, stream, ctr)
    return _su3_from_rows(a[:, 0:3], a[:, 3:6])


def random_su3_links(L: Sequence[int], seed: int = SEED_LINKS, device="cpu",
                     chunk: int = 1 << 20, out: torch.Tensor | None = None) -> torch.Tensor:
    """Canonical gauge field, float64 (4, V, 3, 3, 2).  Link number ``mu*V + lex`` is U_mu(lex)."""
    V = volume(L)
    if out is None:
        out = torch.empty((4, V, 3, 3, 2), dtype=torch.float64, device=device)
    flat = out.view(4 * V, 3, 3, 2)
    for first in range(0, 4 * V, chunk):
        count = min(chunk, 4 * V - first)
        u = _random_su3(seed, _STREAM_LINKS, first, count, out.device)
        flat[first:first + count] = torch.view_as_real(u)
    return out


def slab_sites(L: Sequence[int], rank: int, nranks: int) -> tuple[int, int]:
    """(first lexicographic site, number of sites) of the slab of time slices rank r of nranks owns (the slab
    decomposition cuts the slowest index t into nranks equal parts)."""
    V = volume(L)
    assert L[3] % nranks == 0
    return rank * (V // nranks), V // nranks


def random_su3_links_slab(L: Sequence[int], rank: int, nranks: int, seed: int = SEED_LINKS, device="cpu",
                          chunk: int = 1 << 20) -> torch.Tensor:
    """The part of ``random_su3_links(L)`` that leaves the sites of one slab, (4, V/nranks, 3, 3, 2), drawn
    directly (same counters, hence the same values) so that no rank ever holds the whole field."""
    V = volume(L)
    first_site, n = slab_sites(L, rank, nranks)
    out = torch.empty((4, n, 3, 3, 2), dtype=torch.float64, device=device)
    for mu in range(4):
        for a in range(0, n, chunk):
            count = min(chunk, n - a)
            u = _random_su3(seed, _STREAM_LINKS, mu * V + first_site + a, count, out.device)
            out[mu, a:a + count] = torch.view_as_real(u)
    return out


def gaussian_field_slab(L: Sequence[int], rank: int, nranks: int, seed: int = SEED_SOURCE, device="cpu") -> torch.Tensor:
    """The part of ``gaussian_field(L)`` on the sites of one slab, (V/nranks, 3, 2)."""
    first_site, n = slab_sites(L, rank, nranks)
    ctr = torch.arange(3 * first_site, 3 * (first_site + n), dtype=torch.int64, device=device)
    return torch.view_as_real(complex_gaussian(seed, _STREAM_FIELD, ctr)).reshape(n, 3, 2).contiguous()


def unit_links(L: Sequence[int], device="cpu") -> torch.Tensor:
    """Free field: every link is the identity."""
    V = volume(L)
    out = torch.zeros((4, V, 3, 3, 2), dtype=torch.float64, device=device)
    for a in range(3):
        out[:, :, a, a, 0] = 1.0
    return out


def gaussian_field(L: Sequence[int], seed: int = SEED_SOURCE, device="cpu",
                   chunk: int = 1 << 22) -> torch.Tensor:
    """Site field on the *whole* lattice, float64 (V, 3, 2), re and im iid N(0,1).

    Which parity of it is used is the caller's business (the even-site source of the BASELINE configs is
    the restriction of this field to even sites; the values on the other parity are simply ignored)."""
    V = volume(L)
    out = torch.empty((V, 3, 2), dtype=torch.float64, device=device)
    flat = out.view(3 * V, 2)
    for first in range(0, 3 * V, chunk):
        count = min(chunk, 3 * V - first)
        ctr = torch.arange(first, first + count, dtype=torch.int64, device=device)
        flat[first:first + count] = torch.view_as_real(complex_gaussian(seed, _STREAM_FIELD, ctr))
    return out


def random_gauge_transform(L: Sequence[int], seed: int, device="cpu") -> torch.Tensor:
    """One SU(3) matrix per site, float64 (V, 3, 3, 2) -- input of the gauge-covariance test."""
    V = volume(L)
    return torch.view_as_real(_random_su3(seed, _STREAM_GAUGE_XFORM, 0, V, device)).contiguous()


def random_u1_phases(L: Sequence[int], seed: int = SEED_LINKS, device="cpu") -> torch.Tensor:
    """U(1) phase field theta_mu(x), float64 (4, V), uniform in (-pi, pi): a stand-in for the imaginary chemical
    potential / background field phases of PAPER.md:L159 (canonical layout: theta[mu, lex] belongs to the link
    leaving lex along +mu)."""
    V = volume(L)
    ctr = torch.arange(4 * V, dtype=torch.int64, device=device)
    return ((2.0 * uniform01(seed, _STREAM_U1, ctr) - 1.0) * math.pi).view(4, V)


def shifts_geometric(first: float, last: float, n: int) -> list[float]:
    """sigma_i, i=0..n-1, geometric from `first` to `last` (BASELINE configs 2, 4, 5)."""
    if n == 1:
        return [first]
    ratio = (last / first) ** (1.0 / (n - 1))
    return [first * ratio ** i for i in range(n)]


# The BASELINE.json configs as data (sizes, mass, shifts, tolerance); the inputs are drawn as above.
CONFIGS = {
    "config1_4^4": dict(L=(4, 4, 4, 4), mass=0.01, shifts=[0.0], tol=1e-10),
    "config2_16^4": dict(L=(16, 16, 16, 16), mass=0.01,
                         shifts=[1e-4 * 10 ** (i / 2) for i in range(8)], tol=1e-10),
    "config3_32^4": dict(L=(32, 32, 32, 32), mass=0.01, shifts=[0.0], tol=1e-10),
    "config4_48^4": dict(L=(48, 48, 48, 48), mass=0.0075, shifts=shifts_geometric(1e-5, 1.0, 16),
                         tol=1e-10),
    "config5_64^4": dict(L=(64, 64, 64, 64), mass=0.005, shifts=shifts_geometric(1e-5, 1.0, 16),
                         tol=1e-10),
}
