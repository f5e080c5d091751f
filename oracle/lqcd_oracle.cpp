// lqcd_oracle.cpp -- CPU ORACLE for the staggered Dslash and the multi-shift CG.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
// header, table or helper with the CUDA library (paper_1801_01473_b200/csrc): different language unit,
// different storage (array-of-structs std::complex<double> indexed through full lexicographic
// coordinates, against the CUDA side's per-parity structure-of-arrays double2 with checkerboard index
// arithmetic), written directly from the paper and the readings listed in DESIGN.md.
//
// What it computes, and from where:
//   * D_oe / D_eo, the off-diagonal even/odd blocks of the staggered Dirac matrix: nearest-neighbour
//     hopping "proportional to U_mu(x)", multiplied by the U(1) field that carries the
//     staggered phases and the antiperiodic time boundary, with D_oe^dagger = -D_eo
//     (PAPER.md:L80).  Normalisation 1/2 and the eta convention are DESIGN.md readings R1, R2, R3:
//         (D psi)(x) = 1/2 sum_mu [ s_mu(x) U_mu(x) psi(x+mu) - s_mu(x-mu) U_mu(x-mu)^dagger psi(x-mu) ]
//         s_mu(x) = eta_mu(x) bc_mu(x); eta = (1, (-1)^x, (-1)^(x+y), (-1)^(x+y+z));
//         bc_t(x) = -1 on links leaving the last time slice (antiperiodic), +1 otherwise.
//     This is the plain definition written out: four nested coordinate loops, no blocking.
//   * optionally (the *_u1 entry points) the general U(1) field u_mu(x) = cos(theta_mu(x)) + i sin(theta_mu(x))
//     by which "pseudofermions must be multiplied" together with U_mu(x) -- imaginary chemical potential and
//     background fields; theta is stored, u recomputed, as the paper does.
//   * third-row reconstruction r2 = conj(r0 x r1) of a compressed link.
//   * the rational function alpha0 b + sum_i alpha_i x_i of the Eq. 2 operator.
//   * the shifted ("multimass") conjugate gradient for (m^2 - D_eo D_oe + sigma_i) x_i = b
//     (Eq. 2; refs 32, 33).  The paper gives no pseudo-code; the algorithm is
//     followed step by step in the order and notation of DESIGN.md reading R5.
//
// Pins (tests/test_oracle_pins.py, all CPU): anti-hermiticity, gauge covariance, free-field closed form
// (periodic and antiperiodic), dense 2^4 / small-lattice inversion with numpy for every shift, unitarity
// of reconstructed links, CG invariants, and the stop / freeze iterations and the frozen iterates against an
// independent textbook CG per shifted system on the dense matrix.  No function here is "parity unpinned".
//
// Storage conventions of this file:
//   lex = x + Lx*(y + Ly*(z + Lz*t)),  parity(lex) = (x+y+z+t)&1, even = 0.
//   gauge field  U[mu][lex][row][col]            (the canonical user layout of include/lqcd.h)
//   parity field f[lex>>1][colour]               (array-of-structs over the sites of one parity;
//                                                 Lx is even so lex>>1 numbers them 0..V/2-1)
//   boundary ("vec3_soa") layout v[colour*Vh + (lex>>1)]: see oracle_soa_to_aos.
//
// Reductions are deterministic: one partial per time slice, partials added in slice order, so the
// result does not depend on the OpenMP thread count (reading R8).

#include <complex>
#include <cstdint>
#include <cstring>
#include <cmath>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;

namespace {

struct Lattice {
    int L[4];
    int64_t V, Vh;
    int64_t lex(int x, int y, int z, int t) const {
        return x + (int64_t)L[0] * (y + (int64_t)L[1] * (z + (int64_t)L[2] * t));
    }
};

Lattice make_lattice(const int* L) {
    Lattice lat;
    for (int i = 0; i < 4; ++i) lat.L[i] = L[i];
    lat.V = (int64_t)L[0] * L[1] * L[2] * L[3];
    lat.Vh = lat.V / 2;
    return lat;
}

// staggered phase eta_mu at a site (R2)
int eta(int mu, const int c[4]) {
    int e = 0;
    for (int nu = 0; nu < mu; ++nu) e += c[nu];
    return (e & 1) ? -1 : 1;
}

// sign of the link (site c, direction mu): eta times the antiperiodic boundary sign (R3)
double link_sign(const Lattice& lat, int mu, const int c[4], int antiperiodic) {
    double s = eta(mu, c);
    if (antiperiodic && mu == 3 && c[3] == lat.L[3] - 1) s = -s;
    return s;
}

// U(1) factor of the link (site lex, direction mu) beyond the staggered phase and the boundary sign:
// u = cos(theta) + i sin(theta) with theta_mu(x) stored, as the paper does for the imaginary chemical
// potential and background fields.  theta == NULL means no such field (u = 1).
cplx u1_factor(const double* theta, int64_t V, int mu, int64_t lex) {
    if (!theta) return cplx(1.0, 0.0);
    const double th = theta[(int64_t)mu * V + lex];
    return cplx(std::cos(th), std::sin(th));
}

// Apply D to a field living on parity 1-p, result on the sites of parity p.  The hopping term between x and
// x+mu is s_mu(x) u_mu(x) U_mu(x) forwards and its negative adjoint backwards.
void dslash(const Lattice& lat, const cplx* U, const double* theta, const cplx* in, cplx* out, int p,
            int antiperiodic) {
    const int64_t V = lat.V;
#pragma omp parallel for collapse(2) schedule(static)
    for (int t = 0; t < lat.L[3]; ++t)
        for (int z = 0; z < lat.L[2]; ++z)
            for (int y = 0; y < lat.L[1]; ++y)
                for (int x = 0; x < lat.L[0]; ++x) {
                    if (((x + y + z + t) & 1) != p) continue;
                    const int c[4] = {x, y, z, t};
                    const int64_t here = lat.lex(x, y, z, t);
                    cplx acc[3] = {0.0, 0.0, 0.0};
                    for (int mu = 0; mu < 4; ++mu) {
                        int cf[4] = {x, y, z, t}, cb[4] = {x, y, z, t};
                        cf[mu] = (c[mu] + 1) % lat.L[mu];
                        cb[mu] = (c[mu] + lat.L[mu] - 1) % lat.L[mu];
                        const int64_t fwd = lat.lex(cf[0], cf[1], cf[2], cf[3]);
                        const int64_t bwd = lat.lex(cb[0], cb[1], cb[2], cb[3]);
                        const cplx* Uf = U + ((int64_t)mu * V + here) * 9;   // U_mu(x)
                        const cplx* Ub = U + ((int64_t)mu * V + bwd) * 9;    // U_mu(x-mu)
                        const cplx* vf = in + (fwd >> 1) * 3;
                        const cplx* vb = in + (bwd >> 1) * 3;
                        const cplx sf = link_sign(lat, mu, c, antiperiodic) * u1_factor(theta, V, mu, here);
                        const cplx sb = link_sign(lat, mu, cb, antiperiodic) * std::conj(u1_factor(theta, V, mu, bwd));
                        for (int a = 0; a < 3; ++a) {
                            cplx f = 0.0, b = 0.0;
                            for (int bb = 0; bb < 3; ++bb) {
                                f += Uf[3 * a + bb] * vf[bb];
                                b += std::conj(Ub[3 * bb + a]) * vb[bb];
                            }
                            acc[a] += sf * f - sb * b;
                        }
                    }
                    for (int a = 0; a < 3; ++a) out[(here >> 1) * 3 + a] = 0.5 * acc[a];
                }
}

// Re <u, v> = Re sum conj(u) v over a parity field; one partial per time slice, added in slice order
// (sum_order 0: increasing t, the default reading R8; 1: decreasing t -- an equally valid order, used by
// the tests to measure how far the iteration count moves under a rounding-level perturbation, R9).
double re_dot(const Lattice& lat, const cplx* u, const cplx* v, int sum_order = 0) {
    const int Lt = lat.L[3];
    const int64_t per_slice = lat.Vh / Lt * 3;
    std::vector<double> partial(Lt, 0.0);
#pragma omp parallel for schedule(static)
    for (int t = 0; t < Lt; ++t) {
        double s = 0.0;
        for (int64_t j = t * per_slice; j < (t + 1) * per_slice; ++j)
            s += u[j].real() * v[j].real() + u[j].imag() * v[j].imag();
        partial[t] = s;
    }
    double s = 0.0;
    if (sum_order == 0)
        for (int t = 0; t < Lt; ++t) s += partial[t];
    else
        for (int t = Lt - 1; t >= 0; --t) s += partial[t];
    return s;
}

// y += a x
void axpy(int64_t n, double a, const cplx* x, cplx* y) {
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j) y[j] += a * x[j];
}

// y = a x + b y
void axpby(int64_t n, double a, const cplx* x, double b, cplx* y) {
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j) y[j] = a * x[j] + b * y[j];
}

}  // namespace

extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// out (parity p, Vh*3 complex, AoS) = D in (parity 1-p).  U canonical [4][V][3][3].
void oracle_dslash(const int* L, const double* U, const double* in, double* out, int out_parity,
                   int antiperiodic) {
    Lattice lat = make_lattice(L);
    dslash(lat, (const cplx*)U, nullptr, (const cplx*)in, (cplx*)out, out_parity, antiperiodic);
}

// Same with the U(1) field u_mu(x) = exp(i theta_mu(x)), theta[mu][lex].
void oracle_dslash_u1(const int* L, const double* U, const double* theta, const double* in, double* out,
                      int out_parity, int antiperiodic) {
    Lattice lat = make_lattice(L);
    dslash(lat, (const cplx*)U, theta, (const cplx*)in, (cplx*)out, out_parity, antiperiodic);
}

// D_oe: even -> odd;  D_eo: odd -> even
void oracle_doe(const int* L, const double* U, const double* in_even, double* out_odd, int antiperiodic) {
    oracle_dslash(L, U, in_even, out_odd, 1, antiperiodic);
}
void oracle_deo(const int* L, const double* U, const double* in_odd, double* out_even, int antiperiodic) {
    oracle_dslash(L, U, in_odd, out_even, 0, antiperiodic);
}

// out = (m^2 + sigma) in - D_eo D_oe in       (Eq. 2; even -> even)
void oracle_mdagm_u1(const int* L, const double* U, const double* theta, double mass, double sigma,
                     const double* in_even, double* out_even, int antiperiodic) {
    Lattice lat = make_lattice(L);
    std::vector<cplx> tmp(lat.Vh * 3);
    const cplx* in = (const cplx*)in_even;
    cplx* out = (cplx*)out_even;
    dslash(lat, (const cplx*)U, theta, in, tmp.data(), 1, antiperiodic);
    dslash(lat, (const cplx*)U, theta, tmp.data(), out, 0, antiperiodic);
    const double c = mass * mass + sigma;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < lat.Vh * 3; ++j) out[j] = c * in[j] - out[j];
}
void oracle_mdagm(const int* L, const double* U, double mass, double sigma, const double* in_even,
                  double* out_even, int antiperiodic) {
    oracle_mdagm_u1(L, U, nullptr, mass, sigma, in_even, out_even, antiperiodic);
}

// Gauge-link compression: overwrite the third row of every link by conj(r0 x r1).
void oracle_reconstruct_third_row(int64_t nlinks, double* U) {
    cplx* u = (cplx*)U;
    for (int64_t n = 0; n < nlinks; ++n) {
        cplx* r0 = u + n * 9;
        cplx* r1 = r0 + 3;
        cplx* r2 = r0 + 6;
        r2[0] = std::conj(r0[1] * r1[2] - r0[2] * r1[1]);
        r2[1] = std::conj(r0[2] * r1[0] - r0[0] * r1[2]);
        r2[2] = std::conj(r0[0] * r1[1] - r0[1] * r1[0]);
    }
}

// Layout helpers between this file's AoS parity fields and the boundary layout of include/lqcd.h
// (the paper's vec3_soa): soa[c*Vh + k] <-> aos[k*3 + c], k = lex>>1.
void oracle_soa_to_aos(int64_t Vh, const double* soa, double* aos) {
    const cplx* s = (const cplx*)soa;
    cplx* a = (cplx*)aos;
    for (int64_t k = 0; k < Vh; ++k)
        for (int c = 0; c < 3; ++c) a[k * 3 + c] = s[c * Vh + k];
}
void oracle_aos_to_soa(int64_t Vh, const double* aos, double* soa) {
    const cplx* a = (const cplx*)aos;
    cplx* s = (cplx*)soa;
    for (int64_t k = 0; k < Vh; ++k)
        for (int c = 0; c < 3; ++c) s[c * Vh + k] = a[k * 3 + c];
}

// Restriction of a whole-lattice field [V][3] to the sites of one parity -> AoS parity field, and back
// (sites of the other parity are left untouched by the scatter).
void oracle_restrict(const int* L, int parity, const double* full, double* aos) {
    Lattice lat = make_lattice(L);
    const cplx* f = (const cplx*)full;
    cplx* a = (cplx*)aos;
    for (int t = 0; t < lat.L[3]; ++t)
        for (int z = 0; z < lat.L[2]; ++z)
            for (int y = 0; y < lat.L[1]; ++y)
                for (int x = 0; x < lat.L[0]; ++x) {
                    if (((x + y + z + t) & 1) != parity) continue;
                    const int64_t l = lat.lex(x, y, z, t);
                    for (int c = 0; c < 3; ++c) a[(l >> 1) * 3 + c] = f[l * 3 + c];
                }
}
void oracle_scatter(const int* L, int parity, const double* aos, double* full) {
    Lattice lat = make_lattice(L);
    const cplx* a = (const cplx*)aos;
    cplx* f = (cplx*)full;
    for (int t = 0; t < lat.L[3]; ++t)
        for (int z = 0; z < lat.L[2]; ++z)
            for (int y = 0; y < lat.L[1]; ++y)
                for (int x = 0; x < lat.L[0]; ++x) {
                    if (((x + y + z + t) & 1) != parity) continue;
                    const int64_t l = lat.lex(x, y, z, t);
                    for (int c = 0; c < 3; ++c) f[l * 3 + c] = a[(l >> 1) * 3 + c];
                }
}

// Multi-shift CG, reading R5, step by step.
//   b, x[i]: AoS even-parity fields (Vh*3 complex).  x is nshift fields stored back to back.
//   Outputs: *iters; freeze_iter[nshift] (iteration after which shift i stopped being updated, or the
//   final count if it never froze); *rel_res = sqrt(rr/bb) of the base recurrence residual.
//   sum_order: order in which the per-slice partials of every scalar product are added (see re_dot).
//   Returns 0 on convergence, 1 if max_iter was reached, 2 on breakdown (pAp <= 0 or non-finite).
//   theta: the U(1) field of oracle_dslash_u1, or NULL.
int oracle_mshift_cg_u1(const int* L, const double* U, const double* theta, double mass, int antiperiodic,
                        const double* b_even, const double* shifts, int nshift, double tol, int max_iter,
                        int sum_order, double* x_out, int* iters, int* freeze_iter, double* rel_res) {
    Lattice lat = make_lattice(L);
    const int64_t n = lat.Vh * 3;
    const cplx* Uc = (const cplx*)U;
    const cplx* b = (const cplx*)b_even;
    cplx* x = (cplx*)x_out;

    int i0 = 0;
    for (int i = 1; i < nshift; ++i)
        if (shifts[i] < shifts[i0]) i0 = i;
    const double sigma0 = shifts[i0];
    std::vector<double> delta(nshift);
    for (int i = 0; i < nshift; ++i) delta[i] = shifts[i] - sigma0;

    std::vector<cplx> r(b, b + n), s(n), tmp(n);
    std::vector<std::vector<cplx>> p(nshift, std::vector<cplx>(b, b + n));   // p[i0] is the base p
    std::memset((void*)x, 0, sizeof(cplx) * n * nshift);

    std::vector<double> zeta(nshift, 1.0), zeta_prev(nshift, 1.0), zeta_new(nshift, 1.0);
    std::vector<char> active(nshift, 1);
    double a_prev = 1.0, b_prev = 0.0;
    double rr = re_dot(lat, r.data(), r.data(), sum_order);
    const double bb = rr;
    const double c0 = mass * mass + sigma0;
    int it = 0, status = 0;
    for (int i = 0; i < nshift; ++i) freeze_iter[i] = 0;

    if (bb == 0.0) {
        *iters = 0;
        *rel_res = 0.0;
        return 0;
    }

    for (;;) {
        // s = B(p) = (m^2 + sigma0) p - D_eo (D_oe p)
        cplx* pb = p[i0].data();
        dslash(lat, Uc, theta, pb, tmp.data(), 1, antiperiodic);
        dslash(lat, Uc, theta, tmp.data(), s.data(), 0, antiperiodic);
#pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < n; ++j) s[j] = c0 * pb[j] - s[j];

        const double pAp = re_dot(lat, pb, s.data(), sum_order);
        if (!(pAp > 0.0) || !std::isfinite(pAp)) { status = 2; break; }
        const double a = rr / pAp;

        for (int i = 0; i < nshift; ++i) {
            if (!active[i]) continue;
            zeta_new[i] = zeta[i] * zeta_prev[i] * a_prev /
                          (a_prev * zeta_prev[i] * (1.0 + delta[i] * a) +
                           a * b_prev * (zeta_prev[i] - zeta[i]));
            const double a_i = a * zeta_new[i] / zeta[i];
            axpy(n, a_i, p[i].data(), x + (int64_t)i * n);
        }

        axpy(n, -a, s.data(), r.data());
        const double rr_new = re_dot(lat, r.data(), r.data(), sum_order);
        const double bt = rr_new / rr;

        axpby(n, 1.0, r.data(), bt, pb);
        for (int i = 0; i < nshift; ++i) {
            if (!active[i] || i == i0) continue;
            const double ratio = zeta_new[i] / zeta[i];
            const double b_i = bt * ratio * ratio;
            axpby(n, zeta_new[i], r.data(), b_i, p[i].data());
        }

        for (int i = 0; i < nshift; ++i) {
            if (!active[i]) continue;
            zeta_prev[i] = zeta[i];
            zeta[i] = zeta_new[i];
        }
        a_prev = a;
        b_prev = bt;
        rr = rr_new;
        ++it;

        for (int i = 0; i < nshift; ++i) {
            if (!active[i]) continue;
            if (zeta[i] * zeta[i] * rr <= tol * tol * bb) {
                active[i] = 0;
                freeze_iter[i] = it;
            }
        }
        if (rr <= tol * tol * bb) break;
        if (it >= max_iter) { status = 1; break; }
    }
    for (int i = 0; i < nshift; ++i)
        if (active[i]) freeze_iter[i] = it;
    *iters = it;
    *rel_res = std::sqrt(rr / bb);
    return status;
}

int oracle_mshift_cg(const int* L, const double* U, double mass, int antiperiodic, const double* b_even,
                     const double* shifts, int nshift, double tol, int max_iter, int sum_order,
                     double* x_out, int* iters, int* freeze_iter, double* rel_res) {
    return oracle_mshift_cg_u1(L, U, nullptr, mass, antiperiodic, b_even, shifts, nshift, tol, max_iter, sum_order,
                               x_out, iters, freeze_iter, rel_res);
}

// Rational function of the operator of Eq. 2 applied to a vector,
//     y = alpha0 b + sum_i alpha_i (m^2 - D_eo D_oe + sigma_i)^{-1} b ,
// the partial-fraction form in which the RHMC uses the solutions of Eq. 2: "the fractional power of M(U)
// is approximated ... by a rational function of M(U)" whose poles are the sigma_i.
// Plain definition: solve Eq. 2 for every shift with oracle_mshift_cg, then add the terms in index order.
// Returns the status of the solve.
int oracle_rational_apply(const int* L, const double* U, double mass, int antiperiodic, const double* b_even,
                          double alpha0, const double* alpha, const double* shifts, int nshift, double tol,
                          int max_iter, double* y_out, int* iters, double* rel_res) {
    Lattice lat = make_lattice(L);
    const int64_t n = lat.Vh * 3;
    std::vector<double> x((size_t)nshift * n * 2);
    std::vector<int> freeze(nshift);
    const int status = oracle_mshift_cg(L, U, mass, antiperiodic, b_even, shifts, nshift, tol, max_iter, 0, x.data(),
                                        iters, freeze.data(), rel_res);
    const cplx* b = (const cplx*)b_even;
    const cplx* xs = (const cplx*)x.data();
    cplx* y = (cplx*)y_out;
    for (int64_t j = 0; j < n; ++j) {
        cplx acc = alpha0 * b[j];
        for (int i = 0; i < nshift; ++i) acc += alpha[i] * xs[(int64_t)i * n + j];
        y[j] = acc;
    }
    return status;
}

}  // extern "C"
