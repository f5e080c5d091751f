// cg.cuh -- the vector sweeps of the multi-shift CG (steps A7, A8 of DESIGN.md) and layout kernels.
//
// One CG iteration is four launches ("scalar products and sums" + the two operators):
//   K1  t  = D_oe p                                         dslash_kernel<.,0>
//   K2  s  = (m^2+sigma0) p - D_eo t ;  Re<p,s>  -> a, zeta_new_i, a_i      dslash_kernel<.,1>
//   K3  r -= a s ;  |r|^2  -> beta, b_i, freeze flags, stop flag            cg_update_r_kernel
//   K4  for every shift active in this iteration:  x_i += a_i p_i ;  p_i = zeta_new_i r + b_i p_i
//                                                                           cg_update_xp_kernel
// p_i is read once per iteration (x_i and p_i updates share the load).  All scalars stay on the device.
#ifndef LQCD_CG_CUH
#define LQCD_CG_CUH

#include "lqcd_internal.cuh"
#include "reduce.cuh"

#define CG_BLOCK 256

// K0: r = p_i = b, x_i = 0, |b|^2.  In every sweep the vectors are V2<T>; scalars and sums are double.
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_init_kernel(const V2<T>* __restrict__ b, V2<T>* __restrict__ r,
                                                           CgState* st, double* partials, size_t n, double tol) {
    __shared__ double red[32];
    __shared__ int last_flag;
    const int ns = st->nshift;
    const int rational = st->rational;
    const T alpha0 = (T)st->alpha0;
    V2<T>* __restrict__ y = (V2<T>*)st->y;
    double acc = 0.0;
    const V2<T> zero = make_v2((T)0, (T)0);
    for (size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x; j < n; j += (size_t)gridDim.x * CG_BLOCK) {
        const V2<T> v = b[j];
        r[j] = v;
        for (int i = 0; i < ns; ++i) ((V2<T>*)st->p[i])[j] = v;
        if (rational) {
            y[j] = make_v2(alpha0 * v.x, alpha0 * v.y);
        } else {
            for (int i = 0; i < ns; ++i) ((V2<T>*)st->x[i])[j] = zero;
        }
        acc = fma((double)v.x, (double)v.x, acc);
        acc = fma((double)v.y, (double)v.y, acc);
    }
    const double bsum = block_sum<CG_BLOCK>(acc, red);
    if (publish_partial<CG_BLOCK>(bsum, partials, &st->ticket[0], &last_flag)) {
        const double bb = final_sum<CG_BLOCK>(partials, gridDim.x, red);
        if (threadIdx.x == 0) {
            st->ticket[0] = 0;
            cg_scalars_init(st, bb, tol);
        }
    }
}

// K3: r -= a s, |r|^2, then the scalar step that needs it
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_update_r_kernel(V2<T>* __restrict__ r, const V2<T>* __restrict__ s,
                                                               CgState* st, double* partials, size_t n) {
    if (st->stop) return;
    __shared__ double red[32];
    __shared__ int last_flag;
    const T a = (T)st->a;
    double acc = 0.0;
    const size_t stride = (size_t)gridDim.x * CG_BLOCK;
    size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x;
    for (; j + 3 * stride < n; j += 4 * stride) {
        V2<T> rv[4], sv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            rv[u] = r[j + u * stride];
            sv[u] = s[j + u * stride];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            rv[u].x = fma(-a, sv[u].x, rv[u].x);
            rv[u].y = fma(-a, sv[u].y, rv[u].y);
            r[j + u * stride] = rv[u];
            acc = fma((double)rv[u].x, (double)rv[u].x, acc);
            acc = fma((double)rv[u].y, (double)rv[u].y, acc);
        }
    }
    for (; j < n; j += stride) {
        V2<T> rv = r[j];
        const V2<T> sv = s[j];
        rv.x = fma(-a, sv.x, rv.x);
        rv.y = fma(-a, sv.y, rv.y);
        r[j] = rv;
        acc = fma((double)rv.x, (double)rv.x, acc);
        acc = fma((double)rv.y, (double)rv.y, acc);
    }
    const double bsum = block_sum<CG_BLOCK>(acc, red);
    if (publish_partial<CG_BLOCK>(bsum, partials, &st->ticket[2], &last_flag)) {
        const double rr = final_sum<CG_BLOCK>(partials, gridDim.x, red);
        if (threadIdx.x == 0) {
            st->ticket[2] = 0;
            cg_scalars_after_rr(st, rr);
        }
    }
}

// K4: x_i += a_i p_i ; p_i = zeta_new_i r + b_i p_i   for the shifts on this iteration's list
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_update_xp_kernel(const V2<T>* __restrict__ r, const CgState* st, size_t n) {
    if (st->stop4) return;
    __shared__ V2<T>* sx[LQCD_MAX_SHIFTS];
    __shared__ V2<T>* sp[LQCD_MAX_SHIFTS];
    __shared__ T sa[LQCD_MAX_SHIFTS], sz[LQCD_MAX_SHIFTS], sb[LQCD_MAX_SHIFTS];
    const int nl = st->nlist;
    for (int e = threadIdx.x; e < nl; e += CG_BLOCK) {
        const int i = st->list_idx[e];
        sx[e] = (V2<T>*)st->x[i];
        sp[e] = (V2<T>*)st->p[i];
        sa[e] = (T)st->list_a[e];
        sz[e] = (T)st->list_zn[e];
        sb[e] = (T)st->list_b[e];
    }
    __syncthreads();
    const size_t stride = (size_t)gridDim.x * CG_BLOCK;
    for (size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x; j < n; j += stride) {
        const V2<T> rv = r[j];
        int e = 0;
        for (; e + 4 <= nl; e += 4) {
            V2<T> xv[4], pv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                xv[u] = sx[e + u][j];
                pv[u] = sp[e + u][j];
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const T a = sa[e + u], zn = sz[e + u], bi = sb[e + u];
                xv[u].x = fma(a, pv[u].x, xv[u].x);
                xv[u].y = fma(a, pv[u].y, xv[u].y);
                pv[u].x = fma(zn, rv.x, bi * pv[u].x);
                pv[u].y = fma(zn, rv.y, bi * pv[u].y);
                sx[e + u][j] = xv[u];
                sp[e + u][j] = pv[u];
            }
        }
        for (; e < nl; ++e) {
            V2<T> xv = sx[e][j], pv = sp[e][j];
            const T a = sa[e], zn = sz[e], bi = sb[e];
            xv.x = fma(a, pv.x, xv.x);
            xv.y = fma(a, pv.y, xv.y);
            pv.x = fma(zn, rv.x, bi * pv.x);
            pv.y = fma(zn, rv.y, bi * pv.y);
            sx[e][j] = xv;
            sp[e][j] = pv;
        }
    }
}

// K4 of lqcd_rational_apply: y += sum_i (alpha_i a_i) p_i ; p_i = zeta_new_i r + b_i p_i.  The x_i are never
// stored: 96 B per site and active shift instead of 192 (the sum is taken in list order, per element).
template <typename T>
__global__ void __launch_bounds__(CG_BLOCK) cg_update_yp_kernel(const V2<T>* __restrict__ r, const CgState* st, size_t n) {
    if (st->stop4) return;
    __shared__ V2<T>* sp[LQCD_MAX_SHIFTS];
    __shared__ T sa[LQCD_MAX_SHIFTS], sz[LQCD_MAX_SHIFTS], sb[LQCD_MAX_SHIFTS];
    const int nl = st->nlist;
    for (int e = threadIdx.x; e < nl; e += CG_BLOCK) {
        sp[e] = (V2<T>*)st->p[st->list_idx[e]];
        sa[e] = (T)st->list_a[e];
        sz[e] = (T)st->list_zn[e];
        sb[e] = (T)st->list_b[e];
    }
    __syncthreads();
    V2<T>* __restrict__ y = (V2<T>*)st->y;
    const size_t stride = (size_t)gridDim.x * CG_BLOCK;
    for (size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x; j < n; j += stride) {
        const V2<T> rv = r[j];
        V2<T> yv = y[j];
        int e = 0;
        for (; e + 4 <= nl; e += 4) {
            V2<T> pv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) pv[u] = sp[e + u][j];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const T a = sa[e + u], zn = sz[e + u], bi = sb[e + u];
                yv.x = fma(a, pv[u].x, yv.x);
                yv.y = fma(a, pv[u].y, yv.y);
                pv[u].x = fma(zn, rv.x, bi * pv[u].x);
                pv[u].y = fma(zn, rv.y, bi * pv[u].y);
                sp[e + u][j] = pv[u];
            }
        }
        for (; e < nl; ++e) {
            V2<T> pv = sp[e][j];
            const T a = sa[e], zn = sz[e], bi = sb[e];
            yv.x = fma(a, pv.x, yv.x);
            yv.y = fma(a, pv.y, yv.y);
            pv.x = fma(zn, rv.x, bi * pv.x);
            pv.y = fma(zn, rv.y, bi * pv.y);
            sp[e][j] = pv;
        }
        y[j] = yv;
    }
}

// ---- layout kernels (step A1 and the pack/unpack convenience calls) -------------------------------

__device__ __forceinline__ size_t lex_of(const Geom& g, int k, int par) {
    const unsigned int r1 = fastdiv((unsigned)k, g.dxh);
    const unsigned int r2 = fastdiv(r1, g.dy);
    const int y = (int)r1 - (int)r2 * g.Ly;
    const int t = (int)fastdiv(r2, g.dz);
    const int z = (int)r2 - t * g.Lz;
    const int q = (y + z + t + par) & 1;
    return (size_t)2 * k + q;
}

__device__ __forceinline__ void atomic_max_nonneg(double* addr, double v) {
    // v >= 0: IEEE order equals unsigned integer order
    atomicMax((unsigned long long*)addr, (unsigned long long)__double_as_longlong(v));
}

// canonical links[mu][lex][3][3] -> W[((mu*2+par)*NE + e)*Vh + k]; one thread per (mu, par, k).
// With RECON=12 also records max |r2 - conj(r0 x r1)| over all links.
// The input is always the double-precision canonical field; T is the precision it is stored in.
template <typename T, int RECON>
__global__ void __launch_bounds__(256) repack_gauge_kernel(Geom g, const double2* __restrict__ links, V2<T>* __restrict__ W,
                                                           double* __restrict__ dev_max) {
    constexpr int NE = (RECON == 12) ? 6 : 9;
    const size_t vh = (size_t)g.Vh;
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= 8 * vh) return;
    const int k = (int)(idx % vh);
    const int mp = (int)(idx / vh);          // mu*2 + par
    const int mu = mp >> 1, par = mp & 1;
    const size_t lex = lex_of(g, k, par);
    const double2* __restrict__ src = links + ((size_t)mu * 2 * vh + lex) * 9;
    double2 u[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) u[e] = src[e];
#pragma unroll
    for (int e = 0; e < NE; ++e) W[((size_t)mp * NE + e) * vh + k] = make_v2((T)u[e].x, (T)u[e].y);
    if (RECON == 12) {
        double dev = 0.0;
        const int ia[3] = {1, 2, 0}, ib[3] = {2, 0, 1};
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double2 a0 = u[ia[c]], b1 = u[3 + ib[c]], a1 = u[ib[c]], b0 = u[3 + ia[c]];
            const double re = (a0.x * b1.x - a0.y * b1.y) - (a1.x * b0.x - a1.y * b0.y);
            const double im = (a0.x * b1.y + a0.y * b1.x) - (a1.x * b0.y + a1.y * b0.x);
            dev = fmax(dev, fmax(fabs(u[6 + c].x - re), fabs(u[6 + c].y + im)));
        }
        dev = fmax(dev, 0.0);
        if (!(dev == dev)) dev = 1e300;       // NaN in the input counts as "not SU(3)"
        // one atomic per warp
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
        if ((threadIdx.x & 31) == 0) atomic_max_nonneg(dev_max, dev);
    }
}

// canonical U(1) angles theta[mu][lex] -> Th[(mu*2+par)*Vh + k] (theta is what is stored)
template <typename T>
__global__ void __launch_bounds__(256) repack_theta_kernel(Geom g, const double* __restrict__ theta, T* __restrict__ Th) {
    const size_t vh = (size_t)g.Vh;
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= 8 * vh) return;
    const int k = (int)(idx % vh);
    const int mp = (int)(idx / vh);          // mu*2 + par
    Th[idx] = (T)theta[(size_t)(mp >> 1) * 2 * vh + lex_of(g, k, mp & 1)];
}

// site field [lex][3] <-> parity vector [c][k]
template <typename T>
__global__ void __launch_bounds__(256) pack_vector_kernel(Geom g, int par, const V2<T>* __restrict__ site, V2<T>* __restrict__ pv) {
    const int k = blockIdx.x * 256 + threadIdx.x;
    if (k >= g.Vh) return;
    const size_t lex = lex_of(g, k, par);
#pragma unroll
    for (int c = 0; c < 3; ++c) pv[(size_t)c * g.Vh + k] = site[lex * 3 + c];
}
template <typename T>
__global__ void __launch_bounds__(256) unpack_vector_kernel(Geom g, int par, const V2<T>* __restrict__ pv, V2<T>* __restrict__ site) {
    const int k = blockIdx.x * 256 + threadIdx.x;
    if (k >= g.Vh) return;
    const size_t lex = lex_of(g, k, par);
#pragma unroll
    for (int c = 0; c < 3; ++c) site[lex * 3 + c] = pv[(size_t)c * g.Vh + k];
}

// precision conversion of a parity vector (n complex numbers)
template <typename TO, typename FROM>
__global__ void __launch_bounds__(256) convert_vector_kernel(const V2<FROM>* __restrict__ in, V2<TO>* __restrict__ out, size_t n) {
    for (size_t j = (size_t)blockIdx.x * 256 + threadIdx.x; j < n; j += (size_t)gridDim.x * 256) {
        const V2<FROM> v = in[j];
        out[j] = make_v2((TO)v.x, (TO)v.y);
    }
}

#endif
