// dslash.cuh -- the even/odd staggered Dirac operator on sm_100a (steps A2-A5 of DESIGN.md).
//
//   out(x) = 1/2 sum_mu [ s_mu(x) U_mu(x) in(x+mu) - s_mu(x-mu) U_mu(x-mu)^+ in(x-mu) ]
//
// One thread per output site, in double or single precision (template parameter T).
// All traffic is one complex number per thread and instruction (128-bit double2 / 64-bit float2) and
// unit-stride in the site index k:
//   links   W[((mu*2 + parity_of_origin)*NE + e)*Vh + k],  e = 3*row+col, NE = 9 (18-real) or 6 (12-real)
//   vectors v[c*Vh + k]
// Neighbour indices, staggered phases eta_mu and the antiperiodic sign are computed in registers from
// k (no tables: they would add 32 B/site); signs are applied by flipping the IEEE sign bit on the
// integer pipe, so the FP64 pipe only sees the 8 x 9 complex multiply-adds.
// Links are streamed once (L1 no-allocate, L2 evict-first policy); neighbour vectors are re-used 8 times
// across sites and are kept in L1/L2 (evict-last policy).
//
// U1 = 1 : every hop also carries the general U(1) factor u_mu(x) = exp(i theta_mu(x)) (imaginary chemical
//          potential, background fields).  As in the paper theta is what is stored and read
//          (8 B per link in double instead of 16 for u) and cos/sin are recomputed in registers: the kernel is
//          HBM-bound, the FP pipes have room.  Th[(mu*2 + parity_of_origin)*Vh + k].
//
// SLAB = 1 : the lattice is one slab [t_off, t_off + Lt) of a lattice cut along t over several GPUs (the paper's
//          1-D decomposition).  The input vector's time slices t_off-1 and t_off+Lt live in
//          two halo buffers filled by the neighbour ranks (layout [c][face], face = Lxh*Ly*Lz), and the t-links
//          that leave the slice below the slab in a third one (filled once, at lqcd_set_gauge).  The launch covers
//          one or two ranges of sites, so that the interior (t = 1..Lt-2, no halo needed) runs while the faces
//          are in flight and the two border slices afterwards (Alg. 1).
//
// SLAB = 2 : the interior launch of a slab: the same site range and global time coordinate as SLAB = 1, but no hop
//          crosses a face, so the hops are those of the whole-lattice kernel (no halo pointers, no runtime strides).
//
// EPI = 0 : out = D in
// EPI = 2 : out = coef*pv - D in  (the paper's separate zaxpy kernel, fused into the D_eo epilogue)
//
// The two launches of one fused CG iteration (cg.cuh has the whole picture; "scalar products and sums"
// + the two operators, with every sum and scalar product folded into the operators' own sweeps):
// EPI = 4 : K1.  The input is not a stored vector: it is the search direction p = r + beta p_old formed in
//           registers at each of the eight neighbours from the residual `in` and the previous direction `in2`.
//           out = D p (odd sites), and the block partial of  <p, A p> = c0 |p|^2 + |D_oe p|^2  (D_eo = -D_oe^+,
//           PAPER.md:L80): |out|^2 of the site plus c0/8 |p|^2 of each neighbour (every even site is the
//           neighbour of exactly eight odd sites).  cg_reduce_scalar_kernel sums and runs the scalar step (a, zeta_i).
// EPI = 5 : K2.  in = t = D_oe p.  At its own (even) site the thread forms p = r + beta p_old again and stores
//           it (p_out), s = c0 p - D_eo t (never stored), r_new = r - a s (r_out, the next ring slot),
//           x_0 += a p (unless the base system is block-deferred like the shifted ones), and the block partial of
//           |r_new|^2.  cg_reduce_scalar_kernel sums and runs the scalar step (beta, b_i, freeze and stop flags).
// With SLAB = 1 a sweep is two launches (interior, borders) that write their partials at partials[part_off + blockIdx.x];
// the sum over blocks, launches and ranks and the scalar step follow in their own small kernels, and across the slab
// faces K1 finds p itself in the halo (formed by its owner, slab_pack_p_kernel).
#ifndef LQCD_DSLASH_CUH
#define LQCD_DSLASH_CUH

#include "lqcd_internal.cuh"
#include "reduce.cuh"

#ifndef DS_BLOCK
#define DS_BLOCK 128
#endif
#ifndef DS_MINB
#define DS_MINB 4
#endif
#ifndef DS_MINB_F32
#define DS_MINB_F32 6
#endif
static_assert(DS_BLOCK >= LQCD_MAX_SHIFTS, "the scalar step of the epilogue needs one thread per shift");

__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_normal() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// 0: evict_first, 1: evict_normal, 2: evict_last
__device__ __forceinline__ uint64_t l2_policy(int code);
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

__device__ __forceinline__ uint64_t l2_policy(int code) {
    return code == 0 ? l2_policy_evict_first() : (code == 1 ? l2_policy_evict_normal() : l2_policy_evict_last());
}

// streamed once: bypass L1 allocation, first to leave L2
__device__ __forceinline__ double2 ld_stream(const double2* p, uint64_t pol) {
    double2 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;"
        : "=d"(v.x), "=d"(v.y)
        : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_stream(const float2* p, uint64_t pol) {
    float2 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;"
        : "=f"(v.x), "=f"(v.y)
        : "l"(p), "l"(pol));
    return v;
}
// re-used by neighbouring sites: allocate in L1, last to leave L2
__device__ __forceinline__ double2 ld_reuse(const double2* p, uint64_t pol) {
    double2 v;
    asm("ld.global.nc.L1::evict_last.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;"
        : "=d"(v.x), "=d"(v.y)
        : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_reuse(const float2* p, uint64_t pol) {
    float2 v;
    asm("ld.global.nc.L1::evict_last.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;"
        : "=f"(v.x), "=f"(v.y)
        : "l"(p), "l"(pol));
    return v;
}

// The same without .nc, for vectors that other blocks of the SAME kernel write between grid-wide barriers (the
// persistent solver): .nc data must be read-only for the lifetime of the kernel, an ordinary load is ordered by
// the barrier's fence.
__device__ __forceinline__ double2 ld_reuse_coherent(const double2* p, uint64_t pol) {
    double2 v;
    asm volatile("ld.global.L1::evict_last.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;"
                 : "=d"(v.x), "=d"(v.y)
                 : "l"(p), "l"(pol)
                 : "memory");
    return v;
}
__device__ __forceinline__ float2 ld_reuse_coherent(const float2* p, uint64_t pol) {
    float2 v;
    asm volatile("ld.global.L1::evict_last.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;"
                 : "=f"(v.x), "=f"(v.y)
                 : "l"(p), "l"(pol)
                 : "memory");
    return v;
}
template <bool COH, typename V>
__device__ __forceinline__ V ld_vec(const V* p, uint64_t pol) {
    return COH ? ld_reuse_coherent(p, pol) : ld_reuse(p, pol);
}

// x -> +-x by flipping the sign bit (mask is 0 or 0x80000000); integer pipe, not the FP pipe
__device__ __forceinline__ double flip(double x, unsigned int mask) {
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}
__device__ __forceinline__ float flip(float x, unsigned int mask) {
    return __int_as_float(__float_as_int(x) ^ (int)mask);
}

// acc += u * v
template <typename T>
__device__ __forceinline__ void cmad(T& ar, T& ai, const V2<T> u, const T vr, const T vi) {
    ar = fma(u.x, vr, ar);
    ar = fma(-u.y, vi, ar);
    ai = fma(u.x, vi, ai);
    ai = fma(u.y, vr, ai);
}
// acc += conj(u) * v
template <typename T>
__device__ __forceinline__ void cmad_conj(T& ar, T& ai, const V2<T> u, const T vr, const T vi) {
    ar = fma(u.x, vr, ar);
    ar = fma(u.y, vi, ar);
    ai = fma(u.x, vi, ai);
    ai = fma(-u.y, vr, ai);
}

template <typename V>
__device__ __forceinline__ V cmul(const V a, const V b) {
    return make_v2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// streamed scalar (the U(1) angle of one link)
__device__ __forceinline__ double ld_stream_scalar(const double* p, uint64_t pol) {
    double v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float ld_stream_scalar(const float* p, uint64_t pol) {
    float v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ void sincos_t(double th, double* s, double* c) { sincos(th, s, c); }
__device__ __forceinline__ void sincos_t(float th, float* s, float* c) { sincosf(th, s, c); }

// v <- exp(+-i theta) v  (sgn = +1: forward hop, u; sgn = -1: backward hop, conj(u))
template <typename T, int SGN>
__device__ __forceinline__ void u1_rotate(const T* __restrict__ th, uint64_t pol, T (&vr)[3], T (&vi)[3]) {
    T s, c;
    sincos_t(ld_stream_scalar(th, pol), &s, &c);
    if (SGN < 0) s = -s;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const T re = fma(c, vr[a], -(s * vi[a]));
        const T im = fma(c, vi[a], s * vr[a]);
        vr[a] = re;
        vi[a] = im;
    }
}

// Load one link (9 complex).  12-real storage: rows 0,1 are read, r2 = conj(r0 x r1).
template <typename T, int RECON>
__device__ __forceinline__ void load_link(const V2<T>* __restrict__ w, const size_t vh, uint64_t pol, V2<T> (&u)[9]) {
    constexpr int NE = (RECON == 12) ? 6 : 9;
#pragma unroll
    for (int e = 0; e < NE; ++e) u[e] = ld_stream(w + e * vh, pol);
    if (RECON == 12) {
        V2<T> c;
        c = cmul(u[1], u[5]); { const V2<T> d = cmul(u[2], u[4]); u[6] = make_v2(c.x - d.x, -(c.y - d.y)); }
        c = cmul(u[2], u[3]); { const V2<T> d = cmul(u[0], u[5]); u[7] = make_v2(c.x - d.x, -(c.y - d.y)); }
        c = cmul(u[0], u[4]); { const V2<T> d = cmul(u[1], u[3]); u[8] = make_v2(c.x - d.x, -(c.y - d.y)); }
    }
}

// the vector operand of a hop.  MODE 0: a stored vector.  MODE 1: p = r + beta p_old formed in registers from the
// residual v and the previous search direction v2 (same index); pp accumulates |p|^2 for the <p,Ap> identity of
// EPI = 4.  MODE 2: p was formed by the rank that owns the site and arrived in a halo buffer (slab faces of
// EPI = 4): a stored vector whose |p|^2 is accumulated all the same.
template <typename T, int MODE, bool COH>
__device__ __forceinline__ void load_vec(const V2<T>* __restrict__ v, const V2<T>* __restrict__ v2, const size_t vs,
                                         uint64_t pol, unsigned int mask, const T beta, T (&vr)[3], T (&vi)[3],
                                         double& pp) {
    if (MODE != 1) {
        T n2 = (T)0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const V2<T> t = ld_vec<COH>(v + c * vs, pol);
            if (MODE == 2) {
                n2 = fma(t.x, t.x, n2);
                n2 = fma(t.y, t.y, n2);
            }
            vr[c] = flip(t.x, mask);
            vi[c] = flip(t.y, mask);
        }
        if (MODE == 2) pp += (double)n2;
    } else {
        V2<T> r[3], q[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            r[c] = ld_vec<COH>(v + c * vs, pol);
            q[c] = ld_vec<COH>(v2 + c * vs, pol);
        }
        T n2 = (T)0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const T x = fma(beta, q[c].x, r[c].x), y = fma(beta, q[c].y, r[c].y);
            n2 = fma(x, x, n2);
            n2 = fma(y, y, n2);
            vr[c] = flip(x, mask);
            vi[c] = flip(y, mask);
        }
        pp += (double)n2;
    }
}

// One hop.  FWD: acc += sign * U v (the sign is already folded into v);  !FWD: acc += sign * U^dagger v (the caller
// passes the mask of -s).  ws, vs: element strides of the link and of the vector (they differ from Vh only for the
// halo buffers of a slab face).
template <typename T, int RECON, int U1, bool FWD, int MODE, bool COH = false>
__device__ __forceinline__ void hop(T (&ar)[3], T (&ai)[3], const V2<T>* __restrict__ w, const size_t ws,
                                    const V2<T>* __restrict__ v, const V2<T>* __restrict__ v2, const size_t vs,
                                    unsigned int mask, uint64_t pol_s, uint64_t pol_r, const T* __restrict__ th,
                                    const T beta, double& pp) {
    V2<T> u[9];
    T vr[3], vi[3];
    load_link<T, RECON>(w, ws, pol_s, u);
    load_vec<T, MODE, COH>(v, v2, vs, pol_r, mask, beta, vr, vi, pp);
    if (U1) u1_rotate<T, FWD ? +1 : -1>(th, pol_s, vr, vi);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            if (FWD) cmad<T>(ar[a], ai[a], u[3 * a + b], vr[b], vi[b]);
            else cmad_conj<T>(ar[a], ai[a], u[3 * b + a], vr[b], vi[b]);
        }
}

template <typename T>
struct DslashArgs {
    Geom g;
    const V2<T>* W;          // stored links
    const T* Th;             // U1 == 1: stored U(1) angles theta_mu(x)
    const V2<T>* in;         // parity 1-par (EPI == 4: the residual r)
    const V2<T>* in2;        // EPI == 4: the previous search direction p_old, parity 1-par
    V2<T>* out;              // parity par (not written by EPI == 5)
    int par;                 // parity of the output sites
    const V2<T>* pv;         // EPI == 2: vector of parity par;  EPI == 5: p_old
    double coef;             // EPI == 2: m^2 + sigma
    double* partials;        // EPI 4,5
    CgState* st;             // EPI 4,5, or any EPI with check_stop
    int check_stop;          // 1: return at once if st->stop (CG already converged)
    int pol_links, pol_vecs; // L2 eviction priority of the link / neighbour-vector loads (l2_policy codes)
    // EPI == 5 only (all of parity par)
    const V2<T>* r_in;       // residual r^(n)
    V2<T>* r_out;            // residual r^(n+1): the next slot of the ring (may be r_in itself)
    V2<T>* p_out;            // search direction p^(n) (may be pv itself)
    V2<T>* p_keep;           // not NULL: p^(n) is also stored here (first iteration of a block, base system deferred)
    int defer_base;          // 1: x_0 is updated by the block sweep like the shifted systems, not here
    // SLAB == 1 only
    const V2<T>* in_lo;      // halo: time slice t_off-1 of `in`, [c][face]
    const V2<T>* in_hi;      // halo: time slice t_off+Lt of `in`, [c][face]
    const V2<T>* Wt_lo;      // halo: t-links leaving slice t_off-1, [parity of origin][e][face]
    const T* Th_lo;          // halo (U1): their U(1) angles, [parity of origin][face]
    int k0a, na, k0b, nsites;    // thread idx < na: site k0a+idx; else site k0b+(idx-na); nsites in all
    int part_off;            // EPI 4,5: first slot of this launch in `partials`
    // FS == 1 only (small lattices: the scalar step rides in the next sweep instead of a launch of its own)
    const double* red_in;    // block partials of the PREVIOUS sweep (K1: those of K2, K2: those of K1), red_n of them
    int red_n;
    int pending;             // K1: 1 = the scalar step after K2 of the previous iteration has not been run yet
    unsigned int *clear0, *clear1;   // not NULL (border launch, peer-memory transport): the arrival words of the halos
                             // this launch consumes, cleared for their next use (p2p.cuh)
};

// registers: double needs ~126 (4 blocks of 128 threads per SM); single fits 6 blocks
#ifndef DS_MINB_K1
#define DS_MINB_K1 3     // K1 loads two vectors per neighbour: 168 registers (3 blocks) keep more loads in flight than 128
#endif
#ifndef DS_MINB_K2
#define DS_MINB_K2 DS_MINB
#endif
template <typename T, int EPI> struct DsOcc { static constexpr int minb = (EPI == 4) ? DS_MINB_K1 : (EPI == 5) ? DS_MINB_K2 : DS_MINB; };
template <int EPI> struct DsOcc<float, EPI> { static constexpr int minb = DS_MINB_F32; };

// The eight hops of one output site k of parity `par`: acc = sum_mu [ s U in(x+mu) - s U^+ in(x-mu) ] (without the
// factor 1/2).  FLY: the input is p = in + beta in2 formed at each neighbour, and pp accumulates its |p|^2.
// COH: the input vectors are written by other blocks of the same kernel (see ld_reuse_coherent).
template <typename T, int RECON, int U1, int SLAB, bool FLY, bool COH = false>
__device__ __forceinline__ void dslash_hops(const DslashArgs<T>& A, const int par, const int k,
                                            const V2<T>* __restrict__ in, const V2<T>* __restrict__ in2, const T beta,
                                            T (&ar)[3], T (&ai)[3], double& pp) {
    constexpr int NE = (RECON == 12) ? 6 : 9;
    const Geom& g = A.g;
    const size_t vh = (size_t)g.Vh;

    // step A3: coordinates, neighbours, phases
    const unsigned int r1 = fastdiv((unsigned)k, g.dxh);
    const int xh = k - (int)r1 * g.Lxh;
    const unsigned int r2 = fastdiv(r1, g.dy);
    const int y = (int)r1 - (int)r2 * g.Ly;
    const int t = (int)fastdiv(r2, g.dz);
    const int z = (int)r2 - t * g.Lz;
    const int q = (y + z + t + par) & 1;
    const int x = 2 * xh + q;

    const int kxf = k + (q ? ((xh == g.Lxh - 1) ? 1 - g.Lxh : 1) : 0);
    const int kxb = k - (q ? 0 : ((xh == 0) ? 1 - g.Lxh : 1));
    const int kyf = k + ((y == g.Ly - 1) ? -(g.Ly - 1) * g.sy : g.sy);
    const int kyb = k + ((y == 0) ? (g.Ly - 1) * g.sy : -g.sy);
    const int kzf = k + ((z == g.Lz - 1) ? -(g.Lz - 1) * g.sz : g.sz);
    const int kzb = k + ((z == 0) ? (g.Lz - 1) * g.sz : -g.sz);
    const int ktf = k + ((t == g.Lt - 1) ? -(g.Lt - 1) * g.st : g.st);
    const int ktb = k + ((t == 0) ? (g.Lt - 1) * g.st : -g.st);

    const unsigned int SB = 0x80000000u;
    const unsigned int my = (unsigned)(x & 1) << 31;                    // eta_y = (-1)^x
    const unsigned int mz = (unsigned)((x + y) & 1) << 31;              // eta_z = (-1)^(x+y)
    const unsigned int mt = (unsigned)((x + y + z) & 1) << 31;          // eta_t = (-1)^(x+y+z)
    // the boundary sign sits on the links that leave the last time slice of the WHOLE lattice
    const int tg = SLAB ? t + g.t_off : t;
    const int Ltg = SLAB ? g.Lt_glob : g.Lt;
    const unsigned int mtf = mt ^ ((g.antiperiodic && tg == Ltg - 1) ? SB : 0u);   // link (x,t) leaves Lt-1
    const unsigned int mtb = mt ^ ((g.antiperiodic && tg == 0) ? SB : 0u);         // link (x-t,t) leaves Lt-1

    // links: streamed once per application -- first to leave L2; unless the whole gauge field fits in L2 beside the
    // vectors (small lattices), where it is what should stay for the next application
    const uint64_t pol_r = l2_policy(A.pol_vecs);
    const uint64_t pol_s = l2_policy(A.pol_links);

    const V2<T>* __restrict__ Wf = A.W + (size_t)par * NE * vh + k;              // links of the output parity
    const V2<T>* __restrict__ Wb = A.W + (size_t)(1 - par) * NE * vh;            // links of the input parity
    const size_t mu_stride = (size_t)2 * NE * vh;
    const T* __restrict__ Tf = U1 ? A.Th + (size_t)par * vh + k : nullptr;       // angles of the forward links
    const T* __restrict__ Tb = U1 ? A.Th + (size_t)(1 - par) * vh : nullptr;     // angles of the backward links
    const size_t th_stride = 2 * vh;
#define HOP_F(mu, kn, mask) \
    hop<T, RECON, U1, true, FLY ? 1 : 0, COH>(ar, ai, Wf + (mu) * mu_stride, vh, in + (kn), in2 + (kn), vh, mask, pol_s, pol_r, \
                                 Tf + (mu) * th_stride, beta, pp)
#define HOP_B(mu, kn, mask) \
    hop<T, RECON, U1, false, FLY ? 1 : 0, COH>(ar, ai, Wb + (mu) * mu_stride + (kn), vh, in + (kn), in2 + (kn), vh, (mask) ^ SB, pol_s, \
                                  pol_r, Tb + (mu) * th_stride + (kn), beta, pp)
    HOP_F(0, kxf, 0u);
    HOP_B(0, kxb, 0u);
    HOP_F(1, kyf, my);
    HOP_B(1, kyb, my);
    HOP_F(2, kzf, mz);
    HOP_B(2, kzb, mz);
    if (SLAB != 1) {
        // whole lattice, or the interior launch of a slab (SLAB == 2: t = 1 .. Lt-2, no hop leaves the slab)
        HOP_F(3, ktf, mtf);
        HOP_B(3, ktb, mtb);
    } else {
        // across the slab faces the neighbour vector (and, downwards, the link) comes from the halo buffers; with
        // FLY the halo holds p itself, formed by the rank that owns those sites (slab_pack_p_kernel)
        const size_t face = (size_t)g.st;
        const int kf = k - t * g.st;                                  // index inside a time slice
        const bool top = (t == g.Lt - 1), bot = (t == 0);
        const V2<T>* wf = Wf + 3 * mu_stride;
        const T* tf = Tf + 3 * th_stride;
        const V2<T>* wb = bot ? A.Wt_lo + (size_t)(1 - par) * NE * face + kf : Wb + 3 * mu_stride + k - g.st;
        const T* tb = U1 ? (bot ? A.Th_lo + (size_t)(1 - par) * face + kf : Tb + 3 * th_stride + k - g.st) : nullptr;
        const size_t wbs = bot ? face : vh;
        if (!FLY) {
            const V2<T>* vf = top ? A.in_hi + kf : in + k + g.st;
            hop<T, RECON, U1, true, 0>(ar, ai, wf, vh, vf, vf, top ? face : vh, mtf, pol_s, pol_r, tf, beta, pp);
            const V2<T>* vb = bot ? A.in_lo + kf : in + k - g.st;
            hop<T, RECON, U1, false, 0>(ar, ai, wb, wbs, vb, vb, bot ? face : vh, mtb ^ SB, pol_s, pol_r, tb, beta, pp);
        } else {
            if (top) hop<T, RECON, U1, true, 2>(ar, ai, wf, vh, A.in_hi + kf, A.in_hi + kf, face, mtf, pol_s, pol_r, tf, beta, pp);
            else hop<T, RECON, U1, true, 1>(ar, ai, wf, vh, in + k + g.st, in2 + k + g.st, vh, mtf, pol_s, pol_r, tf, beta, pp);
            if (bot) hop<T, RECON, U1, false, 2>(ar, ai, wb, wbs, A.in_lo + kf, A.in_lo + kf, face, mtb ^ SB, pol_s, pol_r, tb, beta, pp);
            else hop<T, RECON, U1, false, 1>(ar, ai, wb, wbs, in + k - g.st, in2 + k - g.st, vh, mtb ^ SB, pol_s, pol_r, tb, beta, pp);
        }
    }
#undef HOP_F
#undef HOP_B
}

// K1 of the fused iteration, after the hops: t = D_oe p is stored; returns this site's share of
// <p, A p> = c0 |p|^2 + |t|^2 (|p|^2 of the eight neighbours, each counted 1/8)
template <typename T>
__device__ __forceinline__ double k1_finish(V2<T>* __restrict__ out, const size_t vh, const int k, const bool valid,
                                            const T (&ar)[3], const T (&ai)[3], const double pp, const double c0) {
    double dot = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const V2<T> o = make_v2((T)0.5 * ar[c], (T)0.5 * ai[c]);
        if (valid) {
            out[c * vh + k] = o;
            dot = fma((double)o.x, (double)o.x, dot);
            dot = fma((double)o.y, (double)o.y, dot);
        }
    }
    if (valid) dot = fma(0.125 * c0, pp, dot);
    return dot;
}

// What K2 needs besides the hops, the same for every site of a launch
template <typename T>
struct K2Coef {
    T beta, a, c0, ax;       // ax: coefficient of p in the update of x_0 (alpha_i0 * a in rational-sum mode)
    V2<T>* xp;               // x_0 (or y in rational-sum mode)
    V2<T>* p_out;
    V2<T>* r_out;
    V2<T>* p_keep;           // may be NULL
    int defer_base;
};

// K2 of the fused iteration, after the hops (acc = 2 D_eo t): p = r + beta p_old;  s = c0 p - D_eo t;
// r_new = r - a s;  x_0 += a p;  returns |r_new|^2 of the site
template <typename T>
__device__ __forceinline__ double k2_finish(const K2Coef<T>& C, const size_t vh, const int k, const bool valid,
                                            const V2<T> (&pold)[3], const V2<T> (&rv)[3], const T (&ar)[3],
                                            const T (&ai)[3]) {
    double dot = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const V2<T> r = rv[c];
        const V2<T> p = make_v2(fma(C.beta, pold[c].x, r.x), fma(C.beta, pold[c].y, r.y));
        const V2<T> sv = make_v2(fma((T)-0.5, ar[c], C.c0 * p.x), fma((T)-0.5, ai[c], C.c0 * p.y));
        const V2<T> rn = make_v2(fma(-C.a, sv.x, r.x), fma(-C.a, sv.y, r.y));
        if (valid) {
            C.p_out[c * vh + k] = p;
            C.r_out[c * vh + k] = rn;
            if (C.p_keep) C.p_keep[c * vh + k] = p;
            if (!C.defer_base) {
                V2<T> xv = C.xp[c * vh + k];
                xv.x = fma(C.ax, p.x, xv.x);
                xv.y = fma(C.ax, p.y, xv.y);
                C.xp[c * vh + k] = xv;
            }
            dot = fma((double)rn.x, (double)rn.x, dot);
            dot = fma((double)rn.y, (double)rn.y, dot);
        }
    }
    return dot;
}

template <typename T>
__device__ __forceinline__ K2Coef<T> k2_coef_from_state(const CgState* st, const double a, V2<T>* p_out, V2<T>* r_out,
                                                        V2<T>* p_keep, int defer_base) {
    K2Coef<T> C;
    const int rational = st->rational, i0 = st->i0;
    C.beta = (T)st->b_prev;
    C.a = (T)a;
    C.c0 = (T)st->c0;
    C.ax = (T)(rational ? st->alpha[i0] * a : a);
    C.xp = (V2<T>*)(rational ? st->y : st->x[i0]);
    C.p_out = p_out;
    C.r_out = r_out;
    C.p_keep = p_keep;
    C.defer_base = defer_base;
    return C;
}

// FS = 1 (EPI 4, 5 on small whole lattices, where a one-block kernel per scalar step is a third of the iteration): the
// launch has one block more than the sites need.  EVERY block first adds the block partials of the previous sweep in
// the same fixed order (a few hundred numbers from L2; the same bits in every block) and takes from the sum the one
// scalar it needs -- K2: a = |r|^2 / <p,Ap>;  K1: beta = |r_new|^2 / |r|^2 and the stop decision -- while the extra block
// runs the scalar step proper on the device state (zeta_i, block coefficients, freeze flags) for everybody else's
// later use.  The fields the sweeping blocks read (rr, b_prev in K2; rr_keep, iter_keep in K1) are not written by the
// scalar step that runs beside them.  `stop` IS written beside them (after K2's sum: when the solve is over; after
// K1's: on a breakdown), so a block does not let each thread read it: thread 0 reads it once and the block decides as
// one (threads that disagreed would leave some of them out of the sum below).  Blocks may still read different values;
// those that read 0 reach, from the sum, the decision the scalar step reached (the returns below).  The step after K2
// of the last iteration of a block (and of a batch) is run by cg_reduce_scalar_kernel before the block sweep; K1 of the
// next iteration is then launched with pending = 0.
template <typename T, int RECON, int EPI, int U1, int SLAB = 0, int FS = 0>
__global__ void __launch_bounds__(DS_BLOCK, (DsOcc<T, EPI>::minb)) dslash_kernel(const DslashArgs<T> A) {
    constexpr bool FLY = (EPI == 4);
    static_assert(EPI == 0 || EPI == 2 || EPI == 4 || EPI == 5, "EPI");
    static_assert(!FS || (!SLAB && (EPI == 4 || EPI == 5)), "FS");
    if (SLAB && A.clear0 && blockIdx.x == 0 && threadIdx.x == 0) {
        // peer-memory transport: the two arrival words of the halos this launch reads are cleared for their next use --
        // unless a neighbour that gave up wrote LQCD_P2P_POISON there (the halo is then not a halo): that stays, and
        // the solve ends with LQCD_ECOMM
        const unsigned int w0 = *(volatile unsigned int*)A.clear0, w1 = *(volatile unsigned int*)A.clear1;
        if (w0 != LQCD_P2P_POISON) *A.clear0 = 0u;
        if (w1 != LQCD_P2P_POISON) *A.clear1 = 0u;
        if (w0 == LQCD_P2P_POISON || w1 == LQCD_P2P_POISON) {
            A.st->status = LQCD_ECOMM_DEV;
            A.st->stop = 1;
        }
    }
    if (!FS && A.check_stop && A.st->stop) return;      // iterations launched beyond the one that converged
    double a_fs = 0.0, beta_fs = 0.0;
    if (FS) {
        __shared__ double redf[32];
        __shared__ int stop_sh;
        if (threadIdx.x == 0) stop_sh = A.check_stop ? A.st->stop : 0;
        const bool have = (EPI == 5) || A.pending;
        double sum_in = 0.0;
        if (have) sum_in = broadcast0(final_sum<DS_BLOCK>(A.red_in, A.red_n, redf), redf);   // barriers inside
        else __syncthreads();
        if (stop_sh) return;                     // iterations launched beyond the one that converged
        if (blockIdx.x == gridDim.x - 1) {       // the block that owns no sites
            if (have) {
                if (EPI == 5) cg_scalars_after_pAp(A.st, sum_in);
                else cg_scalars_after_rr(A.st, sum_in);
            }
            return;
        }
        if (EPI == 5) {
            if (!(sum_in > 0.0) || !isfinite(sum_in)) return;            // breakdown: the scalar step records it
            a_fs = A.st->rr / sum_in;
        } else if (have) {
            if (sum_in <= A.st->tol2bb || A.st->iter_keep + 1 >= A.st->max_iter) return;   // the solve is over
            beta_fs = sum_in / A.st->rr_keep;
        } else {
            beta_fs = A.st->b_prev;
        }
    }
    const Geom& g = A.g;
    const int kraw = blockIdx.x * DS_BLOCK + threadIdx.x;
    bool valid;
    int k;
    if (SLAB) {
        valid = kraw < A.nsites;
        const int i = valid ? kraw : A.nsites - 1;
        k = (i < A.na) ? A.k0a + i : A.k0b + (i - A.na);
    } else {
        valid = kraw < g.Vh;
        k = valid ? kraw : g.Vh - 1;
    }
    const size_t vh = (size_t)g.Vh;

    // epilogue operands are requested first, so that their latency hides behind the eight hops
    T coef = (T)0, beta = (T)0;
    V2<T> pv[3], rv[3];
    if (EPI != 0) {
        // CG: m^2 + sigma0 from the device state (graph-invariant)
        coef = (T)((EPI == 2) ? A.coef : A.st->c0);
        if (EPI == 4) beta = (T)(FS ? beta_fs : A.st->b_prev);
        if (EPI != 4) {
#pragma unroll
            for (int c = 0; c < 3; ++c) pv[c] = A.pv[c * vh + k];
        }
        if (EPI == 5) {
#pragma unroll
            for (int c = 0; c < 3; ++c) rv[c] = A.r_in[c * vh + k];
        }
    }

    T ar[3] = {(T)0, (T)0, (T)0}, ai[3] = {(T)0, (T)0, (T)0};
    double pp = 0.0;                            // EPI == 4: sum of |p|^2 over the neighbours
    dslash_hops<T, RECON, U1, SLAB, FLY>(A, A.par, k, A.in, FLY ? A.in2 : A.in, beta, ar, ai, pp);

    if (EPI == 0) {
        if (valid) {
#pragma unroll
            for (int c = 0; c < 3; ++c) A.out[c * vh + k] = make_v2((T)0.5 * ar[c], (T)0.5 * ai[c]);
        }
        return;
    }

    double dot = 0.0;                           // scalar products are summed in double whatever T is
    if (EPI == 4) {
        dot = k1_finish<T>(A.out, vh, k, valid, ar, ai, pp, A.st->c0);
    } else if (EPI == 5) {
        K2Coef<T> C = k2_coef_from_state<T>(A.st, FS ? a_fs : A.st->a, A.p_out, A.r_out, A.p_keep, A.defer_base);
        dot = k2_finish<T>(C, vh, k, valid, pv, rv, ar, ai);
    } else {
        // out = coef*pv - D in
        if (valid) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const V2<T> p = pv[c];
                A.out[c * vh + k] = make_v2(fma((T)-0.5, ar[c], coef * p.x), fma((T)-0.5, ai[c], coef * p.y));
            }
        }
        return;
    }
    // Only the block partial is written here; the sum over blocks (over the launches of a slab's sweep, over the ranks)
    // and the scalar step follow in one small kernel (cg_reduce_scalar_kernel; slabs: sum_partials_kernel, the
    // transport's all-reduce, cg_scalar_kernel).  Having the block that finishes last do it instead (partial, fence,
    // atomic ticket in every block) saved the launch and cost 10-12 us per sweep of 20,736 blocks.
    __shared__ double red[32];
    const double bsum = block_sum<DS_BLOCK>(dot, red);
    if (threadIdx.x == 0) A.partials[A.part_off + blockIdx.x] = bsum;
}

// Slab mode, before K1: the two faces (time slices 0 and Lt-1) of p = r + beta p_old, formed by the rank that owns the
// sites with the formula K1 uses at the neighbours (load_vec, MODE 1: same operands, same bits), packed as [c][face]
// each: into the send buffers of the ring exchange, or (peer-memory transport) straight into the neighbours' halo
// buffers over NVLink.  One thread per complex number.
template <typename T>
__global__ void __launch_bounds__(256) slab_pack_p_kernel(const V2<T>* __restrict__ r, const V2<T>* __restrict__ p_old,
                                                          V2<T>* __restrict__ send_lo, V2<T>* __restrict__ send_hi,
                                                          const CgState* st, size_t vh, size_t face) {
    if (st->stop) return;
    const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= 6 * face) return;
    const T beta = (T)st->b_prev;
    const size_t hi = i / (3 * face), rem = i - hi * 3 * face;
    const size_t c = rem / face, kf = rem - c * face;
    const size_t src = c * vh + (hi ? vh - face : 0) + kf;
    const V2<T> rv = r[src], q = p_old[src];
    (hi ? send_hi : send_lo)[rem] = make_v2(fma(beta, q.x, rv.x), fma(beta, q.y, rv.y));
}

#endif
