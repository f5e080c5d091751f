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
// EPI = 0 : out = D in
// EPI = 1 : out = coef*pv - D in, plus the block partial of Re<pv, out> and the CG scalar step
//           (this is the paper's separate zaxpy kernel, fused into the D_eo epilogue)
// EPI = 2 : out = coef*pv - D in only
// EPI = 3 : as 1, but only the block partial is written (at partials[part_off + blockIdx.x]); the sum over
//           blocks, launches and ranks and the scalar step follow in their own small kernels (slab mode)
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
#ifndef EPI_PLOAD
#define EPI_PLOAD 1      // 0: load p in the epilogue, 1: load p into registers up front, 2: L2 prefetch up front
#endif

__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
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

template <typename T>
__device__ __forceinline__ void load_vec(const V2<T>* __restrict__ v, const size_t vh, uint64_t pol, unsigned int mask,
                                         T (&vr)[3], T (&vi)[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const V2<T> t = ld_reuse(v + c * vh, pol);
        vr[c] = flip(t.x, mask);
        vi[c] = flip(t.y, mask);
    }
}

// acc += sign * U v          (forward hop; the sign is already folded into v)
template <typename T, int RECON, int U1>
__device__ __forceinline__ void hop_fwd(T (&ar)[3], T (&ai)[3], const V2<T>* __restrict__ w,
                                        const V2<T>* __restrict__ v, const size_t vh, unsigned int mask,
                                        uint64_t pol_s, uint64_t pol_r, const T* __restrict__ th) {
    V2<T> u[9];
    T vr[3], vi[3];
    load_link<T, RECON>(w, vh, pol_s, u);
    load_vec<T>(v, vh, pol_r, mask, vr, vi);
    if (U1) u1_rotate<T, +1>(th, pol_s, vr, vi);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) cmad<T>(ar[a], ai[a], u[3 * a + b], vr[b], vi[b]);
}

// acc += sign * U^dagger v   (backward hop; caller passes the mask of -s)
template <typename T, int RECON, int U1>
__device__ __forceinline__ void hop_bwd(T (&ar)[3], T (&ai)[3], const V2<T>* __restrict__ w,
                                        const V2<T>* __restrict__ v, const size_t vh, unsigned int mask,
                                        uint64_t pol_s, uint64_t pol_r, const T* __restrict__ th) {
    V2<T> u[9];
    T vr[3], vi[3];
    load_link<T, RECON>(w, vh, pol_s, u);
    load_vec<T>(v, vh, pol_r, mask, vr, vi);
    if (U1) u1_rotate<T, -1>(th, pol_s, vr, vi);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) cmad_conj<T>(ar[a], ai[a], u[3 * b + a], vr[b], vi[b]);
}

// the same two hops with separate element strides for the link and the vector (slab faces: halo buffers)
template <typename T, int RECON, int U1>
__device__ __forceinline__ void hop_fwd_s(T (&ar)[3], T (&ai)[3], const V2<T>* __restrict__ w, const size_t ws,
                                          const V2<T>* __restrict__ v, const size_t vs, unsigned int mask,
                                          uint64_t pol_s, uint64_t pol_r, const T* __restrict__ th) {
    V2<T> u[9];
    T vr[3], vi[3];
    load_link<T, RECON>(w, ws, pol_s, u);
    load_vec<T>(v, vs, pol_r, mask, vr, vi);
    if (U1) u1_rotate<T, +1>(th, pol_s, vr, vi);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) cmad<T>(ar[a], ai[a], u[3 * a + b], vr[b], vi[b]);
}
template <typename T, int RECON, int U1>
__device__ __forceinline__ void hop_bwd_s(T (&ar)[3], T (&ai)[3], const V2<T>* __restrict__ w, const size_t ws,
                                          const V2<T>* __restrict__ v, const size_t vs, unsigned int mask,
                                          uint64_t pol_s, uint64_t pol_r, const T* __restrict__ th) {
    V2<T> u[9];
    T vr[3], vi[3];
    load_link<T, RECON>(w, ws, pol_s, u);
    load_vec<T>(v, vs, pol_r, mask, vr, vi);
    if (U1) u1_rotate<T, -1>(th, pol_s, vr, vi);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) cmad_conj<T>(ar[a], ai[a], u[3 * b + a], vr[b], vi[b]);
}

template <typename T>
struct DslashArgs {
    Geom g;
    const V2<T>* W;          // stored links
    const T* Th;             // U1 == 1: stored U(1) angles theta_mu(x)
    const V2<T>* in;         // parity 1-par
    V2<T>* out;              // parity par
    int par;                 // parity of the output sites
    const V2<T>* pv;         // EPI >= 1: vector of parity par
    double coef;             // EPI >= 1: m^2 + sigma
    double* partials;        // EPI == 1
    CgState* st;             // EPI == 1, or any EPI with check_stop
    int check_stop;          // 1: return at once if st->stop (CG already converged)
    // SLAB == 1 only
    const V2<T>* in_lo;      // halo: time slice t_off-1 of `in`, [c][face]
    const V2<T>* in_hi;      // halo: time slice t_off+Lt of `in`, [c][face]
    const V2<T>* Wt_lo;      // halo: t-links leaving slice t_off-1, [parity of origin][e][face]
    const T* Th_lo;          // halo (U1): their U(1) angles, [parity of origin][face]
    int k0a, na, k0b, nsites;    // thread idx < na: site k0a+idx; else site k0b+(idx-na); nsites in all
    int part_off;            // EPI == 3: first slot of this launch in `partials`
};

// registers: double needs ~126 (4 blocks of 128 threads per SM); single fits 6 blocks
template <typename T> struct DsOcc { static constexpr int minb = DS_MINB; };
template <> struct DsOcc<float> { static constexpr int minb = DS_MINB_F32; };

template <typename T, int RECON, int EPI, int U1, int SLAB = 0>
__global__ void __launch_bounds__(DS_BLOCK, DsOcc<T>::minb) dslash_kernel(const DslashArgs<T> A) {
    constexpr int NE = (RECON == 12) ? 6 : 9;
    if (A.check_stop) {
        if (A.st->stop) {
            // tell the x/p update kernel of the *following* iterations to do nothing (see cg.cuh)
            if (EPI == 0 && blockIdx.x == 0 && threadIdx.x == 0) A.st->stop4 = 1;
            return;
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

    // step A3: coordinates, neighbours, phases
    const unsigned int r1 = fastdiv((unsigned)k, g.dxh);
    const int xh = k - (int)r1 * g.Lxh;
    const unsigned int r2 = fastdiv(r1, g.dy);
    const int y = (int)r1 - (int)r2 * g.Ly;
    const int t = (int)fastdiv(r2, g.dz);
    const int z = (int)r2 - t * g.Lz;
    const int q = (y + z + t + A.par) & 1;
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

    const uint64_t pol_s = l2_policy_evict_first();
    const uint64_t pol_r = l2_policy_evict_last();

    const V2<T>* __restrict__ Wf = A.W + (size_t)A.par * NE * vh + k;            // links of the output parity
    const V2<T>* __restrict__ Wb = A.W + (size_t)(1 - A.par) * NE * vh;          // links of the input parity
    const size_t mu_stride = (size_t)2 * NE * vh;
    const V2<T>* __restrict__ in = A.in;

    // epilogue operands are requested first, so that their latency hides behind the eight hops
    T coef = (T)0;
    V2<T> pv[3];
    if (EPI != 0) {
        coef = (T)((EPI == 1 || EPI == 3) ? A.st->c0 : A.coef);     // CG: m^2 + sigma0 from the device state (graph-invariant)
#if EPI_PLOAD == 1
#pragma unroll
        for (int c = 0; c < 3; ++c) pv[c] = A.pv[c * vh + k];
#elif EPI_PLOAD == 2
#pragma unroll
        for (int c = 0; c < 3; ++c) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.pv + c * vh + k));
#endif
    }

    T ar[3] = {(T)0, (T)0, (T)0}, ai[3] = {(T)0, (T)0, (T)0};
    const T* __restrict__ Tf = U1 ? A.Th + (size_t)A.par * vh + k : nullptr;     // angles of the forward links
    const T* __restrict__ Tb = U1 ? A.Th + (size_t)(1 - A.par) * vh : nullptr;   // angles of the backward links
    const size_t th_stride = 2 * vh;
    hop_fwd<T, RECON, U1>(ar, ai, Wf + 0 * mu_stride, in + kxf, vh, 0u, pol_s, pol_r, Tf + 0 * th_stride);
    hop_bwd<T, RECON, U1>(ar, ai, Wb + 0 * mu_stride + kxb, in + kxb, vh, SB, pol_s, pol_r, Tb + 0 * th_stride + kxb);
    hop_fwd<T, RECON, U1>(ar, ai, Wf + 1 * mu_stride, in + kyf, vh, my, pol_s, pol_r, Tf + 1 * th_stride);
    hop_bwd<T, RECON, U1>(ar, ai, Wb + 1 * mu_stride + kyb, in + kyb, vh, my ^ SB, pol_s, pol_r, Tb + 1 * th_stride + kyb);
    hop_fwd<T, RECON, U1>(ar, ai, Wf + 2 * mu_stride, in + kzf, vh, mz, pol_s, pol_r, Tf + 2 * th_stride);
    hop_bwd<T, RECON, U1>(ar, ai, Wb + 2 * mu_stride + kzb, in + kzb, vh, mz ^ SB, pol_s, pol_r, Tb + 2 * th_stride + kzb);
    if (!SLAB) {
        hop_fwd<T, RECON, U1>(ar, ai, Wf + 3 * mu_stride, in + ktf, vh, mtf, pol_s, pol_r, Tf + 3 * th_stride);
        hop_bwd<T, RECON, U1>(ar, ai, Wb + 3 * mu_stride + ktb, in + ktb, vh, mtb ^ SB, pol_s, pol_r, Tb + 3 * th_stride + ktb);
    } else {
        // across the slab faces the neighbour vector (and, downwards, the link) comes from the halo buffers
        const size_t face = (size_t)g.st;
        const int kf = k - t * g.st;                                  // index inside a time slice
        const bool top = (t == g.Lt - 1), bot = (t == 0);
        const V2<T>* vf = top ? A.in_hi + kf : in + k + g.st;
        hop_fwd_s<T, RECON, U1>(ar, ai, Wf + 3 * mu_stride, vh, vf, top ? face : vh, mtf, pol_s, pol_r, Tf + 3 * th_stride);
        const V2<T>* vb = bot ? A.in_lo + kf : in + k - g.st;
        const V2<T>* wb = bot ? A.Wt_lo + (size_t)(1 - A.par) * NE * face + kf : Wb + 3 * mu_stride + k - g.st;
        const T* tb = U1 ? (bot ? A.Th_lo + (size_t)(1 - A.par) * face + kf : Tb + 3 * th_stride + k - g.st) : nullptr;
        hop_bwd_s<T, RECON, U1>(ar, ai, wb, bot ? face : vh, vb, bot ? face : vh, mtb ^ SB, pol_s, pol_r, tb);
    }

    if (EPI == 0) {
        if (valid) {
#pragma unroll
            for (int c = 0; c < 3; ++c) A.out[c * vh + k] = make_v2((T)0.5 * ar[c], (T)0.5 * ai[c]);
        }
        return;
    }

    // epilogue: out = coef*pv - D in;  Re<pv, out> (summed in double whatever T is)
    double dot = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#if EPI_PLOAD == 1
        const V2<T> p = pv[c];
#else
        const V2<T> p = A.pv[c * vh + k];
#endif
        const V2<T> o = make_v2(fma((T)-0.5, ar[c], coef * p.x), fma((T)-0.5, ai[c], coef * p.y));
        if (valid) {
            A.out[c * vh + k] = o;
            dot = fma((double)p.x, (double)o.x, dot);
            dot = fma((double)p.y, (double)o.y, dot);
        }
    }
    if (EPI == 3) {
        __shared__ double red3[32];
        const double bsum = block_sum<DS_BLOCK>(dot, red3);
        if (threadIdx.x == 0) A.partials[A.part_off + blockIdx.x] = bsum;
    }
    if (EPI == 1) {
        __shared__ double red[32];
        __shared__ int last_flag;
        const double bsum = block_sum<DS_BLOCK>(dot, red);
        if (publish_partial<DS_BLOCK>(bsum, A.partials, &A.st->ticket[1], &last_flag)) {
            const double pAp = broadcast0(final_sum<DS_BLOCK>(A.partials, gridDim.x, red), red);
            if (threadIdx.x == 0) A.st->ticket[1] = 0;
            cg_scalars_after_pAp(A.st, pAp);
        }
    }
}

#endif
