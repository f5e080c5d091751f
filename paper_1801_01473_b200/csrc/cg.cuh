// cg.cuh -- the vector sweeps of the multi-shift CG (steps A7, A8 of DESIGN.md) and layout kernels.
//
// One CG iteration is the two operator launches of dslash.cuh ("scalar products and sums" + the two
// operators, every sum and scalar product of the base system folded into the operators' own sweeps), plus one sweep
// over all systems every m iterations:
//   K1  t = D_oe p with p = r + beta p_old formed at the neighbours;  block partials of <p,Ap>    dslash_kernel<.,4>
//       sum -> a, zeta_new_i                                                          cg_reduce_scalar_kernel (1 block)
//   K2  p, s = (m^2+sigma0) p - D_eo t, r_new = r - a s at the own site;  block partials of |r_new|^2
//                                                                                                 dslash_kernel<.,5>
//       sum -> beta, b_i, block coefficients, freeze flags, stop flag                 cg_reduce_scalar_kernel (1 block)
//   every m-th iteration (and once after the stop), for every system of the block:
//         x_i += CP_i p_i + sum_l D_il r_l ;  p_i = B_i p_i + sum_l E_il r_l                      cg_flush_kernel
// K2 writes r_new into a ring of m residual vectors instead of over r, so that the m residuals of a block
// are still there when the sweep runs: the 192 B per site and active shift of the x_i/p_i update are paid once per
// block instead of once per iteration (CgState in lqcd_internal.cuh has the algebra).
// All scalars stay on the device.
#ifndef LQCD_CG_CUH
#define LQCD_CG_CUH

#include "lqcd_internal.cuh"
#include "reduce.cuh"

#define CG_BLOCK 256
static_assert(CG_BLOCK >= LQCD_MAX_SHIFTS, "the scalar step needs one thread per shift");

// K0: r = p = b (base system), |b|^2.  In every sweep the vectors are V2<T>; scalars and sums are double.
// r is the ring slot that holds r^(n0) of the first block.  The shifted p_i = b and the x_i = 0 are NOT written here:
// the first block sweep produces them (CgState::first_block), which saves 2 x nshift vector writes and nshift + 1
// vector reads per solve.  Only what is read before that sweep is initialised: the base p, x_0 when it is updated
// every iteration (no deferral), and y = alpha0 b in rational-sum mode.
// FUSED = false (slab mode): only the block partial is written; the sum over blocks and ranks and the scalar
// step follow in sum_partials_kernel / cg_scalar_kernel.
template <typename T, bool FUSED = true>
__global__ void __launch_bounds__(CG_BLOCK) cg_init_kernel(const V2<T>* __restrict__ b, V2<T>* __restrict__ r,
                                                           CgState* st, double* partials, size_t n, double tol) {
    __shared__ double red[32];
    __shared__ int last_flag;
    const int rational = st->rational;
    const T alpha0 = (T)st->alpha0;
    V2<T>* __restrict__ y = (V2<T>*)st->y;
    V2<T>* __restrict__ p0 = (V2<T>*)st->p[st->i0];
    V2<T>* __restrict__ x0 = (!rational && !st->defer_base) ? (V2<T>*)st->x[st->i0] : nullptr;
    double acc = 0.0;
    const V2<T> zero = make_v2((T)0, (T)0);
    for (size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x; j < n; j += (size_t)gridDim.x * CG_BLOCK) {
        const V2<T> v = b[j];
        r[j] = v;
        p0[j] = v;
        if (rational) y[j] = make_v2(alpha0 * v.x, alpha0 * v.y);
        if (x0) x0[j] = zero;
        acc = fma((double)v.x, (double)v.x, acc);
        acc = fma((double)v.y, (double)v.y, acc);
    }
    const double bsum = block_sum<CG_BLOCK>(acc, red);
    if (!FUSED) {
        if (threadIdx.x == 0) partials[blockIdx.x] = bsum;
        return;
    }
    if (publish_partial<CG_BLOCK>(bsum, partials, &st->ticket[0], &last_flag)) {
        const double bb = final_sum<CG_BLOCK>(partials, gridDim.x, red);
        if (threadIdx.x == 0) {
            st->ticket[0] = 0;
            cg_scalars_init(st, bb, tol);
        }
    }
}

// ---- slab mode (1-D decomposition along t): a scalar product is the sum over the blocks of
// this rank (sum_partials_kernel, fixed order), then over the ranks (all-reduce of one double: "global
// reductions" of PAPER.md:L112), then the scalar step runs on every rank on bit-identical input
// (cg_scalar_kernel), so that all ranks take the same decisions.
__global__ void __launch_bounds__(CG_BLOCK) sum_partials_kernel(const double* __restrict__ partials, int n,
                                                                double* __restrict__ out, const CgState* st,
                                                                int check_stop, const PeerPush* __restrict__ push) {
    __shared__ double red[32];
    // peer-memory transport (push != NULL): the rank's sum goes straight into every rank's window; when the solve is
    // over a dummy still goes, because every rank still waits for every rank's contribution
    if (check_stop && st->stop) {
        if (push) peer_push(push, 0.0);
        return;
    }
    const double v = broadcast0(final_sum<CG_BLOCK>(partials, n, red), red);
    if (threadIdx.x == 0) *out = v;
    if (push) peer_push(push, v);
}
// whole lattice: the sum of the block partials of K1 (which = 1) / K2 (which = 2) and the scalar step, one block
__global__ void __launch_bounds__(CG_BLOCK) cg_reduce_scalar_kernel(CgState* st, const double* __restrict__ partials, int n,
                                                                    int which) {
    if (st->stop) return;
    __shared__ double red[32];
    const double v = broadcast0(final_sum<CG_BLOCK>(partials, n, red), red);
    if (which == 1) cg_scalars_after_pAp(st, v);
    else cg_scalars_after_rr(st, v);
}
// which = 0: after |b|^2 ; 1: after <p,Ap> ; 2: after |r_new|^2.  One block of >= LQCD_MAX_SHIFTS threads.
__global__ void __launch_bounds__(64) cg_scalar_kernel(CgState* st, const double* __restrict__ value, int which,
                                                       double tol) {
    const double v = *value;
    if (which == 0) {
        if (threadIdx.x == 0) cg_scalars_init(st, v, tol);
        return;
    }
    if (st->stop) return;
    if (which == 1) cg_scalars_after_pAp(st, v);
    else cg_scalars_after_rr(st, v);
}

// The same after the peer-memory transport's push (p2p.cuh): the ranks' contributions sit in this rank's window,
// slots[r * stride]; they are added in rank order (same bits on every rank), their arrival flags cleared.
__global__ void __launch_bounds__(64) cg_scalar_slots_kernel(CgState* st, const double* slots, unsigned int* flags,
                                                             int nranks, int stride, int which) {
    __shared__ double sv;
    __shared__ int poisoned;
    if (threadIdx.x == 0) {
        double acc = 0.0;
        for (int r = 0; r < nranks; ++r) acc += __ldcv(slots + r * stride);
        sv = acc;
        poisoned = 0;
    }
    __syncthreads();
    // a rank that gave up left LQCD_P2P_POISON instead of 1 (p2p.cuh): its slot holds nothing; the mark stays
    if (threadIdx.x < nranks) {
        if (*(volatile unsigned int*)(flags + threadIdx.x) == LQCD_P2P_POISON) poisoned = 1;
        else flags[threadIdx.x] = 0u;
    }
    __syncthreads();
    if (poisoned) {
        if (threadIdx.x == 0) {
            st->status = LQCD_ECOMM_DEV;
            st->stop = 1;
        }
        return;
    }
    if (st->stop) return;
    if (which == 1) cg_scalars_after_pAp(st, sv);
    else cg_scalars_after_rr(st, sv);
}

// The block sweep: the deferred updates of one block, for every shifted system that was active when the block began.
// nres = st->blk_j residuals r_l = hist[l] are used (nres = m for a full block, less after the stop).
//   x_i += CP_i p_i + sum_l D_il r_l   (rational mode: y += sum_i of that; alpha_i is inside CP, D)
//   p_i  = B_i p_i + sum_l E_il r_l
// MM = compile-time bound on nres (registers for the residuals).  The block that finishes last closes the
// block of iterations (blk_j = 0), which also makes a second launch of this kernel a no-op.
// FLUSH_UNR = shifted systems whose x_i, p_i loads are in flight together.  The sweep is latency-bound at the
// 2 blocks per SM its registers allow (ncu: long-scoreboard stalls, 25 % occupancy): 4 shifts (8 x 16 B per
// thread) in flight instead of 2 took it from 5.6 to 6.3 TB/s at 48^4 (profiles/ncu_full_r01.md).
#ifndef FLUSH_UNR
#define FLUSH_UNR 8          // MM <= 16
#endif
#ifndef FLUSH_UNR_LONG
#define FLUSH_UNR_LONG 4     // MM = 32: the 32 residuals of a site already take 128 registers
#endif
template <typename T, int MM, bool RATIONAL, bool FULL, int U>
__device__ __forceinline__ void cg_flush_body(const int nres, const int nl, const int e_base, const bool first, const bool last,
                                              V2<T>* const* sx, V2<T>* const* sp, const V2<T>* const* sq,
                                              const V2<T>* const* sr, const T* sCP, const T* sB, const V2<T>* sDE,
                                              const T* sY, V2<T>* __restrict__ y, const size_t n) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        V2<T> rv[MM];
#pragma unroll
        for (int l = 0; l < MM; ++l)
            if (FULL || l < nres) rv[l] = sr[l][j];
        V2<T> yv;
        if (RATIONAL) {
            yv = y[j];
#pragma unroll
            for (int l = 0; l < MM; ++l)
                if (FULL || l < nres) {
                    yv.x = fma(sY[l], rv[l].x, yv.x);
                    yv.y = fma(sY[l], rv[l].y, yv.y);
                }
        }
        // U shifts at a time (the last group is clamped to the last shift and its surplus lanes are not stored)
        for (int e0 = 0; e0 < nl; e0 += U) {
            V2<T> pv[U], xv[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int e = min(e0 + u, nl - 1);
                pv[u] = sq[e][j];                              // first block: the source b for every shifted system
                if (!RATIONAL) xv[u] = first ? make_v2((T)0, (T)0) : sx[e][j];
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int e = e0 + u;
                if (e < nl) {
                    const T cp = sCP[e], bb = sB[e];
                    T dx = cp * pv[u].x, dy = cp * pv[u].y;
                    T px = bb * pv[u].x, py = bb * pv[u].y;
#pragma unroll
                    for (int l = 0; l < MM; ++l)
                        if (FULL || l < nres) {
                            const V2<T> de = sDE[e * MM + l];
                            if (!RATIONAL) {
                                dx = fma(de.x, rv[l].x, dx);
                                dy = fma(de.x, rv[l].y, dy);
                            }
                            px = fma(de.y, rv[l].x, px);
                            py = fma(de.y, rv[l].y, py);
                        }
                    if (!RATIONAL) {
                        xv[u].x += dx;
                        xv[u].y += dy;
                        sx[e][j] = xv[u];
                    } else {
                        yv.x += dx;
                        yv.y += dy;
                    }
                    if (e != e_base && !last) sp[e][j] = make_v2(px, py);   // the base system's p is kept by K2; after the last
                                                                            // iteration of a solve no p_i is needed any more
                }
            }
        }
        if (RATIONAL) y[j] = yv;
    }
}

// The sweep as a block-level function (every thread of every block of the grid calls it; blockDim.x >=
// LQCD_MAX_SHIFTS + MM): used by cg_flush_kernel and, between grid-wide barriers, by the persistent solver.
template <typename T, int MM, int U = ((MM <= 16) ? FLUSH_UNR : FLUSH_UNR_LONG)>
__device__ __forceinline__ void cg_flush_block(const CgState* st, const size_t n, const int nres, const bool last) {
    __shared__ V2<T>* sx[LQCD_MAX_SHIFTS];
    __shared__ V2<T>* sp[LQCD_MAX_SHIFTS];           // p_i as written
    __shared__ const V2<T>* sq[LQCD_MAX_SHIFTS];     // P as read: p_i, p_keep (base system), or b in the first block
    const bool first = st->first_block != 0;
    __shared__ const V2<T>* sr[MM];
    __shared__ T sCP[LQCD_MAX_SHIFTS], sB[LQCD_MAX_SHIFTS], sY[MM];
    __shared__ V2<T> sDE[LQCD_MAX_SHIFTS * MM];
    __shared__ int cnt[2];
    __shared__ int s_ebase;
    const int tid = threadIdx.x;
    if (tid == 0) s_ebase = -1;
    const int rational = st->rational;
    // compact list of the shifts of this block (two warps, one thread per shift)
    int inb = 0;
    unsigned int bal = 0;
    if (tid < LQCD_MAX_SHIFTS) {
        inb = (tid < st->nshift) ? st->in_block[tid] : 0;
        bal = __ballot_sync(0xffffffffu, inb);
        if ((tid & 31) == 0) cnt[tid >> 5] = __popc(bal);
    }
    if (tid >= LQCD_MAX_SHIFTS && tid < LQCD_MAX_SHIFTS + MM) {
        const int l = tid - LQCD_MAX_SHIFTS;
        sr[l] = (const V2<T>*)st->hist[l < nres ? l : 0];
    }
    __syncthreads();
    const int nl = cnt[0] + cnt[1];
    if (inb) {
        const int e = __popc(bal & ((1u << (tid & 31)) - 1u)) + ((tid >= 32) ? cnt[0] : 0);
        sx[e] = (V2<T>*)st->x[tid];
        sp[e] = (V2<T>*)st->p[tid];
        if (tid == st->i0) {                     // block-deferred base system: P = p^(n0), read only
            sq[e] = (const V2<T>*)st->p_keep;
            s_ebase = e;
        } else {
            sq[e] = first ? (const V2<T>*)st->b_src : (const V2<T>*)st->p[tid];
        }
        sCP[e] = (T)st->blk_CP[tid];
        sB[e] = (T)st->blk_B[tid];
#pragma unroll
        for (int l = 0; l < MM; ++l)
            sDE[e * MM + l] = (l < nres) ? make_v2((T)st->blk_D[l * LQCD_MAX_SHIFTS + tid], (T)st->blk_E[l * LQCD_MAX_SHIFTS + tid])
                                         : make_v2((T)0, (T)0);
    }
    __syncthreads();
    if (rational && tid < MM) {                  // y += sum_l (sum_i D_il) r_l
        T acc = (T)0;
        for (int e = 0; e < nl; ++e) acc += sDE[e * MM + tid].x;
        sY[tid] = acc;
    }
    __syncthreads();
    V2<T>* __restrict__ y = (V2<T>*)st->y;
    if (nl > 0) {
        if (rational) {
            if (nres == MM) cg_flush_body<T, MM, true, true, U>(nres, nl, s_ebase, first, last, sx, sp, sq, sr, sCP, sB, sDE, sY, y, n);
            else cg_flush_body<T, MM, true, false, U>(nres, nl, s_ebase, first, last, sx, sp, sq, sr, sCP, sB, sDE, sY, y, n);
        } else {
            if (nres == MM) cg_flush_body<T, MM, false, true, U>(nres, nl, s_ebase, first, last, sx, sp, sq, sr, sCP, sB, sDE, sY, y, n);
            else cg_flush_body<T, MM, false, false, U>(nres, nl, s_ebase, first, last, sx, sp, sq, sr, sCP, sB, sDE, sY, y, n);
        }
    }
}

template <typename T, int MM>
__global__ void __launch_bounds__(CG_BLOCK, (MM <= 8 ? 2 : 1)) cg_flush_kernel(CgState* st, size_t n) {
    const int nres = st->blk_j;
    if (nres == 0) return;                       // nothing accumulated (solve already over); same in every block
    cg_flush_block<T, MM>(st, n, nres, st->stop != 0);      // stop is set: this is the sweep that ends the solve
    // the last block to finish closes the block of iterations; every block has read the state by then
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(&st->ticket[3], 1u);
        if (t == gridDim.x - 1) {
            st->ticket[3] = 0;
            st->blk_j = 0;
            st->first_block = 0;
        }
    }
}

// ---- mixed precision: single-precision CG with double-precision reliable updates -------------------------------
// ("fp32 inner, fp64 reliable updates"; the paper keeps its fields in either precision,
// PAPER.md:L147, and runs MD in single, Metropolis in double.)
// The float CG iterates on a recurrence residual r and accumulates its solution in a float vector y.  At a
// reliable update the accumulated y is added to the double-precision solution x (and cleared), the TRUE residual
// b - (A + sigma) x is computed with the double-precision operator, and replaces r; the search direction is kept
// (p = r_true + beta p_old), so the Krylov sequence is not restarted.

// x64 += y32 ; y32 = 0
__global__ void __launch_bounds__(CG_BLOCK) mixed_accumulate_kernel(double2* __restrict__ x, float2* __restrict__ y, size_t n) {
    for (size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x; j < n; j += (size_t)gridDim.x * CG_BLOCK) {
        const float2 v = y[j];
        double2 xv = x[j];
        xv.x += (double)v.x;
        xv.y += (double)v.y;
        x[j] = xv;
        y[j] = make_float2(0.f, 0.f);
    }
}

// r_true = b - ax (double; ax == NULL: r_true = b);  |r_true|^2 -> *rr_out;  r_out = float(r_true).
// replace != 0: r_out is the ring slot the next iteration reads its residual from, and |r_true|^2 replaces the
// recurrence value on the device.  The search direction needs no correction: the fused iteration forms
// p = r + beta p_old from whatever residual it finds there, so p = r_true + beta p_old, the direction is kept and
// the Krylov sequence is not restarted.
// resume != 0: the float solver had stopped on its recurrence residual and is started again.
__global__ void __launch_bounds__(CG_BLOCK) mixed_residual_kernel(const double2* __restrict__ b, const double2* __restrict__ ax,
                                                                  float2* __restrict__ r_out, CgState* st, double* partials,
                                                                  double* rr_out, size_t n, int replace, int resume) {
    __shared__ double red[32];
    __shared__ int last_flag;
    double acc = 0.0;
    for (size_t j = (size_t)blockIdx.x * CG_BLOCK + threadIdx.x; j < n; j += (size_t)gridDim.x * CG_BLOCK) {
        double2 r = b[j];
        if (ax) {
            const double2 a = ax[j];
            r.x -= a.x;
            r.y -= a.y;
        }
        acc = fma(r.x, r.x, acc);
        acc = fma(r.y, r.y, acc);
        r_out[j] = make_float2((float)r.x, (float)r.y);
    }
    const double bsum = block_sum<CG_BLOCK>(acc, red);
    if (publish_partial<CG_BLOCK>(bsum, partials, &st->ticket[4], &last_flag)) {
        const double rr = final_sum<CG_BLOCK>(partials, gridDim.x, red);
        if (threadIdx.x == 0) {
            st->ticket[4] = 0;
            *rr_out = rr;
            if (replace) st->rr = rr;
            if (resume) {
                st->stop = 0;
                st->active[st->i0] = 1;
            }
        }
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
