// reduce.cuh -- deterministic two-stage reductions and the device-side CG scalar recurrences.
//
// Stage 1: every block reduces its threads' values with a fixed shuffle tree and writes ONE partial.
// Stage 2: ONE block adds all partials in a fixed order (final_sum) -- a one-block kernel launched after the sweep
// (the CG iteration: cg_reduce_scalar_kernel, sum_partials_kernel), or, in the kernels that run once per solve, the
// block that finishes last (publish_partial: fence + atomic ticket in every block, too dear for 20,000 blocks twice
// per iteration).  No floating-point atomics anywhere, so a solve is bit-reproducible for a given lattice
// (R8).  The block that holds the sum then runs the scalar part of the iteration (steps A6 and A9).
#ifndef LQCD_REDUCE_CUH
#define LQCD_REDUCE_CUH

#include "lqcd_internal.cuh"

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; result valid in thread 0.  `red` holds >= 32 doubles of shared memory.
// One barrier; the caller must put a barrier between two calls that use the same `red`.
template <int BLOCK>
__device__ __forceinline__ double block_sum(double v, double* red) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) red[w] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < BLOCK / 32; ++i) s += red[i];
    }
    return s;
}

// Writes this block's partial, then tells whether this block is the last one of the grid to do so.
// When it returns true (for every thread of that block) all partials of the grid are visible.
// The barrier inside also separates the caller's block_sum from a following final_sum.
template <int BLOCK>
__device__ __forceinline__ bool publish_partial(double block_value, double* partials, unsigned int* ticket,
                                                int* flag_smem) {
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = block_value;
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        *flag_smem = (t == gridDim.x - 1);
    }
    __syncthreads();
    return *flag_smem != 0;
}

// Sum of n partials by one whole block, fixed order; result valid in thread 0.  Sixteen independent loads
// per thread are in flight at a time: with ~20k partials (48^4) a one-load-at-a-time loop costs tens of
// microseconds of exposed L2 latency at the tail of the kernel.
template <int BLOCK>
__device__ __forceinline__ double final_sum(const double* partials, int n, double* red) {
    constexpr int U = 16;
    double a[U];
#pragma unroll
    for (int u = 0; u < U; ++u) a[u] = 0.0;
    int i = threadIdx.x;
    for (; i + (U - 1) * BLOCK < n; i += U * BLOCK) {
        double v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) v[u] = __ldcg(partials + i + u * BLOCK);
#pragma unroll
        for (int u = 0; u < U; ++u) a[u] += v[u];
    }
    for (; i < n; i += BLOCK) a[0] += __ldcg(partials + i);
#pragma unroll
    for (int w = U / 2; w > 0; w >>= 1)
#pragma unroll
        for (int u = 0; u < w; ++u) a[u] += a[u + w];
    return block_sum<BLOCK>(a[0], red);
}

// value of thread 0 -> every thread of the block (red is the scratch of the block_sum that produced it)
__device__ __forceinline__ double broadcast0(double v, double* red) {
    __syncthreads();
    if (threadIdx.x == 0) red[0] = v;
    __syncthreads();
    return red[0];
}

// ---- scalar recurrences (SURVEY.md §8(c2) / DESIGN.md R5) ------------------------------------------
// Run by the block that holds the sum, ALL its threads calling (blockDim.x >= LQCD_MAX_SHIFTS): thread i
// carries shift i, thread 0 also the scalars of the base system, so the tail of the kernel costs one chain
// of dependent operations instead of nshift of them.  Besides the zeta recurrences the threads carry the
// block coefficients B, E, CP, D of the deferred shift updates (lqcd_internal.cuh, CgState).

// after |b|^2 is known (solve start); thread 0 only
__device__ inline void cg_scalars_init(CgState* st, double bb, double tol) {
    st->rr = bb;
    st->bb = bb;
    st->tol2bb = tol * tol * bb;
    st->a_prev = 1.0;
    st->b_prev = 0.0;
    st->iter = 0;
    st->status = 0;
    st->blk_j = 0;
    st->first_block = 1;
    const int stop = (bb == 0.0) ? 1 : 0;       // zero source: x_i = 0 is the answer
    st->stop = stop;
    for (int i = 0; i < st->nshift; ++i) {
        st->zeta[i] = 1.0;
        st->zeta_prev[i] = 1.0;
        st->zeta_new[i] = 1.0;
        st->active[i] = 1;
        st->in_block[i] = 0;
        st->freeze_iter[i] = 0;
    }
}

// after pAp = Re<p, B p> is known: step length, zeta_new_i, and the x-part of the block coefficients
//   x_i += a_i p_i  with  p_i = B P + sum_l E_l r_l   =>   CP += a_i B ;  D_l += a_i E_l  (l < j)
__device__ __noinline__ void cg_scalars_after_pAp(CgState* st, double pAp) {
    const int tid = threadIdx.x;
    const double rr = st->rr, a_prev = st->a_prev, b_prev = st->b_prev;
    const int j = st->blk_j, ns = st->nshift, i0 = st->i0, rational = st->rational;
    if (!(pAp > 0.0) || !isfinite(pAp)) {
        if (tid == 0) {
            st->pAp = pAp;
            st->status = -6;                     // LQCD_EBREAKDOWN
            st->stop = 1;
        }
        return;
    }
    const double a = rr / pAp;
    if (tid < ns) {
        const int i = tid;
        const int act = st->active[i];
        const int inb = (j == 0) ? (act && (i != i0 || st->defer_base)) : st->in_block[i];
        if (j == 0) st->in_block[i] = inb;
        if (act) {
            const double z = st->zeta[i], zp = st->zeta_prev[i];
            const double zn = z * zp * a_prev / (a_prev * zp * (1.0 + st->delta[i] * a) + a * b_prev * (zp - z));
            st->zeta_new[i] = zn;
            if (inb) {
                double ai = a * zn / z;
                if (rational) ai *= st->alpha[i];
                if (j == 0) {
                    st->blk_B[i] = 1.0;
                    st->blk_CP[i] = ai;
                } else {
                    st->blk_CP[i] = fma(ai, st->blk_B[i], st->blk_CP[i]);
                    double e[LQCD_MAX_BLOCK], d[LQCD_MAX_BLOCK];
#pragma unroll
                    for (int l = 0; l < LQCD_MAX_BLOCK; ++l)
                        if (l < j) {
                            e[l] = st->blk_E[l * LQCD_MAX_SHIFTS + i];
                            d[l] = st->blk_D[l * LQCD_MAX_SHIFTS + i];
                        }
#pragma unroll
                    for (int l = 0; l < LQCD_MAX_BLOCK; ++l)
                        if (l < j) st->blk_D[l * LQCD_MAX_SHIFTS + i] = fma(ai, e[l], d[l]);
                }
            }
        }
    }
    if (tid == 0) {
        st->pAp = pAp;
        st->a = a;
        st->rr_keep = rr;
        st->iter_keep = st->iter;
    }
}

// after |r_new|^2 is known: beta, b_i, the p-part of the block coefficients
//   p_i = zeta_new_i r_new + b_i p_i   =>   B *= b_i ;  E_l *= b_i (l < j) ;  E_j = zeta_new_i ;  D_j = 0
// then the shift of the recurrence, freezing and the stopping rule
__device__ __noinline__ void cg_scalars_after_rr(CgState* st, double rr_new) {
    const int tid = threadIdx.x;
    const double rr_old = st->rr, a = st->a, tol2bb = st->tol2bb;
    const int j = st->blk_j, ns = st->nshift, it = st->iter + 1, max_iter = st->max_iter;
    const double bt = rr_new / rr_old;
    if (tid < ns) {
        const int i = tid;
        const int act = st->active[i], inb = st->in_block[i];
        if (act) {
            const double z = st->zeta[i], zn = st->zeta_new[i];
            const double ratio = zn / z;
            const double bi = bt * ratio * ratio;
            if (inb) {
                st->blk_B[i] = (j == 0 ? 1.0 : st->blk_B[i]) * bi;
                double e[LQCD_MAX_BLOCK];
#pragma unroll
                for (int l = 0; l < LQCD_MAX_BLOCK; ++l)
                    if (l < j) e[l] = st->blk_E[l * LQCD_MAX_SHIFTS + i];
#pragma unroll
                for (int l = 0; l < LQCD_MAX_BLOCK; ++l)
                    if (l < j) st->blk_E[l * LQCD_MAX_SHIFTS + i] = e[l] * bi;
                st->blk_E[j * LQCD_MAX_SHIFTS + i] = zn;
                st->blk_D[j * LQCD_MAX_SHIFTS + i] = 0.0;
            }
            st->zeta_prev[i] = z;
            st->zeta[i] = zn;
            if (zn * zn * rr_new <= tol2bb) {
                st->active[i] = 0;
                st->freeze_iter[i] = it;
            }
        } else if (inb) {                        // frozen earlier in this block: its x_i no longer moves
            st->blk_E[j * LQCD_MAX_SHIFTS + i] = 0.0;
            st->blk_D[j * LQCD_MAX_SHIFTS + i] = 0.0;
        }
    }
    __syncthreads();                             // every thread has read the old scalars
    if (tid == 0) {
        st->a_prev = a;
        st->b_prev = bt;
        st->rr = rr_new;
        st->iter = it;
        st->blk_j = j + 1;
        if (rr_new <= tol2bb) {
            st->stop = 1;
        } else if (it >= max_iter) {
            st->stop = 1;
            st->status = -5;                     // LQCD_ENOCONV
        }
    }
}

#endif
