// reduce.cuh -- deterministic two-stage reductions and the device-side CG scalar recurrences.
//
// Stage 1: every block reduces its threads' values with a fixed shuffle tree and writes ONE partial.
// Stage 2: the block that finishes last (atomic ticket) adds all partials in a fixed order.  No
// floating-point atomics anywhere, so a solve is bit-reproducible for a given lattice (R8).
// The same last block then runs the scalar part of the iteration (steps A6 and A9).
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

// ---- scalar recurrences (SURVEY.md §8(c2) / DESIGN.md R5), run by thread 0 of the last block ------

// after |b|^2 is known (solve start)
__device__ inline void cg_scalars_init(CgState* st, double bb, double tol) {
    st->rr = bb;
    st->bb = bb;
    st->tol2bb = tol * tol * bb;
    st->a_prev = 1.0;
    st->b_prev = 0.0;
    st->iter = 0;
    st->status = 0;
    st->nlist = 0;
    const int stop = (bb == 0.0) ? 1 : 0;       // zero source: x_i = 0 is the answer
    st->stop = stop;
    st->stop4 = stop;
    for (int i = 0; i < st->nshift; ++i) {
        st->zeta[i] = 1.0;
        st->zeta_prev[i] = 1.0;
        st->zeta_new[i] = 1.0;
        st->active[i] = 1;
        st->freeze_iter[i] = 0;
    }
}

// after pAp = Re<p, B p> is known: step length and the shifted coefficients
__device__ inline void cg_scalars_after_pAp(CgState* st, double pAp) {
    st->pAp = pAp;
    if (!(pAp > 0.0) || !isfinite(pAp)) {
        st->status = -6;                         // LQCD_EBREAKDOWN
        st->stop = 1;
        st->stop4 = 1;
        st->nlist = 0;
        return;
    }
    const double a = st->rr / pAp;
    st->a = a;
    const double a_prev = st->a_prev, b_prev = st->b_prev;
    int n = 0;
    for (int i = 0; i < st->nshift; ++i) {
        if (!st->active[i]) continue;
        const double z = st->zeta[i], zp = st->zeta_prev[i];
        const double zn = z * zp * a_prev / (a_prev * zp * (1.0 + st->delta[i] * a) + a * b_prev * (zp - z));
        st->zeta_new[i] = zn;
        st->list_idx[n] = i;
        st->list_a[n] = st->rational ? st->alpha[i] * (a * zn / z) : a * zn / z;
        st->list_zn[n] = zn;
        ++n;
    }
    st->nlist = n;
}

// after |r_new|^2 is known: direction coefficients, shift of the recurrence, freezing, stopping rule
__device__ inline void cg_scalars_after_rr(CgState* st, double rr_new) {
    const double bt = rr_new / st->rr;
    for (int e = 0; e < st->nlist; ++e) {
        const int i = st->list_idx[e];
        const double ratio = st->zeta_new[i] / st->zeta[i];
        st->list_b[e] = bt * ratio * ratio;
        st->zeta_prev[i] = st->zeta[i];
        st->zeta[i] = st->zeta_new[i];
    }
    st->a_prev = st->a;
    st->b_prev = bt;
    st->rr = rr_new;
    const int it = st->iter + 1;
    st->iter = it;
    for (int i = 0; i < st->nshift; ++i) {
        if (!st->active[i]) continue;
        if (st->zeta[i] * st->zeta[i] * rr_new <= st->tol2bb) {
            st->active[i] = 0;
            st->freeze_iter[i] = it;
        }
    }
    if (rr_new <= st->tol2bb) {
        st->stop = 1;
    } else if (it >= st->max_iter) {
        st->stop = 1;
        st->status = -5;                         // LQCD_ENOCONV
    }
}

#endif
