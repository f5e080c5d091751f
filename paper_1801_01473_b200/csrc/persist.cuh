// persist.cuh -- the whole multi-shift CG solve as ONE cooperative kernel, for lattices that live in L2.
//
// "Small lattices are launch-bound".  At 16^4 (BASELINE config 2) links and vectors stay in L2 and
// one operator application is ~2.5 us of work; the iteration of two launches (cg.cuh) then spends more time in
// launch gaps, kernel tails and the single-block reduction + scalar step at the end of each launch than in the
// operators (measured: 20 us per iteration against 2 x 4.5 us for two bare applications in a CUDA graph).
//
// Here the grid is resident for the whole solve.  One iteration is the same two sweeps K1, K2 of cg.cuh (the same
// device functions: dslash_hops, k1_finish, k2_finish, cg_flush_block), separated by two grid-wide barriers:
//
//   K1 sweep -> block partial of <p,Ap> -> BARRIER -> every block adds the partials in the same fixed order
//            -> every block holds a = rr/pAp;  the scalar block advances the full scalar state (zeta_i, coefficients)
//   K2 sweep -> block partial of |r_new|^2 -> BARRIER -> every block adds the partials
//            -> every block holds beta, the iteration count and the stop decision;  the scalar block advances the state
//   every m-th iteration (and at the stop): BARRIER (the scalar block's coefficients are visible) -> block sweep
//
// Every block carries the few scalars the sweeps need (rr, a, beta, iteration count, stop) redundantly in registers
// -- same operands, same operations, hence the same bits in every block.  The recurrences of the shifted systems,
// the block coefficients, freeze flags and statistics are advanced on the device state exactly as the one-block
// kernels do on the multi-launch path (same functions), by ONE EXTRA BLOCK that owns no sites: its scalar step
// (a few dependent round trips to L2, ~2.5 us) runs while the other blocks are in the next sweep, so it is off the
// critical path (measured at 16^4: with block 0 doing it on top of its sites every barrier waited for it and the
// iteration took 22 us, no better than two launches).  No host round trip until the solve is over.
#ifndef LQCD_PERSIST_CUH
#define LQCD_PERSIST_CUH

#include <cooperative_groups.h>

#include "cg.cuh"
#include "dslash.cuh"

// threads per block of the persistent solver: the cost of a grid-wide barrier grows with the number of blocks, so
// few large blocks (one per SM) beat many small ones here
#ifndef PS_BLOCK
#define PS_BLOCK 256
#endif
// longest block of deferred updates the persistent solver handles (registers of the sweep)
#define PS_MAX_BLOCK 16
static_assert(PS_BLOCK >= LQCD_MAX_SHIFTS + LQCD_MAX_BLOCK, "scalar step and sweep set-up need one thread per shift / residual");

template <typename T>
struct PersistArgs {
    DslashArgs<T> D;         // geometry, links, angles, cache policy (the vector pointers in it are not used)
    CgState* st;
    double* partials;        // 2 x gridDim.x doubles
    V2<T>* p;                // search direction of the base system
    V2<T>* t;                // D_oe p (odd sites)
    V2<T>* p_keep;           // p of the first iteration of the current block (base system deferred)
    int m;                   // block length of the deferred updates
    int defer_base;
};

// sum of the grid's partials, fixed order, the same value in every thread of every block
__device__ __forceinline__ double persist_sum(const double* partials, int n, double* red) {
    return broadcast0(final_sum<PS_BLOCK>(partials, n, red), red);
}

template <typename T, int RECON, int U1>
__global__ void __launch_bounds__(PS_BLOCK, 1) cg_persistent_kernel(const PersistArgs<T> P) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ double red[32];
    CgState* st = P.st;
    if (st->stop) return;                                   // zero source
    const Geom& g = P.D.g;
    const size_t vh = (size_t)g.Vh;
    // the last block of the grid owns no sites: it advances the scalar state while the others sweep
    const int nsb = (int)gridDim.x - 1;                     // blocks that own sites
    const bool scalar_block = ((int)blockIdx.x == nsb);
    // sites are dealt out evenly: block b owns the contiguous range [b*chunk, (b+1)*chunk), so that every SM carries
    // the same load even when there are fewer sites than resident threads (16^4: 223 sites for each of 147 blocks)
    const int chunk = (g.Vh + nsb - 1) / nsb;
    const int k_begin = scalar_block ? g.Vh : min((int)blockIdx.x * chunk, g.Vh);
    const int k_end = scalar_block ? g.Vh : min(k_begin + chunk, g.Vh);
    const int m = P.m;
    double* part1 = P.partials;
    double* part2 = P.partials + gridDim.x;

    // the scalars every block carries (the scalar block keeps the device state in step with them)
    double rr = st->rr, beta = st->b_prev;
    const double tol2bb = st->tol2bb, c0 = st->c0;
    const int max_iter = st->max_iter, rational = st->rational, i0 = st->i0;
    const double alpha_i0 = rational ? st->alpha[i0] : 1.0;
    int iter = st->iter;
    K2Coef<T> C;
    C.c0 = (T)c0;
    C.xp = (V2<T>*)(rational ? st->y : st->x[i0]);
    C.p_out = P.p;
    C.defer_base = P.defer_base;
    __shared__ V2<T>* hist[LQCD_MAX_BLOCK];                  // the residual ring
    if (threadIdx.x < LQCD_MAX_BLOCK) hist[threadIdx.x] = (V2<T>*)st->hist[threadIdx.x < m ? threadIdx.x : 0];
    __syncthreads();

    int pos = 0;                    // position inside the block of m iterations
    bool close_block = false;       // the sweep of the previous iteration closed a block: blk_j is to be reset
    for (;;) {
        __syncthreads();                                     // red: the previous iteration's broadcast has been read
        const V2<T>* r_in = hist[(pos + m - 1) % m];
        V2<T>* r_out = hist[pos];

        // ---- K1: t = D_oe p, p = r + beta p_old at the neighbours;  <p,Ap>
        double dot = 0.0;
        for (int k = k_begin + (int)threadIdx.x; k < k_end; k += PS_BLOCK) {
            T ar[3] = {(T)0, (T)0, (T)0}, ai[3] = {(T)0, (T)0, (T)0};
            double pp = 0.0;
            dslash_hops<T, RECON, U1, 0, true, true>(P.D, 1, k, r_in, P.p, (T)beta, ar, ai, pp);
            dot += k1_finish<T>(P.t, vh, k, true, ar, ai, pp, c0);
        }
        double bsum = block_sum<PS_BLOCK>(dot, red);
        if (threadIdx.x == 0 && !scalar_block) part1[blockIdx.x] = bsum;
        grid.sync();
        const double pAp = persist_sum(part1, nsb, red);
        if (scalar_block) {
            if (close_block && threadIdx.x == 0) {                  // every block is past the sweep by now
                st->blk_j = 0;
                st->first_block = 0;
            }
            __syncthreads();
            cg_scalars_after_pAp(st, pAp);
        }
        close_block = false;
        const bool breakdown = !(pAp > 0.0) || !isfinite(pAp);      // the scalar block records it in the state
        bool stop = breakdown;
        if (!breakdown) {
            const double a = rr / pAp;
            C.beta = (T)beta;
            C.a = (T)a;
            C.ax = (T)(alpha_i0 * a);
            C.r_out = r_out;
            C.p_keep = (P.defer_base && pos == 0) ? P.p_keep : nullptr;

            // ---- K2: p, s = c0 p - D_eo t, r_new = r - a s, x_0 += a p at the thread's own sites;  |r_new|^2
            dot = 0.0;
            for (int k = k_begin + (int)threadIdx.x; k < k_end; k += PS_BLOCK) {
                V2<T> pold[3], rv[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    pold[c] = P.p[c * vh + k];
                    rv[c] = r_in[c * vh + k];
                }
                T ar[3] = {(T)0, (T)0, (T)0}, ai[3] = {(T)0, (T)0, (T)0};
                double pp = 0.0;
                dslash_hops<T, RECON, U1, 0, false, true>(P.D, 0, k, P.t, P.t, (T)0, ar, ai, pp);
                dot += k2_finish<T>(C, vh, k, true, pold, rv, ar, ai);
            }
            __syncthreads();                                 // red is reused
            bsum = block_sum<PS_BLOCK>(dot, red);
            if (threadIdx.x == 0 && !scalar_block) part2[blockIdx.x] = bsum;
            grid.sync();
            const double rr_new = persist_sum(part2, nsb, red);
            if (scalar_block) cg_scalars_after_rr(st, rr_new);
            beta = rr_new / rr;
            rr = rr_new;
            ++iter;
            stop = (rr_new <= tol2bb) || (iter >= max_iter);
        }

        // ---- the deferred updates of the block (every m-th iteration, and whatever has accumulated at the stop)
        const int nres = breakdown ? pos : pos + 1;          // iterations accumulated in the current block
        if ((pos == m - 1 || stop) && nres > 0) {
            grid.sync();                                     // the scalar block's coefficients are visible
            cg_flush_block<T, PS_MAX_BLOCK, 4>(st, 3 * vh, nres, stop);     // 4 systems in flight: the registers this kernel has
            close_block = true;
        }
        if (stop) break;
        pos = (pos + 1 == m) ? 0 : pos + 1;
    }
    if (close_block) {
        grid.sync();                                         // every block has read the coefficients
        if (scalar_block && threadIdx.x == 0) {
            st->blk_j = 0;
            st->first_block = 0;
        }
    }
}

#endif
