// lqcd_internal.cuh -- shared declarations of the CUDA library (not part of the C ABI).
#ifndef LQCD_INTERNAL_CUH
#define LQCD_INTERNAL_CUH

#include <cuda_runtime.h>
#include <stdint.h>

#include "fastdiv.h"

#define LQCD_MAX_SHIFTS 64          // r of Eq. 2; rational approximations use <= ~20

// The path exists in the two precisions the paper runs in ("double (or float) C99 complex numbers",
// PAPER.md:L147; single precision for the MD evolution).  Every kernel is a template on the
// real type T; a complex number is the 2-vector V2<T> (128-bit loads in double, 64-bit in single).
template <typename T> struct Cplx;
template <> struct Cplx<double> { typedef double2 type; };
template <> struct Cplx<float> { typedef float2 type; };
template <typename T> using V2 = typename Cplx<T>::type;
__host__ __device__ __forceinline__ double2 make_v2(double x, double y) { return make_double2(x, y); }
__host__ __device__ __forceinline__ float2 make_v2(float x, float y) { return make_float2(x, y); }

// Geometry of one parity of the lattice in the checkerboard index k = lex>>1 =
// xh + Lxh*(y + Ly*(z + Lz*t)), xh = x>>1 ("Data layout").
struct Geom {
    FastDiv dxh, dy, dz;            // divisions by Lxh, Ly, Lz
    int Lxh, Ly, Lz, Lt;
    int Vh;                         // sites per parity
    int sy, sz, st;                 // strides of y, z, t in k
    int antiperiodic;               // bc_t = -1 on links leaving t = Lt-1
    int t_off, Lt_glob;             // slab mode: this lattice is time slices [t_off, t_off+Lt) of Lt_glob
};

// Peer-memory transport (p2p.cuh): where the rank's share of a scalar product goes -- one slot and one flag word in
// every rank's window (its own included).  Lives in device memory, one per generation of the all-reduce.
#define LQCD_P2P_MAX_RANKS 16
#define LQCD_P2P_RED_MAX 4          // doubles per all-reduce slot
// Written into the arrival words of its peers by a rank that gives up (p2p.cuh, poison): it satisfies every
// ">= 1" stream wait (the comparison is a signed difference), is never written otherwise, and the kernels that consume
// a halo or the slots of an all-reduce leave it in place and record LQCD_ECOMM in the CG state instead of clearing it.
#define LQCD_P2P_POISON 0x40000000u
#define LQCD_ECOMM_DEV (-8)         // LQCD_ECOMM of include/lqcd.h
struct PeerPush {
    double* slot[LQCD_P2P_MAX_RANKS];
    unsigned int* flag[LQCD_P2P_MAX_RANKS];
    int nranks;
};
// value -> every rank's slot, then (system-wide fence) 1 -> every rank's flag; threads 0..nranks-1 of one block
__device__ __forceinline__ void peer_push(const PeerPush* __restrict__ d, const double value) {
    const int q = threadIdx.x;
    if (q < d->nranks) {
        *(volatile double*)d->slot[q] = value;
        __threadfence_system();
        *(volatile unsigned int*)d->flag[q] = 1u;
    }
}

#ifndef LQCD_MAX_BLOCK
#define LQCD_MAX_BLOCK 32           // longest block of iterations whose shift updates are applied in one sweep
#endif

// Device-resident state of one multi-shift CG solve (steps A6, A9): every scalar of the recurrence
// lives here, so an iteration needs no host round trip.
//
// Block-deferred shift updates.  Within a block of m iterations that starts at
// iteration n0 with P = p_i, X = x_i, the recurrences  x_i += a_i p_i ;  p_i = zeta_i r + b_i p_i  unroll to
//     p_i^(n0+j) = B_j P + sum_{l=1..j} E_{j,l} r^(n0+l)
//     x_i^(n0+j) = X + CP_j P + sum_{l=1..j-1} D_{j,l} r^(n0+l)
// so the shifted x_i, p_i need not be touched until the block ends if the m residuals of the block are kept
// (m x 48 B per site, shared by all shifts) and the scalar coefficients B, E, CP, D are carried along.
// The base system's p is needed by the operator every iteration and is updated every iteration.
struct CgState {
    double rr, bb, pAp, a, a_prev, b_prev, tol2bb, c0;
    int iter, max_iter, stop, status, nshift, i0, blk_m;
    int blk_j;                      // iterations accumulated in the current block (0..blk_m)
    unsigned int ticket[5];
    double delta[LQCD_MAX_SHIFTS];
    double zeta[LQCD_MAX_SHIFTS], zeta_prev[LQCD_MAX_SHIFTS], zeta_new[LQCD_MAX_SHIFTS];
    int active[LQCD_MAX_SHIFTS], freeze_iter[LQCD_MAX_SHIFTS];
    // block coefficients, per shift i (index [l*LQCD_MAX_SHIFTS + i] so that a warp's accesses coalesce)
    int in_block[LQCD_MAX_SHIFTS];  // shift takes part in the current block (was active at its start, not the base)
    double blk_B[LQCD_MAX_SHIFTS], blk_CP[LQCD_MAX_SHIFTS];
    double blk_E[LQCD_MAX_BLOCK * LQCD_MAX_SHIFTS], blk_D[LQCD_MAX_BLOCK * LQCD_MAX_SHIFTS];
    void* x[LQCD_MAX_SHIFTS];       // V2<T>* of the precision the solve runs in
    void* p[LQCD_MAX_SHIFTS];
    void* hist[LQCD_MAX_BLOCK];     // residual ring: r^(n0+l) is in hist[l-1], l = 1..m; r^(n0) in hist[m-1]
    // rational-sum mode (lqcd_rational_apply): y = alpha0 b + sum_i alpha_i x_i is accumulated during the
    // solve and the x_i are never stored; blk_CP, blk_D then carry the factor alpha_i
    int rational;
    double alpha0;
    double alpha[LQCD_MAX_SHIFTS];
    void* y;
    // fused iteration with m >= 2: the base system's x_0 is block-deferred like the shifted ones (zeta = 1).  Its p
    // is still formed every iteration (the operator needs it); p_keep holds p^(n0), the direction of the block's
    // first iteration, which is what the sweep needs besides the block's residuals.
    int defer_base;
    void* p_keep;
    // Until the first block sweep every shifted system still has p_i = b, x_i = 0: cg_init does not write those 2 x
    // nshift vectors; the first sweep reads P from the source b_src (one vector, shared) and X as zero, and writes them.
    int first_block;
    const void* b_src;
    // small lattices (dslash_kernel, FS = 1): |r|^2 and the iteration count as they were BEFORE the scalar step after K2,
    // which runs beside the blocks of the next K1 that still need them
    double rr_keep;
    int iter_keep;
};

#endif
