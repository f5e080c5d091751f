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
};

// Device-resident state of one multi-shift CG solve (steps A6, A9): every scalar of the recurrence
// lives here, so an iteration needs no host round trip.
struct CgState {
    double rr, bb, pAp, a, a_prev, b_prev, tol2bb, c0;
    int iter, max_iter, stop, stop4, status, nshift, i0, nlist;
    unsigned int ticket[4];
    double delta[LQCD_MAX_SHIFTS];
    double zeta[LQCD_MAX_SHIFTS], zeta_prev[LQCD_MAX_SHIFTS], zeta_new[LQCD_MAX_SHIFTS];
    int active[LQCD_MAX_SHIFTS], freeze_iter[LQCD_MAX_SHIFTS];
    // update list of the current iteration (shifts that were active when it started)
    int list_idx[LQCD_MAX_SHIFTS];
    double list_a[LQCD_MAX_SHIFTS], list_zn[LQCD_MAX_SHIFTS], list_b[LQCD_MAX_SHIFTS];
    void* x[LQCD_MAX_SHIFTS];       // V2<T>* of the precision the solve runs in
    void* p[LQCD_MAX_SHIFTS];
    // rational-sum mode (lqcd_rational_apply): y = alpha0 b + sum_i alpha_i x_i is accumulated during the
    // solve and the x_i are never stored; list_a then holds alpha_i * a_i
    int rational;
    double alpha0;
    double alpha[LQCD_MAX_SHIFTS];
    void* y;
};

#endif
