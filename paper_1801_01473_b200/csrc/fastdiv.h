// fastdiv.h -- exact unsigned division of n < 2^31 by a run-time constant d < 2^31 with one
// multiply-high and one shift (site index -> lattice coordinates without integer division; step A3 of
// DESIGN.md).  Plain C++ so that a host-only test can brute-force it (tests/test_host_logic.py).
//
//   d == 1 : q = n                                  (m == 0 marks this case)
//   d >= 2 : l = ceil(log2 d), m = ceil(2^(31+l) / d) < 2^32, q = mulhi32(n, m) >> (l-1)
// Exactness for n < 2^31: m = (2^(31+l) + e)/d with 0 <= e < d <= 2^l, so
//   n*m / 2^(31+l) = n/d + n*e / (d * 2^(31+l)), and n*e < 2^(31+l) keeps the excess below 1/d.
#ifndef LQCD_FASTDIV_H
#define LQCD_FASTDIV_H

#include <stdint.h>

#if defined(__CUDACC__)
#define LQCD_HD __host__ __device__ __forceinline__
#else
#define LQCD_HD inline
#endif

struct FastDiv {
    uint32_t m;    // magic multiplier, 0 for d == 1
    uint32_t sh;   // post-shift
    uint32_t d;    // the divisor itself
};

inline FastDiv make_fastdiv(uint32_t d) {
    FastDiv f;
    f.d = d;
    if (d <= 1) {
        f.m = 0;
        f.sh = 0;
        return f;
    }
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    const uint64_t num = 1ull << (31 + l);
    f.m = (uint32_t)((num + d - 1) / d);
    f.sh = l - 1;
    return f;
}

LQCD_HD uint32_t fastdiv(uint32_t n, const FastDiv& f) {
#if defined(__CUDA_ARCH__)
    const uint32_t hi = __umulhi(n, f.m);
#else
    const uint32_t hi = (uint32_t)(((uint64_t)n * f.m) >> 32);
#endif
    return f.m ? (hi >> f.sh) : n;
}

#endif
