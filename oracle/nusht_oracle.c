/*
 * nusht_oracle.c -- plain, slow CPU oracle for the nonuniform spin-0 spherical harmonic
 * transform of arXiv 2406.14542: direct evaluation of Eq. 3 (synthesis) and
 * Eq. 2 (adjoint).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no
 * code, header, table or constant with the CUDA path under paper_2406_14542_b200/ and neither
 * includes the other.  The product path never falls back to it.
 *
 * Parity pins (tests/test_oracle_pins.py): closed forms Y_00, Y_10, Y_11, Y_20..Y_22; mpmath
 * and scipy library values of Y_lm; the addition theorem; orthonormality under Gauss-Legendre
 * quadrature; the adjoint identity <S a, x> = <a, S^T x>; special cases; every copy of the l loop also in the
 * exponent-rescaling regime (lmax 1500 .. 8191, near-pole points: mpmath values, the adjoint identity, ring_sum
 * against synthesis); oracle_gradient (Eq. C2) by closed forms, finite differences of the synthesis and the ladder
 * identity at lmax = 1500.  No function here is "parity unpinned".
 *
 * Build (done by __graft_entry__.build() and by oracle/oracle.py on first use):
 *   gcc -O2 -fopenmp -fPIC -shared -o liboracle.so nusht_oracle.c -lm
 * -ffast-math is deliberately NOT used.
 *
 * Two instantiations of the same body:  *_d  (binary64 arithmetic) and  *_ld  (x86 80-bit long
 * double arithmetic); inputs and outputs are binary64 arrays in both.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------------- binary64 instantiation ---------------- */
#define REAL double
#define SUF(name) name##_d
#define R_SQRT sqrt
#define R_SIN sin
#define R_COS cos
#define R_FABS fabs
#define R_LDEXP ldexp
#define R_FREXP frexp
#define R_PI 3.14159265358979323846264338327950288
#include "nusht_oracle_impl.inc"
#undef REAL
#undef SUF
#undef R_SQRT
#undef R_SIN
#undef R_COS
#undef R_FABS
#undef R_LDEXP
#undef R_FREXP
#undef R_PI
#undef ORACLE_RESCALE_BITS

/* ---------------- long double instantiation ---------------- */
#define REAL long double
#define SUF(name) name##_ld
#define R_SQRT sqrtl
#define R_SIN sinl
#define R_COS cosl
#define R_FABS fabsl
#define R_LDEXP ldexpl
#define R_FREXP frexpl
#define R_PI 3.14159265358979323846264338327950288L
#include "nusht_oracle_impl.inc"

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int oracle_long_double_bits(void) { return (int)(sizeof(long double) * 8) * 1000 + __LDBL_MANT_DIG__; }
