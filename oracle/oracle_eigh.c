/* oracle_eigh.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * CPU oracle for the dense complex-Hermitian eigenproblem of PAPER.md:105 (Eq. 7),
 * following the 1-stage outline of PAPER.md:148.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it; the product
 * (paper_2310_03341_b200/) never does.  It shares no code with the CUDA path.
 *
 * Two instantiations of oracle_eigh_impl.inc: FP64 (suffix _d) and x87 80-bit
 * long double (suffix _ld, eps ~ 1.1e-19) used as extended-precision truth.
 *
 * Build:  gcc -O2 -fopenmp -shared -fPIC -std=gnu11 oracle_eigh.c -o liboracle_eigh.so -lm
 * (-O2 without -ffast-math: the arithmetic is evaluated as written.)
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): closed-form uniform-pairing BdG
 * spectrum, prescribed-spectrum matrices, N<=4 characteristic polynomial, closed-form
 * tridiagonals (1-2-1 Toeplitz, Clement/Kac, Wilkinson), trace / Frobenius invariants,
 * Q^H H Q = T, long-double agreement, particle-hole symmetry.  Nothing here is
 * "parity unpinned".
 */
#include <complex.h>
#include <float.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define REAL double
#define CPLX double _Complex
#define FN(x) x##_d
#define R_HYPOT hypot
#define R_FABS fabs
#define R_SQRT sqrt
#define R_COPYSIGN copysign
#define R_EPS DBL_EPSILON
#include "oracle_eigh_impl.inc"
#undef REAL
#undef CPLX
#undef FN
#undef R_HYPOT
#undef R_FABS
#undef R_SQRT
#undef R_COPYSIGN
#undef R_EPS

#define REAL long double
#define CPLX long double _Complex
#define FN(x) x##_ld
#define R_HYPOT hypotl
#define R_FABS fabsl
#define R_SQRT sqrtl
#define R_COPYSIGN copysignl
#define R_EPS LDBL_EPSILON
#include "oracle_eigh_impl.inc"

int oracle_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
