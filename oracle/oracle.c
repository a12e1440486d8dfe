/* oracle.c -- see oracle.h.  TEST INFRASTRUCTURE ONLY.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC oracle.c -o liboracle.so -lm
 * (-ffp-contract=off: no fused multiply-add, so every product and sum rounds once in REAL.) */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "oracle.h"

#define REAL double
#define SUF f64
#define SQRT sqrt
#include "oracle_impl.inc"
#undef REAL
#undef SUF
#undef SQRT

#define REAL float
#define SUF f32
#define SQRT sqrtf
#include "oracle_impl.inc"
#undef REAL
#undef SUF
#undef SQRT

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
}
