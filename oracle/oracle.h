/* oracle.h -- CPU oracle for the direct algebraic CT path of arXiv 2412.07631.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code with
 * paper_2412_07631_b200/csrc (the CUDA path) and neither includes the other.
 *
 * What it is: the textbook unblocked Householder QR, reflector-by-reflector Q^T b and scalar
 * back-substitution -- the plain definition of what PAPER.md Eq. 2-3 (L41-48) compute -- in
 * double (f64) and single (f32) precision, all arithmetic in the working type.
 * Pins (tests/test_oracle_pins.py, tests/golden/): hand-computed 3x2 case, triangular and
 * [I; mu I] closed forms, Gram-Schmidt brute force, |diag R| = diag chol(A^T A), orthogonality,
 * exact recovery, normal equations, T^{-1} = striu(V^T V) + diag(1/tau); the transposed substitution by the
 * semi-normal equations R^T R x = A^T b and closed forms.  Parity unpinned: none.
 */
#ifndef CT_ORACLE_H
#define CT_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
int     oracle_qr_f64(double *A, int64_t m, int64_t n, int64_t lda, double *tau);
int     oracle_qr_f32(float *A, int64_t m, int64_t n, int64_t lda, float *tau);
int     oracle_apply_qt_f64(const double *A, int64_t m, int64_t n, int64_t lda, const double *tau, double *B, int64_t ldb, int64_t S);
int     oracle_apply_qt_f32(const float *A, int64_t m, int64_t n, int64_t lda, const float *tau, float *B, int64_t ldb, int64_t S);
int     oracle_apply_q_f64(const double *A, int64_t m, int64_t n, int64_t lda, const double *tau, double *B, int64_t ldb, int64_t S);
int     oracle_apply_q_f32(const float *A, int64_t m, int64_t n, int64_t lda, const float *tau, float *B, int64_t ldb, int64_t S);
int64_t oracle_backsub_f64(const double *A, int64_t n, int64_t lda, const double *C, int64_t ldc, int64_t S, double *X, int64_t ldx);
int64_t oracle_backsub_f32(const float *A, int64_t n, int64_t lda, const float *C, int64_t ldc, int64_t S, float *X, int64_t ldx);
int64_t oracle_backsub_t_f64(const double *A, int64_t n, int64_t lda, const double *C, int64_t ldc, int64_t S, double *Y, int64_t ldy);
int64_t oracle_backsub_t_f32(const float *A, int64_t n, int64_t lda, const float *C, int64_t ldc, int64_t S, float *Y, int64_t ldy);
int     oracle_larft_f64(const double *A, int64_t m, int64_t lda, const double *tau, int64_t j0, int64_t nb, double *T, int64_t ldt);
int     oracle_larft_f32(const float *A, int64_t m, int64_t lda, const float *tau, int64_t j0, int64_t nb, float *T, int64_t ldt);
int     oracle_num_threads(void);
void    oracle_set_num_threads(int nthreads);
#ifdef __cplusplus
}
#endif
#endif
