/* ctqr.h -- C-ABI of the B200-native dense Householder QR + batched solve for direct
 * algebraic CT reconstruction (arXiv 2412.07631; PAPER.md in the reference mount).
 *
 * What the library computes (section 2):
 *   Eq. 2   A = Q R          once per scanner geometry       -> ct_qr_factor
 *   Eq. 3   X = R^{-1}(Q^T B) for a batch of S sinograms     -> ct_qr_solve
 * Q is kept implicit as Householder reflectors in compact-WY blocks (V_k, T_k), R^{-1} is
 * never formed (L48).  The in-core LAPACK analogues named by the paper are dgeqrf, dormqr
 * (printed "dormar") and dtrsm (L52); the out-of-core tiling mirrors section 2.2 (L54-77).
 *
 * Conventions
 *   - All matrices are column-major, leading dimensions in ELEMENTS.
 *   - dtype applies to A, B, X, V, T, R alike (no mixed precision in the product path).
 *   - Every pointer argument says whether it is a DEVICE pointer, a HOST pointer, or EITHER
 *     (detected with cudaPointerGetAttributes; host memory may be pinned or pageable).
 *   - Return value: 0 = success; negative -i = the i-th argument (1-based) is invalid;
 *     positive = runtime failure (CTQR_ERR_*).  Nothing aborts, nothing throws across the
 *     ABI.  ct_qr_last_error() returns a thread-local message for the last non-zero return.
 *   - Calls are synchronous: on return all device work they enqueued has completed.
 *   - A handle is not thread-safe; distinct handles may be used from distinct threads.
 *   - Global state: the thread-local last-error string, and ONE process-wide, mutex-protected cache of freed small
 *     device blocks (the ~20 per-handle buffers: T, tau, workspaces; each <= 256 MiB, <= 1 GiB kept in total), so
 *     that a service which factors or reloads one geometry after another does not pay cudaMalloc / cudaFree per
 *     handle.  The cache is emptied automatically when a device allocation fails, and on request by
 *     ct_qr_trim_cache(); matrix storage is never cached.
 *   - There is NO CPU fallback: without a CUDA device every compute entry point returns
 *     CTQR_ERR_CUDA.
 *
 * Householder convention (reading R4, LAPACK-like): H_j = I - tau_j v_j v_j^T,
 * v_j[j] = 1, beta_j = -sign(alpha_j) ||x_j||_2 with sign(0) = +1, R_jj = beta_j; a column
 * whose sub-diagonal part is exactly zero gets tau_j = 0.
 */
#ifndef CTQR_H
#define CTQR_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ctqr_handle_s* ctqr_handle_t;   /* opaque; owns T, tau, diag(R) blocks, plan, and
                                                  (unless in_place) the V\R storage */

typedef enum { CTQR_F32 = 0, CTQR_F64 = 1 } ctqr_dtype_t;

typedef enum {
    CTQR_OK = 0,
    CTQR_ERR_CUDA = 1,      /* a CUDA runtime call failed, or no device */
    CTQR_ERR_NOMEM = 2,     /* device or host allocation failed / budget too small */
    CTQR_ERR_IO = 3,        /* file tier read/write failed */
    CTQR_ERR_SINGULAR = 4,  /* some R_jj == 0 at solve time (stats.singular_col = first j) */
    CTQR_ERR_STATE = 5      /* handle is not in a state that allows the call */
} ctqr_status_t;

/* Options for ct_qr_factor.  Zero-initialise for defaults. */
typedef struct {
    int32_t nb;                 /* panel width; 0 = default (128). A multiple of ib, at most 128 (the tensor-core
                                   kernels, the merged two-panel update and the fused small-S solve are built
                                   for 128; smaller values exist for the blocking-invariance tests). */
    int32_t ib;                 /* inner (register-resident) panel width: 8, 16 or 32; 0 = default (32) */
    int32_t lookahead;          /* 0 = off, 1 = factor panel k+1 while the rest of update k runs; -1 = default */
    int32_t in_place;           /* 1: A (device) is overwritten and must outlive the handle.
                                   0: A is read-only; the handle owns a copy. */
    int64_t device_budget_bytes;/* 0 = unlimited (in-core if it fits). >0 caps the device bytes used
                                   for matrix tiles: forces the out-of-core path when m*n*w exceeds it */
    int32_t gemm_impl;          /* 0 = default: tensor cores (fp64: mma.sync m8n8k4 = DMMA.8x8x4; fp32: 3xTF32 split on
                                   tcgen05.mma kind::tf32 with TMEM accumulators, warp-level mma.sync tf32 for shapes the
                                   tcgen05 kernel does not take); 1 = SIMT cross-check kernels (DFMA / FFMA), which also
                                   switches the fused small-S solve kernels off */
    int32_t profile;            /* 1: CUDA-event time every trailing-update contraction launch (stats.vtc_*, upd_*) */
    const char* file_path;      /* optional file-backed tier: path of a file holding the column-major m x n matrix
                                   (leading dimension lda, offset 0).  The A argument is then ignored (may be NULL);
                                   the file is mapped read-write, factored out of core through the page cache and
                                   overwritten with the factor, which ct_qr_solve streams from it.  NULL = none */
    void* stream;               /* cudaStream_t the caller's data is ordered on (NULL = legacy default) */
    int64_t lower_bandwidth;    /* 0 = dense.  kl > 0: the caller promises A(i, j) == 0 for i - j > kl (for the Tikhonov-
                                   augmented [A0; sqrt(lambda) I] with m0 rows of A0: kl = m0).  Householder QR keeps that
                                   profile (v_j ends at row kl + j), so every panel and trailing update stops at row
                                   kl + (last column of the block) and the factorisation costs sum_j 4 r_j (n-j-1) flop,
                                   r_j = min(m, kl+j+1) - j, instead of 2mn^2 - 2n^3/3.  The result
                                   is the same factor (the skipped work is arithmetic on exact zeros).  The promise is
                                   checked on the device BEFORE anything is overwritten (-6 if violated, naming the
                                   first offending column; the input -- device matrix, host matrix or file -- is then
                                   untouched): in core on the resident matrix, out of core by one extra streamed pass
                                   over the part of the host matrix below the band.  Out of core it also shortens the
                                   reflector panels streamed over the host link. */
    int32_t trsm_exact;         /* 0 = default: the diagonal tasks X_i = R_ii^{-1} C_i of the blocked TRSM
                                   multiply by the explicitly inverted nb x nb DIAGONAL block (inverted once per handle;
                                   the off-diagonal part of R^{-1} is never formed, L48).  That is only conditionally
                                   backward stable, so the library falls back to back-substitution by itself when a
                                   diagonal block looks ill-conditioned (stats.diag_block_cond > 1/sqrt(eps)).
                                   1 = always back-substitution (trsm_diag_kernel; also disables the fused S <= 8 TRSM). */
    int32_t solve_pairs;        /* 0 = by size (default): large batches apply Q^T two panels at a time (S >= 1024, or S >= 512
                                   when m >= 65536) and the TRSM two diagonal blocks at a time (S >= 512, n >= 32768), where
                                   that was measured to win; 1 = whenever the batch has at least 256 right-hand sides (used
                                   by the tests to reach those paths at oracle-sized problems); -1 = never */
} ctqr_options_t;

/* Per-handle statistics (CUDA-event timed, milliseconds). */
typedef struct {
    int64_t m, n;
    int32_t nb, ib, n_panels, n_superpanels;   /* n_superpanels == 1 when in-core */
    int32_t out_of_core, singular_col;         /* singular_col = -1 when none */
    double factor_ms;          /* whole ct_qr_factor device time */
    double panel_ms;           /* opt->profile: factor_ms minus update_ms (panel chains a1 + a2, narrow updates, T^T W) */
    double update_ms;          /* opt->profile: time inside the two contractions of the trailing updates (a3) */
    double solve_ms;           /* last ct_qr_solve device time */
    double apply_qt_ms;        /* last Q^T B part (a6) */
    double trsm_ms;            /* last triangular solve part (a7) */
    double h2d_bytes, d2h_bytes;   /* bytes moved over the host link by the last factor / solve */
    double factor_flops;       /* 2 m n^2 - 2 n^3 / 3 (the dense count, whatever was run) */
    int64_t kernel_launches;   /* kernels launched by the last factor or solve call */
    /* opt->profile only: the two contractions of every trailing update (a3) of the last factor,
     * each launch bracketed by CUDA events on the stream it runs on.
     *   vtc: W = V_k^T C  (K = m_k),   upd: C <- C - V_k W  (K = nb);  flops = 2*m_k*nb_k*n_c each. */
    double vtc_ms, vtc_flops;  int64_t vtc_launches;
    double upd_ms, upd_flops;  int64_t upd_launches;
    int64_t lower_bandwidth;   /* the band promise the factorisation used (0 = dense) */
    double factor_flops_performed;   /* = factor_flops when dense; the banded count of opt->lower_bandwidth otherwise */
    /* out of core only (last factor or solve call): copy_busy_ms = sum of the durations of all host<->device tile copies
     * (H2D and D2H streams added up); copy_exposed_ms = time the compute stream spent stalled waiting for one of them,
     * i.e. the part of the copies that compute did NOT hide (includes the first load and the last write-back). */
    double copy_busy_ms, copy_exposed_ms;
    double diag_block_cond;    /* max over diagonal blocks of max|R_jj| / min|R_jj| (set by the first solve; 0 before) */
    int32_t trsm_exact;        /* 0: inverted diagonal blocks; 1: back-substitution by option; 2: forced by the guard */
    int32_t apply_qt_path;     /* last Q^T B: 0 = one larfb per panel; 1 = fused small-S kernel (one cooperative launch);
                                  2 = pipelined, TMA-fed small-S kernel (solve_small2.cuh); 3 = streamed (out of core);
                                  4 = medium-S kernel (fp64, 8 < S <= 64 where shared memory allows, solve_mid.cuh);
                                  5 = two panels per larfb (S >= 1024, or S >= 512 when m >= 65536: the 256-wide blocks of the factorisation) */
} ctqr_stats_t;

/* Eq. 2: Householder QR of the m x n matrix A (m >= n >= 1, lda >= m).
 *   A       EITHER. Device pointer: in-core factorisation (in place if opt->in_place, else
 *           on a copy owned by the handle).  Host pointer (pinned preferred): the matrix is
 *           staged through device memory; when m*n*w exceeds opt->device_budget_bytes (or
 *           free device memory) the out-of-core path streams column super-panels from the
 *           host buffer, which is then overwritten with the factor (always in place).
 *   out     receives the handle on success; untouched on failure.
 * On success the factor is: V (unit lower trapezoid, explicit 0/1 on and above the
 * diagonal inside each diagonal block), tau[n], T_k (nb x nb upper) per panel, R
 * (off-diagonal blocks inside the matrix storage, diagonal blocks owned by the handle). */
int ct_qr_factor(void* A, int64_t m, int64_t n, int64_t lda, ctqr_dtype_t dtype,
                 const ctqr_options_t* opt, ctqr_handle_t* out);

/* Eq. 3: X = R^{-1} (Q^T B) for S right-hand sides.
 *   B   EITHER, m x S, ldb >= m, read-only.   X   EITHER, n x S, ldx >= n, written.
 * Returns CTQR_ERR_SINGULAR if some R_jj == 0. */
int ct_qr_solve(ctqr_handle_t h, const void* B, int64_t ldb, int64_t S, void* X, int64_t ldx);

/* First half of Eq. 3 alone: C <- Q^T C in place (C EITHER, m x S, ldc >= m). */
int ct_qr_apply_qt(ctqr_handle_t h, void* C, int64_t ldc, int64_t S);

/* Second half of Eq. 3 alone (blocked TRSM, task list PAPER.md:L62-73): X <- R^{-1} C[0:n,:].
 * C EITHER (n x S used, ldc >= n, read-only), X EITHER (n x S, ldx >= n). */
int ct_qr_trsm(ctqr_handle_t h, const void* C, int64_t ldc, int64_t S, void* X, int64_t ldx);

/* The transposed half: X <- R^{-T} C (forward substitution with R^T, the task list of PAPER.md:L62-73 read for the
 * transposed factor).  C EITHER (n x S, ldc >= n, read-only), X EITHER (n x S, ldx >= n).  In-core factors only
 * (CTQR_ERR_STATE otherwise).  Used by ct_qr_solve_refined; R^{-1} R^{-T} g solves the normal equations A^T A d = g. */
int ct_qr_trsm_t(ctqr_handle_t h, const void* C, int64_t ldc, int64_t S, void* X, int64_t ldx);

/* Least-squares solve with fp64 iterative refinement on top of a working-precision factor (
 * the paper's subject is the fp32 / fp64 quality gap, Table 3):
 *     x_0 = R^{-1}(Q^T b)  in the handle's precision (Eq. 3), then, in fp64,
 *     r = b - A x,  g = A^T r,  x <- x + R^{-1}(R^{-T} g)      (corrected semi-normal equations)
 * with the two triangular solves in the handle's precision on g scaled to max|g| = 1 per slice.  The fixed point
 * is the exact normal-equations solution A^T(b - A x) = 0 of the fp64 operator, also for inconsistent (noisy) b;
 * the error contracts by about cond(A)^2 * eps(handle precision) per sweep.  With an fp32 handle this gives
 * fp64-quality reconstructions from a factor that took half the memory and less than half the time.
 * The operator A (m x n, the matrix that was factored, in fp64) is given EITHER as a CSR pair (A and its transpose
 * At, 0-based, int64 row pointers, int32 column indices, fp64 values; every array EITHER host or device) OR as a
 * dense column-major fp64 DEVICE matrix A_dense (leading dimension lda); pass NULL for the form not used.
 *   B   EITHER, fp64, m x S, ldb >= m.     X   EITHER, fp64, n x S, ldx >= n.
 *   max_iters  refinement sweeps at most (0 = x_0 only);  tol > 0 stops early when max over slices of
 *   ||correction||_2 / ||x||_2 <= tol.   info (required) receives what happened.
 * Errors: argument errors as -i; CTQR_ERR_STATE for an out-of-core handle or a NaN; CTQR_ERR_SINGULAR; CTQR_ERR_CUDA. */
#define CTQR_REFINE_MAX_ITERS 16
typedef struct {
    int64_t m, n, nnz;
    const int64_t* rowptr;     /* m + 1 entries */
    const int32_t* colidx;     /* nnz entries, each < n */
    const double* vals;        /* nnz entries */
} ctqr_csr_t;
typedef struct {
    int32_t iters_done, converged;                 /* sweeps performed; 1 if tol was reached */
    double correction[CTQR_REFINE_MAX_ITERS];      /* per sweep: max over slices of ||d||_2 / ||x||_2 */
    double gradient[CTQR_REFINE_MAX_ITERS];        /* per sweep: max over slices of ||A^T (b - A x)||_2 BEFORE the correction */
    double ms_total, ms_initial_solve, ms_residual, ms_correction;   /* CUDA-event times of the call and its three parts */
} ctqr_refine_info_t;
int ct_qr_solve_refined(ctqr_handle_t h, const ctqr_csr_t* A, const ctqr_csr_t* At, const void* A_dense, int64_t lda,
                        const double* B, int64_t ldb, int64_t S, double* X, int64_t ldx,
                        int32_t max_iters, double tol, ctqr_refine_info_t* info);

/* Accessors (R, V, T, tau may be HOST or DEVICE pointers; output is dense column-major). */
int ct_qr_get_R(ctqr_handle_t h, void* R, int64_t ldr);                  /* n x n upper; strictly lower part zeroed */
int ct_qr_get_V(ctqr_handle_t h, int64_t j0, int64_t ncols, void* V, int64_t ldv); /* m x ncols, unit lower trapezoid */
int ct_qr_get_T(ctqr_handle_t h, int64_t panel, void* T, int64_t ldt);   /* nb_k x nb_k upper (last panel may be narrower) */
int ct_qr_get_tau(ctqr_handle_t h, void* tau);                           /* n values */
int ct_qr_get_stats(ctqr_handle_t h, ctqr_stats_t* s);
int ct_qr_dtype(ctqr_handle_t h);                                        /* CTQR_F32 / CTQR_F64; -1 when h is NULL */
void ct_qr_destroy(ctqr_handle_t h);

/* Factor persistence ("factor once per geometry, reuse for every batch of slices").
 * ct_qr_save writes the whole factor of a factored handle (V\R storage, T_k, diagonal R blocks, tau;
 * in-core or out-of-core handle alike) to `path` (created / truncated; removed again on failure).
 * The file is self-describing (dtype, m, n, nb, ib, the lower_bandwidth the factor was computed under, which the
 * solves of a loaded handle keep using) and holds m*n*w bytes plus O(n*nb*w).
 * ct_qr_load builds a handle from such a file without factoring: the factor is read into device
 * memory when it fits opt->device_budget_bytes (0 = free device memory), otherwise the file is mapped
 * read-only and ct_qr_solve streams its panels through the page cache (out-of-core solve, row a5).
 * Of `opt` only device_budget_bytes, gemm_impl and stream are used (nb / ib come from the file); opt
 * may be NULL.  A loaded handle supports every call a factored one does; its factor_ms is 0.
 * Errors: CTQR_ERR_IO (cannot create/open, short write/read, bad magic/header, truncated file),
 * CTQR_ERR_NOMEM, CTQR_ERR_CUDA; *out is untouched on failure. */
int ct_qr_save(ctqr_handle_t h, const char* path);
int ct_qr_load(const char* path, const ctqr_options_t* opt, ctqr_handle_t* out);

/* Releases the process-wide cache of freed small device blocks (see "Global state" above); returns the bytes freed.
 * Safe at any time from any thread; blocks in use by live handles are not affected. */
int64_t ct_qr_trim_cache(void);

const char* ct_qr_strerror(int code);
const char* ct_qr_last_error(void);
int ct_qr_version(void);

/* Kernel-level entry points used by the parity tests (SURVEY.md test rung T2) and by the
 * micro-benchmarks of bench.py.  All pointers DEVICE.
 *   ct_qr_gemm: C <- alpha*op(A)*B + beta*C with op(A) = A^T when trans_a (A is K x M) else A
 *   (A is M x K); B is K x N; impl 0 = default kernel for the dtype, 1 = SIMT kernel, 2 = (fp32, op(A) = A only) the
 *   TMA-fed tcgen05 kernel with operands pre-split into TF32 hi / lo, as the two-panel trailing update uses it.
 *   ct_qr_peak_probe: runs a register-resident FMA/MMA loop and returns achieved TFLOP/s
 *   (kind 0 = FFMA fp32, 1 = DFMA fp64, 2 = DMMA m8n8k4 fp64). */
int ct_qr_gemm(int trans_a, int64_t M, int64_t N, int64_t K, double alpha, const void* A, int64_t lda,
               const void* B, int64_t ldb, double beta, void* C, int64_t ldc, ctqr_dtype_t dtype, int impl);
int ct_qr_peak_probe(int kind, int iters, double* tflops, double* ms);
/* same loop with `threads` per CTA (multiple of 32, <= 256) and `ctas_per_sm` CTAs per SM: how many
 * resident warps the pipe needs to reach its peak (ct_qr_peak_probe = 256 threads x 8 CTAs). */
int ct_qr_peak_probe_cfg(int kind, int iters, int threads, int ctas_per_sm, double* tflops, double* ms);

/* ---- allocation-free entry point -----------------------------------------------------------------------------
 * ct_qr_vtc_noalloc: W <- V^T C, the split-K product that opens the block-reflector application
 * C <- (I - V T V^T)^T C (C = Q^T B is applied without building Q, "dormqr"; SURVEY.md 8a rows
 * a3 / a6), for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it.  Same result as ct_qr_gemm(trans_a = 1, M, N, K, 1, V, ldv, C, ldc, 0, W, ldw, dtype, 0) up to
 * the summation order.
 *   V: K x M, column-major, leading dimension ldv >= max(K, 1)   (device pointer, read-only)
 *   C: K x N, column-major, leading dimension ldc >= max(K, 1)   (device pointer, read-only)
 *   W: M x N, column-major, leading dimension ldw >= M           (device pointer, overwritten; must not alias V, C)
 *   stream: a cudaStream_t passed as void*; NULL = the default stream.  The call enqueues two kernels on it and
 *           returns without synchronising; the caller owns all three buffers and keeps them alive until they ran.
 * The partial tiles of the split live in a file-scope device array of CTQR_NOALLOC_SCRATCH_BYTES that every GPU
 * which loads the library holds until the process exits; the call never calls cudaMalloc, cudaFree or an allocating
 * library routine (the first call per device fetches the array's address with cudaGetSymbolAddress and loads the
 * kernels: make one call before starting a graph capture).
 * Limit: ceil(M/64) * ceil(N/64) * 64 * 64 * sizeof(element) <= CTQR_NOALLOC_SCRATCH_BYTES, i.e. at most 512 output
 * tiles in fp64 and 1024 in fp32 (e.g. M = 128, N <= 16 384 in fp64); K is unlimited.  Larger sizes are refused with
 * CTQR_ERR_NOMEM and a message naming the limit; nothing is enqueued.
 * All calls share the one array: calls whose kernels may overlap on the GPU (different streams without a
 * dependency, or several host threads) RACE on it; calls on one stream are ordered.  The array keeps the last call's
 * tiles, and nothing in it needs to start at zero: every slot a call reads it has written in full first.
 * Deterministic (fixed split, sums in split order).  Errors: -i for the i-th argument (1-based; host pointers are
 * refused as -4), CTQR_ERR_NOMEM beyond the limit, CTQR_ERR_CUDA. */
#define CTQR_NOALLOC_SCRATCH_BYTES (16u << 20)
int ct_qr_vtc_noalloc(int64_t M, int64_t N, int64_t K, const void* V, int64_t ldv, const void* C, int64_t ldc,
                      void* W, int64_t ldw, ctqr_dtype_t dtype, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CTQR_H */
