"""B200-native dense Householder QR + batched solve for direct algebraic CT (arXiv 2412.07631).

Product path = ``libctqr.so`` (hand-written sm_100a kernels behind the C-ABI of include/ctqr.h)
plus the thin ctypes binding re-exported here.  ``workload`` holds the seeded input generators
(no method arithmetic).  Nothing in this package imports ``oracle/``.
"""
from .binding import (CtqrError, Factor, F32, F64, ct_qr_factor, ct_qr_solve, ct_qr_apply_qt,  # noqa: F401
                      ct_qr_trsm, ct_qr_trsm_t, ct_qr_solve_refined, ct_qr_get_R, ct_qr_get_V, ct_qr_get_T, ct_qr_get_tau, ct_qr_gemm, ct_qr_vtc_noalloc,
                      ct_qr_peak_probe, ct_qr_save, ct_qr_load, ct_qr_trim_cache, colmajor_from_numpy, numpy_from_colmajor, lib)
