"""ctypes binding of ``libctqr.so`` (include/ctqr.h) -- argument marshalling only.

Every step of the hot path (Eq. 2-3) runs inside the CUDA library; this
module only turns torch tensors / numpy arrays into (pointer, leading dimension) pairs.
There is no CPU fallback: if the shared object is missing or no CUDA device is present the
calls raise ``CtqrError``.

Layout convention: the library is column-major.  A torch tensor ``At`` of shape (n, lda)
that is row-major contiguous IS the column-major m x n matrix with leading dimension lda
(m <= lda); the helpers below therefore take / return "transposed-view" tensors:
``colmajor_from_numpy`` gives such a tensor for a numpy (m, n) array.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libctqr.so")
_lib = None

F32, F64 = 0, 1


class CtqrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ctqr error {code}: {msg}")
        self.code = code


class Options(ctypes.Structure):
    _fields_ = [("nb", ctypes.c_int32), ("ib", ctypes.c_int32), ("lookahead", ctypes.c_int32),
                ("in_place", ctypes.c_int32), ("device_budget_bytes", ctypes.c_int64),
                ("gemm_impl", ctypes.c_int32), ("profile", ctypes.c_int32),
                ("file_path", ctypes.c_char_p), ("stream", ctypes.c_void_p),
                ("lower_bandwidth", ctypes.c_int64), ("trsm_exact", ctypes.c_int32), ("solve_pairs", ctypes.c_int32)]


class Stats(ctypes.Structure):
    _fields_ = [("m", ctypes.c_int64), ("n", ctypes.c_int64),
                ("nb", ctypes.c_int32), ("ib", ctypes.c_int32), ("n_panels", ctypes.c_int32),
                ("n_superpanels", ctypes.c_int32), ("out_of_core", ctypes.c_int32),
                ("singular_col", ctypes.c_int32),
                ("factor_ms", ctypes.c_double), ("panel_ms", ctypes.c_double),
                ("update_ms", ctypes.c_double), ("solve_ms", ctypes.c_double),
                ("apply_qt_ms", ctypes.c_double), ("trsm_ms", ctypes.c_double),
                ("h2d_bytes", ctypes.c_double), ("d2h_bytes", ctypes.c_double),
                ("factor_flops", ctypes.c_double), ("kernel_launches", ctypes.c_int64),
                ("vtc_ms", ctypes.c_double), ("vtc_flops", ctypes.c_double), ("vtc_launches", ctypes.c_int64),
                ("upd_ms", ctypes.c_double), ("upd_flops", ctypes.c_double), ("upd_launches", ctypes.c_int64),
                ("lower_bandwidth", ctypes.c_int64), ("factor_flops_performed", ctypes.c_double),
                ("copy_busy_ms", ctypes.c_double), ("copy_exposed_ms", ctypes.c_double),
                ("diag_block_cond", ctypes.c_double), ("trsm_exact", ctypes.c_int32), ("apply_qt_path", ctypes.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


REFINE_MAX_ITERS = 16


class Csr(ctypes.Structure):
    _fields_ = [("m", ctypes.c_int64), ("n", ctypes.c_int64), ("nnz", ctypes.c_int64),
                ("rowptr", ctypes.c_void_p), ("colidx", ctypes.c_void_p), ("vals", ctypes.c_void_p)]


class RefineInfo(ctypes.Structure):
    _fields_ = [("iters_done", ctypes.c_int32), ("converged", ctypes.c_int32),
                ("correction", ctypes.c_double * REFINE_MAX_ITERS), ("gradient", ctypes.c_double * REFINE_MAX_ITERS),
                ("ms_total", ctypes.c_double), ("ms_initial_solve", ctypes.c_double),
                ("ms_residual", ctypes.c_double), ("ms_correction", ctypes.c_double)]


_P, _I64, _I = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
EXPORTS = {
    "ct_qr_factor": ([_P, _I64, _I64, _I64, _I, ctypes.POINTER(Options), ctypes.POINTER(_P)], _I),
    "ct_qr_solve": ([_P, _P, _I64, _I64, _P, _I64], _I),
    "ct_qr_apply_qt": ([_P, _P, _I64, _I64], _I),
    "ct_qr_trsm": ([_P, _P, _I64, _I64, _P, _I64], _I),
    "ct_qr_trsm_t": ([_P, _P, _I64, _I64, _P, _I64], _I),
    "ct_qr_solve_refined": ([_P, ctypes.POINTER(Csr), ctypes.POINTER(Csr), _P, _I64, _P, _I64, _I64, _P, _I64,
                             ctypes.c_int32, ctypes.c_double, ctypes.POINTER(RefineInfo)], _I),
    "ct_qr_get_R": ([_P, _P, _I64], _I),
    "ct_qr_get_V": ([_P, _I64, _I64, _P, _I64], _I),
    "ct_qr_get_T": ([_P, _I64, _P, _I64], _I),
    "ct_qr_get_tau": ([_P, _P], _I),
    "ct_qr_get_stats": ([_P, ctypes.POINTER(Stats)], _I),
    "ct_qr_destroy": ([_P], None),
    "ct_qr_save": ([_P, ctypes.c_char_p], _I),
    "ct_qr_load": ([ctypes.c_char_p, ctypes.POINTER(Options), ctypes.POINTER(_P)], _I),
    "ct_qr_dtype": ([_P], _I),
    "ct_qr_trim_cache": ([], _I64),
    "ct_qr_strerror": ([_I], ctypes.c_char_p),
    "ct_qr_last_error": ([], ctypes.c_char_p),
    "ct_qr_version": ([], _I),
    "ct_qr_gemm": ([_I, _I64, _I64, _I64, ctypes.c_double, _P, _I64, _P, _I64, ctypes.c_double,
                    _P, _I64, _I, _I], _I),
    "ct_qr_vtc_noalloc": ([_I64, _I64, _I64, _P, _I64, _P, _I64, _P, _I64, _I, _P], _I),
    "ct_qr_peak_probe": ([_I, _I, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)], _I),
    "ct_qr_peak_probe_cfg": ([_I, _I, _I, _I, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)], _I),
}


def lib():
    """Load libctqr.so (fails loudly when it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise CtqrError(-1, f"{LIB_PATH} not built; run `python -m paper_2412_07631_b200.build`")
        L = ctypes.CDLL(LIB_PATH)
        for name, (args, res) in EXPORTS.items():
            f = getattr(L, name)
            f.argtypes, f.restype = args, res
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        L = lib()
        msg = L.ct_qr_last_error().decode() or L.ct_qr_strerror(rc).decode()
        raise CtqrError(rc, msg)


def _code_of(x) -> int:
    import torch
    if isinstance(x, torch.Tensor):
        if x.dtype == torch.float64:
            return F64
        if x.dtype == torch.float32:
            return F32
    else:
        if x.dtype == np.float64:
            return F64
        if x.dtype == np.float32:
            return F32
    raise TypeError(f"ctqr supports float32/float64, got {x.dtype}")


def _ptr(x) -> int:
    import torch
    if isinstance(x, torch.Tensor):
        return x.data_ptr()
    return x.ctypes.data


def colmajor_from_numpy(a: np.ndarray, device="cuda", pin: bool = False):
    """(m, n) numpy array -> torch tensor of shape (n, m) whose memory is the column-major
    m x n matrix (lda = m)."""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(np.asarray(a).T))
    if device == "cpu":
        # always a fresh buffer: an out-of-core ct_qr_factor overwrites its host matrix in place
        return t.pin_memory() if pin else t.clone()
    return t.to(device)


def numpy_from_colmajor(t) -> np.ndarray:
    """Inverse of colmajor_from_numpy: (n, m) tensor -> (m, n) Fortran-ordered numpy array."""
    return np.asfortranarray(t.detach().cpu().numpy().T)


class Factor:
    """Handle of one factorisation A = QR (Eq. 2).  ``ct_qr_factor`` / ``ct_qr_solve`` are
    the module-level functions below; this class only keeps the handle alive."""

    def __init__(self, handle: int, m: int, n: int, code: int, keep=None):
        self._h, self.m, self.n, self.code = handle, m, n, code
        self._keep = keep          # the in-place A tensor must outlive the handle

    @property
    def torch_dtype(self):
        import torch
        return torch.float64 if self.code == F64 else torch.float32

    @property
    def np_dtype(self):
        return np.float64 if self.code == F64 else np.float32

    def stats(self) -> dict:
        s = Stats()
        _check(lib().ct_qr_get_stats(self._h, ctypes.byref(s)))
        return s.as_dict()

    def destroy(self):
        if self._h:
            lib().ct_qr_destroy(self._h)
            self._h = None
            self._keep = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def ct_qr_factor(A, m: int, n: int, lda: int | None = None, *, nb: int = 0, ib: int = 0,
                 lookahead: int = -1, in_place: bool = False, device_budget_bytes: int = 0,
                 gemm_impl: int = 0, profile: bool = False, stream=None, file_path: str | None = None,
                 dtype=None, lower_bandwidth: int = 0, trsm_exact: bool = False, solve_pairs: int = 0) -> Factor:
    """Eq. 2.  ``A``: torch tensor (device or pinned/pageable host) or numpy array whose MEMORY
    is the column-major m x n matrix with leading dimension ``lda`` (default m)."""
    code = _code_of(A) if A is not None else (F64 if np.dtype(dtype) == np.float64 else F32)
    lda = m if lda is None else lda
    o = Options(nb=nb, ib=ib, lookahead=lookahead, in_place=int(in_place),
                device_budget_bytes=device_budget_bytes, gemm_impl=gemm_impl, profile=int(profile),
                file_path=file_path.encode() if file_path else None, stream=stream,
                lower_bandwidth=lower_bandwidth, trsm_exact=int(trsm_exact), solve_pairs=int(solve_pairs))
    h = _P()
    _check(lib().ct_qr_factor(_ptr(A) if A is not None else None, m, n, lda, code, ctypes.byref(o), ctypes.byref(h)))
    return Factor(h, m, n, code, keep=A if in_place else None)


def ct_qr_trim_cache() -> int:
    """Release the library's process-wide cache of freed small device blocks; returns the bytes freed."""
    return int(lib().ct_qr_trim_cache())


def ct_qr_save(f: Factor, path: str) -> None:
    """Write the factor (V\\R storage, T_k, diagonal R blocks, tau) to ``path`` (reuse)."""
    _check(lib().ct_qr_save(f._h, os.fsencode(path)))


def ct_qr_load(path: str, *, device_budget_bytes: int = 0, gemm_impl: int = 0, stream=None) -> Factor:
    """Handle from a file written by ``ct_qr_save``; the solve streams the file when the factor
    exceeds ``device_budget_bytes`` (0 = free device memory)."""
    o = Options(lookahead=-1, device_budget_bytes=device_budget_bytes, gemm_impl=gemm_impl, stream=stream)
    h = _P()
    _check(lib().ct_qr_load(os.fsencode(path), ctypes.byref(o), ctypes.byref(h)))
    s = Stats()
    _check(lib().ct_qr_get_stats(h, ctypes.byref(s)))
    return Factor(h, s.m, s.n, lib().ct_qr_dtype(h))     # dtype, m, n are properties of the file


def ct_qr_solve(f: Factor, B, S: int, X, ldb: int | None = None, ldx: int | None = None):
    """Eq. 3.  B: column-major m x S (ldb default m), X: column-major n x S (ldx default n)."""
    _check(lib().ct_qr_solve(f._h, _ptr(B), f.m if ldb is None else ldb, S, _ptr(X), f.n if ldx is None else ldx))
    return X


def ct_qr_apply_qt(f: Factor, C, S: int, ldc: int | None = None):
    _check(lib().ct_qr_apply_qt(f._h, _ptr(C), f.m if ldc is None else ldc, S))
    return C


def ct_qr_trsm(f: Factor, C, S: int, X, ldc: int | None = None, ldx: int | None = None):
    _check(lib().ct_qr_trsm(f._h, _ptr(C), f.n if ldc is None else ldc, S, _ptr(X), f.n if ldx is None else ldx))
    return X


def ct_qr_trsm_t(f: Factor, C, S: int, X, ldc: int | None = None, ldx: int | None = None):
    """X <- R^{-T} C (transposed half of the normal-equations solve)."""
    _check(lib().ct_qr_trsm_t(f._h, _ptr(C), f.n if ldc is None else ldc, S, _ptr(X), f.n if ldx is None else ldx))
    return X


def _csr_struct(a, keep: list) -> Csr:
    """scipy.sparse CSR matrix (any index dtype) -> ctqr_csr_t over host arrays that `keep` holds alive."""
    rp = np.ascontiguousarray(a.indptr, dtype=np.int64)
    ci = np.ascontiguousarray(a.indices, dtype=np.int32)
    va = np.ascontiguousarray(a.data, dtype=np.float64)
    keep += [rp, ci, va]
    return Csr(m=a.shape[0], n=a.shape[1], nnz=int(a.nnz), rowptr=rp.ctypes.data, colidx=ci.ctypes.data, vals=va.ctypes.data)


def ct_qr_solve_refined(f: Factor, B, S: int, X, *, A_csr=None, At_csr=None, A_dense=None, lda: int | None = None,
                        max_iters: int = 3, tol: float = 0.0, ldb: int | None = None, ldx: int | None = None) -> dict:
    """fp64 solution from a working-precision factor by iterative refinement (include/ctqr.h).  The fp64 operator is
    either ``A_csr`` (scipy CSR, m x n; ``At_csr`` defaults to its transpose) or ``A_dense`` (device tensor whose memory
    is the column-major m x n fp64 matrix).  B, X: fp64, column-major m x S / n x S.  Returns the info block as a dict."""
    keep: list = []
    pa = pat = None
    if A_csr is not None:
        a = A_csr.tocsr()
        at = (At_csr if At_csr is not None else a.T).tocsr()
        a.sort_indices(); at.sort_indices()
        sa, sat = _csr_struct(a, keep), _csr_struct(at, keep)
        pa, pat = ctypes.byref(sa), ctypes.byref(sat)
    info = RefineInfo()
    _check(lib().ct_qr_solve_refined(f._h, pa, pat, _ptr(A_dense) if A_dense is not None else None,
                                     (f.m if lda is None else lda), _ptr(B), f.m if ldb is None else ldb, S,
                                     _ptr(X), f.n if ldx is None else ldx, max_iters, tol, ctypes.byref(info)))
    k = info.iters_done
    return {"iters_done": k, "converged": bool(info.converged), "correction": list(info.correction)[:k],
            "gradient": list(info.gradient)[:k], "ms_total": info.ms_total, "ms_initial_solve": info.ms_initial_solve,
            "ms_residual": info.ms_residual, "ms_correction": info.ms_correction}


def ct_qr_get_R(f: Factor) -> np.ndarray:
    R = np.zeros((f.n, f.n), dtype=f.np_dtype, order="F")
    _check(lib().ct_qr_get_R(f._h, _ptr(R), f.n))
    return R


def ct_qr_get_V(f: Factor, j0: int = 0, ncols: int | None = None) -> np.ndarray:
    ncols = f.n - j0 if ncols is None else ncols
    V = np.zeros((f.m, ncols), dtype=f.np_dtype, order="F")
    _check(lib().ct_qr_get_V(f._h, j0, ncols, _ptr(V), f.m))
    return V


def ct_qr_get_T(f: Factor, panel: int) -> np.ndarray:
    st = f.stats()
    nbw = min(st["nb"], f.n - panel * st["nb"])
    T = np.zeros((nbw, nbw), dtype=f.np_dtype, order="F")
    _check(lib().ct_qr_get_T(f._h, panel, _ptr(T), nbw))
    return T


def ct_qr_get_tau(f: Factor) -> np.ndarray:
    tau = np.zeros(f.n, dtype=f.np_dtype)
    _check(lib().ct_qr_get_tau(f._h, _ptr(tau)))
    return tau


def ct_qr_gemm(trans_a: bool, M: int, N: int, K: int, alpha: float, A, lda: int, B, ldb: int,
               beta: float, C, ldc: int, impl: int = 0):
    """Kernel-level test hook (device tensors): C <- alpha op(A) B + beta C, column-major."""
    _check(lib().ct_qr_gemm(int(trans_a), M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(C), ldc,
                            _code_of(C), impl))
    return C


def ct_qr_vtc_noalloc(M: int, N: int, K: int, V, ldv: int, C, ldc: int, W, ldw: int, stream=None):
    """W <- V^T C without any allocation (device tensors, column-major; scratch is a fixed device array of the
    library, see include/ctqr.h for the size limit and the sharing rule).  ``stream``: a torch.cuda.Stream or None
    (the default stream).  Asynchronous."""
    st = ctypes.c_void_p(stream.cuda_stream) if stream is not None else None
    _check(lib().ct_qr_vtc_noalloc(M, N, K, _ptr(V), ldv, _ptr(C), ldc, _ptr(W), ldw, _code_of(W), st))
    return W


def ct_qr_peak_probe(kind: int, iters: int = 4096, threads: int = 256, ctas_per_sm: int = 8):
    """Measured register-resident peak: kind 0 FFMA, 1 DFMA, 2 DMMA.  Returns (TFLOP/s, ms)."""
    tf, ms = ctypes.c_double(), ctypes.c_double()
    _check(lib().ct_qr_peak_probe_cfg(kind, iters, threads, ctas_per_sm, ctypes.byref(tf), ctypes.byref(ms)))
    return tf.value, ms.value
