"""CPU oracle (TEST INFRASTRUCTURE ONLY) -- ctypes front end of ``oracle/oracle.c``.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.  The product
(``paper_2412_07631_b200``) never does, and this package never imports the product.

What it computes: PAPER.md Eq. 2 (A = QR, L41) and Eq. 3 (X = R^{-1}(Q^T B), L43-48) by
their plain definitions -- unblocked Householder QR, reflector-by-reflector Q^T b, scalar
back-substitution -- in fp64 or fp32, every operation in the working precision.
Pins: tests/test_oracle_pins.py.  Parity unpinned: none.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_lib = None

_P = ctypes.c_void_p
_I = ctypes.c_int64


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (-O2 -ffp-contract=off -fopenmp).  Returns the .so path."""
    srcs = [os.path.join(_HERE, f) for f in ("oracle.c", "oracle_impl.inc", "oracle.h")]
    if (not force and os.path.exists(_LIB_PATH)
            and all(os.path.getmtime(_LIB_PATH) >= os.path.getmtime(s) for s in srcs)):
        return _LIB_PATH
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
           os.path.join(_HERE, "oracle.c"), "-o", _LIB_PATH, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        for suf in ("f64", "f32"):
            getattr(lib, f"oracle_qr_{suf}").argtypes = [_P, _I, _I, _I, _P]
            getattr(lib, f"oracle_qr_{suf}").restype = ctypes.c_int
            for nm in ("apply_qt", "apply_q"):
                f = getattr(lib, f"oracle_{nm}_{suf}")
                f.argtypes = [_P, _I, _I, _I, _P, _P, _I, _I]
                f.restype = ctypes.c_int
            f = getattr(lib, f"oracle_backsub_{suf}")
            f.argtypes = [_P, _I, _I, _P, _I, _I, _P, _I]
            f.restype = ctypes.c_int64
            f = getattr(lib, f"oracle_backsub_t_{suf}")
            f.argtypes = [_P, _I, _I, _P, _I, _I, _P, _I]
            f.restype = ctypes.c_int64
            f = getattr(lib, f"oracle_larft_{suf}")
            f.argtypes = [_P, _I, _I, _P, _I, _I, _P, _I]
            f.restype = ctypes.c_int
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def _suf(dtype) -> str:
    dt = np.dtype(dtype)
    if dt == np.float64:
        return "f64"
    if dt == np.float32:
        return "f32"
    raise TypeError(f"oracle supports float32/float64, got {dt}")


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_P)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def qr(A: np.ndarray):
    """Householder QR (Eq. 2).  Returns (VR, tau): VR holds R on/above and v_j below the
    diagonal (Fortran order, same dtype as A); A itself is not modified."""
    A = np.asarray(A)
    suf = _suf(A.dtype)
    m, n = A.shape
    VR = np.array(A, order="F", copy=True)
    tau = np.zeros(n, dtype=A.dtype)
    rc = getattr(_load(), f"oracle_qr_{suf}")(_ptr(VR), m, n, max(m, 1), _ptr(tau))
    if rc != 0:
        raise ValueError(f"oracle_qr: bad argument {-rc}")
    return VR, tau


def apply_qt(VR: np.ndarray, tau: np.ndarray, B: np.ndarray) -> np.ndarray:
    """C = Q^T B (first half of Eq. 3).  Returns a new (m, S) Fortran array."""
    suf = _suf(VR.dtype)
    m, n = VR.shape
    C = np.array(B, dtype=VR.dtype, order="F", copy=True).reshape(m, -1, order="F")
    VRf = np.asfortranarray(VR)
    rc = getattr(_load(), f"oracle_apply_qt_{suf}")(_ptr(VRf), m, n, max(m, 1), _ptr(tau), _ptr(C), max(m, 1), C.shape[1])
    if rc != 0:
        raise ValueError("oracle_apply_qt: bad argument")
    return C


def apply_q(VR: np.ndarray, tau: np.ndarray, B: np.ndarray) -> np.ndarray:
    """Q B (reflectors in reverse order).  Returns a new (m, S) Fortran array."""
    suf = _suf(VR.dtype)
    m, n = VR.shape
    C = np.array(B, dtype=VR.dtype, order="F", copy=True).reshape(m, -1, order="F")
    VRf = np.asfortranarray(VR)
    rc = getattr(_load(), f"oracle_apply_q_{suf}")(_ptr(VRf), m, n, max(m, 1), _ptr(tau), _ptr(C), max(m, 1), C.shape[1])
    if rc != 0:
        raise ValueError("oracle_apply_q: bad argument")
    return C


def backsub(VR: np.ndarray, C: np.ndarray) -> np.ndarray:
    """X = R^{-1} C[0:n] (second half of Eq. 3) by back-substitution."""
    suf = _suf(VR.dtype)
    m, n = VR.shape
    Cf = np.asfortranarray(np.asarray(C, dtype=VR.dtype)).reshape(C.shape[0], -1, order="F")
    S = Cf.shape[1]
    X = np.zeros((n, S), dtype=VR.dtype, order="F")
    VRf = np.asfortranarray(VR)
    rc = getattr(_load(), f"oracle_backsub_{suf}")(_ptr(VRf), n, max(m, 1), _ptr(Cf), max(Cf.shape[0], 1), S, _ptr(X), max(n, 1))
    if rc != 0:
        raise ZeroDivisionError(f"oracle_backsub: R[{rc - 1},{rc - 1}] == 0")
    return X


def backsub_t(VR: np.ndarray, C: np.ndarray) -> np.ndarray:
    """Y = R^{-T} C[0:n] by forward substitution with the transposed factor."""
    suf = _suf(VR.dtype)
    m, n = VR.shape
    Cf = np.asfortranarray(np.asarray(C, dtype=VR.dtype)).reshape(C.shape[0], -1, order="F")
    S = Cf.shape[1]
    Y = np.zeros((n, S), dtype=VR.dtype, order="F")
    VRf = np.asfortranarray(VR)
    rc = getattr(_load(), f"oracle_backsub_t_{suf}")(_ptr(VRf), n, max(m, 1), _ptr(Cf), max(Cf.shape[0], 1), S, _ptr(Y), max(n, 1))
    if rc != 0:
        raise ZeroDivisionError(f"oracle_backsub_t: R[{rc - 1},{rc - 1}] == 0")
    return Y


def solve(VR: np.ndarray, tau: np.ndarray, B: np.ndarray) -> np.ndarray:
    """X = R^{-1}(Q^T B) (Eq. 3)."""
    return backsub(VR, apply_qt(VR, tau, B))


def larft(VR: np.ndarray, tau: np.ndarray, j0: int, nb: int) -> np.ndarray:
    """Compact-WY T (nb x nb upper triangular) of reflectors j0 .. j0+nb-1."""
    suf = _suf(VR.dtype)
    m, n = VR.shape
    T = np.zeros((nb, nb), dtype=VR.dtype, order="F")
    VRf = np.asfortranarray(VR)
    rc = getattr(_load(), f"oracle_larft_{suf}")(_ptr(VRf), m, max(m, 1), _ptr(tau), j0, nb, _ptr(T), max(nb, 1))
    if rc != 0:
        raise ValueError("oracle_larft: bad argument")
    return T


# ---- small helpers used by tests (definitions, not algorithms) ---------------------------
def R_of(VR: np.ndarray) -> np.ndarray:
    n = VR.shape[1]
    return np.triu(VR[:n, :])


def V_of(VR: np.ndarray) -> np.ndarray:
    m, n = VR.shape
    V = np.tril(VR, -1)
    V[np.arange(n), np.arange(n)] = 1
    return V


def form_q(VR: np.ndarray, tau: np.ndarray) -> np.ndarray:
    """Explicit thin Q = H_0 ... H_{n-1} [I_n; 0] (tests only, tiny sizes)."""
    m, n = VR.shape
    E = np.zeros((m, n), dtype=VR.dtype, order="F")
    E[np.arange(n), np.arange(n)] = 1
    return apply_q(VR, tau, E)


def sign_normalise(R: np.ndarray) -> np.ndarray:
    """R with each row multiplied by sign(R_ii): the unique positive-diagonal R."""
    s = np.sign(np.diag(R)).copy()
    s[s == 0] = 1
    return R * s[:, None]
