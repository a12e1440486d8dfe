"""ct_qr_vtc_noalloc (include/ctqr.h): the allocation-free W = V^T C, against the library's own path for the same
product (ct_qr_gemm with trans_a = 1, whose split-K partial tiles come from cudaMalloc'd workspace).

Collected last on purpose (file name): the run is `pytest -x`, and this file must pass both alone in a fresh
process and after every other GPU test has run in the same process.
"""
import numpy as np
import pytest

import paper_2412_07631_b200 as ctqr

pytestmark = pytest.mark.gpu

# the kernel-level gates of tests/test_gpu_parity.py::test_gemm_kernel
TOL = {np.float64: 1e-13, np.float32: 2e-5}


def relerr(a, b):
    return float(np.linalg.norm(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64)) /
                 max(np.linalg.norm(np.asarray(b, dtype=np.float64)), 1e-300))


def both_paths(M, N, K, dt, seed, ldv=None, ldc=None, ldw=None):
    """Returns (W of the new entry point, W of the existing path, fp64 definition) on the same seeded inputs."""
    import torch
    rng = np.random.default_rng(seed)
    ldv, ldc, ldw = ldv or max(K, 1), ldc or max(K, 1), ldw or M
    V = np.zeros((ldv, M), dtype=dt, order="F"); V[:K] = rng.standard_normal((K, M)).astype(dt)
    C = np.zeros((ldc, N), dtype=dt, order="F"); C[:K] = rng.standard_normal((K, N)).astype(dt)
    Vt, Ct = ctqr.colmajor_from_numpy(V), ctqr.colmajor_from_numpy(C)
    W_new = ctqr.colmajor_from_numpy(np.full((ldw, N), 7.0, dtype=dt, order="F"))   # must be overwritten, not accumulated
    W_old = ctqr.colmajor_from_numpy(np.full((ldw, N), 7.0, dtype=dt, order="F"))
    ctqr.ct_qr_vtc_noalloc(M, N, K, Vt, ldv, Ct, ldc, W_new, ldw)
    ctqr.ct_qr_gemm(True, M, N, K, 1.0, Vt, ldv, Ct, ldc, 0.0, W_old, ldw, 0)
    torch.cuda.synchronize()
    ref = V[:K].astype(np.float64).T @ C[:K].astype(np.float64)
    return ctqr.numpy_from_colmajor(W_new)[:M], ctqr.numpy_from_colmajor(W_old)[:M], ref


@pytest.mark.parametrize("dt", [np.float64, np.float32])
def test_two_calls_in_a_row_match_the_existing_path(dt):
    """Two calls back to back on the one shared scratch array: a large one (many splits, every slot class used), then a
    smaller, ragged one whose tiles land on slots the first call left full of other numbers."""
    for (M, N, K, seed) in [(128, 1000, 4096, 11), (37, 150, 1001, 12)]:
        new, old, ref = both_paths(M, N, K, dt, seed)
        assert relerr(new, old) <= TOL[dt], (M, N, K, relerr(new, old))
        assert relerr(new, ref) <= TOL[dt], (M, N, K, relerr(new, ref))
        assert relerr(old, ref) <= TOL[dt]


def test_repeat_is_bit_identical_and_strides_are_honoured():
    """Deterministic (fixed split, sums in split order): the same call twice gives the same bits, also after another
    call has used the scratch in between; leading dimensions larger than the extents; rows of W beyond M untouched."""
    import torch
    dt = np.float64
    a1, _, ref = both_paths(130, 9, 777, dt, 5, ldv=800, ldc=790, ldw=140)
    both_paths(64, 64, 64, dt, 6)
    a2, old, _ = both_paths(130, 9, 777, dt, 5, ldv=800, ldc=790, ldw=140)
    assert np.array_equal(a1, a2)
    assert relerr(a1, ref) <= TOL[dt] and relerr(a1, old) <= TOL[dt]
    V = torch.randn((4, 50), dtype=torch.float64, device="cuda")          # K = 50 rows, M = 4 columns (column-major)
    C = torch.randn((3, 50), dtype=torch.float64, device="cuda")
    W = torch.full((3, 10), 7.0, dtype=torch.float64, device="cuda")      # ldw = 10 > M = 4
    ctqr.ct_qr_vtc_noalloc(4, 3, 50, V, 50, C, 50, W, 10)
    torch.cuda.synchronize()
    assert torch.all(W[:, 4:] == 7.0)
    assert torch.allclose(W[:, :4], C @ V.T, rtol=1e-13, atol=1e-13)


def test_k_zero_and_side_stream():
    import torch
    W = torch.full((5, 8), 3.0, dtype=torch.float32, device="cuda")
    V = torch.zeros((8, 1), dtype=torch.float32, device="cuda")
    C = torch.zeros((5, 1), dtype=torch.float32, device="cuda")
    ctqr.ct_qr_vtc_noalloc(8, 5, 0, V, 1, C, 1, W, 8)
    torch.cuda.synchronize()
    assert torch.all(W == 0)
    st = torch.cuda.Stream()
    V = torch.randn((70, 300), dtype=torch.float64, device="cuda")
    C = torch.randn((20, 300), dtype=torch.float64, device="cuda")
    W = torch.zeros((20, 70), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    ctqr.ct_qr_vtc_noalloc(70, 20, 300, V, 300, C, 300, W, 70, stream=st)
    st.synchronize()
    assert torch.allclose(W, C @ V.T, rtol=1e-12, atol=1e-12)


def test_sizes_beyond_the_fixed_scratch_are_refused_and_nothing_is_allocated():
    """512 output tiles of 64 x 64 fp64 (1024 in fp32) is the limit: one more is refused with a message naming it, and
    nothing is written.  The accepted calls do not change the device's free memory (no cudaMalloc behind the call)."""
    import torch
    V = torch.randn((128, 64), dtype=torch.float64, device="cuda")        # K = 64, M = 128
    N_ok, N_bad = 16384, 16385                                            # 2 x 256 tiles / 2 x 257 tiles
    C = torch.randn((N_bad, 64), dtype=torch.float64, device="cuda")
    W = torch.full((N_bad, 128), 5.0, dtype=torch.float64, device="cuda")
    ctqr.ct_qr_vtc_noalloc(128, 8, 64, V, 64, C, 64, W, 128)              # set-up call (symbol address, kernel load)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ctqr.ct_qr_vtc_noalloc(128, N_ok, 64, V, 64, C, 64, W, 128)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.allclose(W[:N_ok], C[:N_ok] @ V.T, rtol=1e-12, atol=1e-12)
    assert torch.all(W[N_ok:] == 5.0)
    W.fill_(5.0)
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_vtc_noalloc(128, N_bad, 64, V, 64, C, 64, W, 128)
    assert ei.value.code == 2 and "scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert torch.all(W == 5.0)
    with pytest.raises(ctqr.CtqrError):                                   # host pointers are refused, not dereferenced
        ctqr.ct_qr_vtc_noalloc(4, 4, 4, np.zeros((4, 4), order="F"), 4, np.zeros((4, 4), order="F"), 4,
                               np.zeros((4, 4), order="F"), 4)
