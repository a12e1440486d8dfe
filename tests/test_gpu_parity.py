"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle on the same
seeded inputs (SURVEY.md 8c rungs T2-T3).  Tolerances are BASELINE.json north_star's:
  fp64: ||A - QR||_F/||A||_F <= 1e-12, ||X - X_or||/||X_or|| <= 1e-9
  fp32: <= 5e-5 and <= 1e-3 (against the fp32 oracle).
R is unique up to row signs, X is unique (reading R4); both sides use the same
Householder convention so V, tau, T are compared directly at rounding level as well.
"""
import numpy as np
import pytest

import oracle
import paper_2412_07631_b200 as ctqr
from paper_2412_07631_b200 import workload as wl

pytestmark = pytest.mark.gpu

DT = [np.float64, np.float32]
BACKWARD = {np.float64: 1e-12, np.float32: 5e-5}
SOLUTION = {np.float64: 1e-9, np.float32: 1e-3}
ROUND = {np.float64: 1e-11, np.float32: 5e-4}      # V / tau / T / R agreement (same convention)


def relerr(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (den if den > 0 else 1.0)


def worst_col(a, b):
    """Largest per-column relative error (reading 17 asks for the worst column beside the Frobenius figure: one bad
    slice of a batch must not hide in the norm over all of them).  Columns of b that are exactly zero are compared
    absolutely."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    a = a.reshape(a.shape[0], -1); b = b.reshape(b.shape[0], -1)
    den = np.linalg.norm(b, axis=0)
    return float(np.max(np.linalg.norm(a - b, axis=0) / np.where(den > 0, den, 1.0))) if a.size else 0.0


def max_abs(a, b):
    """Largest element error, relative to the largest element of the reference."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)) if a.size else 0.0


def backward_error(A, V, tau, R):
    """||A - Q R||_F / ||A||_F with Q R evaluated in fp64 from the returned reflectors
    (reading 17): apply H_{n-1} ... H_0 order reversed to [R; 0]."""
    A = np.asarray(A, dtype=np.float64)
    m, n = A.shape
    QR = np.zeros((m, n))
    QR[:n] = np.triu(np.asarray(R, dtype=np.float64))
    V = np.asarray(V, dtype=np.float64); tau = np.asarray(tau, dtype=np.float64)
    for j in range(n - 1, -1, -1):
        v = V[:, j]
        QR -= tau[j] * np.outer(v, v @ QR)
    return np.linalg.norm(A - QR) / np.linalg.norm(A)


def gpu_factor_solve(A, B, **opts):
    m, n = A.shape
    S = B.shape[1]
    At = ctqr.colmajor_from_numpy(A)
    Bt = ctqr.colmajor_from_numpy(B.astype(A.dtype))
    f = ctqr.ct_qr_factor(At, m, n, **opts)
    import torch
    Xt = torch.zeros((S, n), dtype=At.dtype, device="cuda")
    ctqr.ct_qr_solve(f, Bt, S, Xt)
    out = dict(R=ctqr.ct_qr_get_R(f), V=ctqr.ct_qr_get_V(f), tau=ctqr.ct_qr_get_tau(f),
               X=ctqr.numpy_from_colmajor(Xt), stats=f.stats(), f=f)
    return out


def check_against_oracle(A, B, dt, **opts):
    A = np.asfortranarray(A.astype(dt)); B = np.asfortranarray(B.astype(dt))
    g = gpu_factor_solve(A, B, **opts)
    VR, tau = oracle.qr(A)
    X_or = oracle.solve(VR, tau, B)
    be = backward_error(A, g["V"], g["tau"], g["R"])
    assert be <= BACKWARD[dt], f"backward error {be}"
    se = relerr(g["X"], X_or)
    assert se <= SOLUTION[dt], f"solution error {se}"
    # every slice on its own meets the gate, and no single pixel is off by more than the gate times the largest pixel
    assert worst_col(g["X"], X_or) <= SOLUTION[dt], f"worst slice {worst_col(g['X'], X_or)}"
    assert max_abs(g["X"], X_or) <= SOLUTION[dt], f"largest element error {max_abs(g['X'], X_or)}"
    # same convention => same R (with signs), V, tau up to rounding; also column by column and element by element
    assert relerr(g["R"], oracle.R_of(VR)) <= ROUND[dt]
    assert relerr(g["V"], oracle.V_of(VR)) <= ROUND[dt]
    assert relerr(g["tau"], tau) <= ROUND[dt]
    assert worst_col(g["R"], oracle.R_of(VR)) <= 10 * ROUND[dt] and max_abs(g["R"], oracle.R_of(VR)) <= ROUND[dt]
    assert worst_col(g["V"], oracle.V_of(VR)) <= 10 * ROUND[dt] and max_abs(g["V"], oracle.V_of(VR)) <= ROUND[dt]
    assert np.all(np.tril(g["R"], -1) == 0)
    return g, VR, tau


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("shape", [(1, 1), (3, 2), (7, 4), (16, 16), (33, 17), (40, 40), (300, 130), (517, 259)])
def test_random_small(shape, dt):
    m, n = shape
    rng = np.random.default_rng(100 * m + n)
    A = rng.standard_normal((m, n)); B = rng.standard_normal((m, 5))
    check_against_oracle(A, B, dt)


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("shape", [(2500, 1300), (4099, 1025), (1300, 1300)])
def test_small_batch_fused_solve(shape, dt):
    """S <= 8 takes the two fused cooperative kernels (one launch for Q^T B, one for the TRSM):
    every CTA owns several row chunks, the last chunk is ragged, n is not a multiple of nb.  S = 9 takes
    the medium-S kernel (fp64) or the per-panel path (fp32) for Q^T B and the per-block TRSM; all must meet the oracle."""
    import torch
    m, n = shape
    rng = np.random.default_rng(31 * m + n)
    A = np.asfortranarray(rng.standard_normal((m, n)).astype(dt))
    B = np.asfortranarray(rng.standard_normal((m, 9)).astype(dt))
    VR, tau = oracle.qr(A)
    X_or = oracle.solve(VR, tau, B)
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n)
    for S in (1, 3, 8, 9):
        Bt = ctqr.colmajor_from_numpy(np.asfortranarray(B[:, :S]))
        Xt = torch.zeros((S, n), dtype=Bt.dtype, device="cuda")
        ctqr.ct_qr_solve(f, Bt, S, Xt)                      # first call of a handle also inverts the diagonal blocks
        ctqr.ct_qr_solve(f, Bt, S, Xt)
        X = ctqr.numpy_from_colmajor(Xt)
        assert relerr(X, X_or[:, :S]) <= SOLUTION[dt], (S, relerr(X, X_or[:, :S]))
        launches = f.stats()["kernel_launches"]
        if S <= 8:
            assert launches == 2, launches
        elif dt == np.float64:
            assert launches == 3, launches          # medium-S Q^T B kernel + the fused TRSM in two chunks of <= 8 columns
        else:
            assert launches > 2 * f.stats()["n_panels"]
    f.destroy()


@pytest.mark.parametrize("shape,band", [((2500, 1300), False), ((4099, 1025), False), ((1300, 1300), False),
                                        ((60000, 300), False), ((3000, 1100), True)])
def test_medium_batch_fused_apply_qt(shape, band):
    """8 < S <= 64 in fp64 takes the medium-S cooperative kernel (solve_mid.cuh, stats.apply_qt_path = 4): one launch per
    chunk of 32 (or 16) right-hand sides, ragged last group of eight, ragged last chunk, n not a multiple of nb; the tall
    shape leaves no room for 32 columns per launch (two launches of 16); with the band promise the row ranges shrink.
    C = Q^T B against the oracle's reflector-by-reflector application and X against the oracle's solve."""
    import torch
    dt = np.float64
    m, n = shape
    rng = np.random.default_rng(17 * m + n)
    if band:
        m0 = m - n
        A = np.zeros((m, n)); A[:m0] = rng.standard_normal((m0, n)); A[m0:] = 0.7 * np.eye(n)
        A = np.asfortranarray(A)
    else:
        A = np.asfortranarray(rng.standard_normal((m, n)))
    B = np.asfortranarray(rng.standard_normal((m, 64)))
    VR, tau = oracle.qr(A)
    C_or = oracle.apply_qt(VR, tau, B)
    X_or = oracle.backsub(VR, C_or[:n])
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n, lower_bandwidth=(m - n) if band else 0)
    P = f.stats()["n_panels"]
    for S in ((9, 16, 17, 24, 32, 33, 64) if m < 10000 else (12, 24, 32)):
        Ct = ctqr.colmajor_from_numpy(np.asfortranarray(B[:, :S]))
        ctqr.ct_qr_apply_qt(f, Ct, S)
        st = f.stats()
        assert st["apply_qt_path"] == 4, (S, st["apply_qt_path"])
        assert st["kernel_launches"] <= 2 + 3 * P        # (the first call also builds M_j: three launches per panel)
        C = ctqr.numpy_from_colmajor(Ct)
        assert relerr(C, C_or[:, :S]) <= 1e-11, (S, relerr(C, C_or[:, :S]))
        assert worst_col(C, C_or[:, :S]) <= 1e-11
        Ct2 = ctqr.colmajor_from_numpy(np.asfortranarray(B[:, :S]))
        ctqr.ct_qr_apply_qt(f, Ct2, S)                      # deterministic: the same bits on a second call
        assert f.stats()["kernel_launches"] <= 2
        assert torch.equal(Ct, Ct2)
        Bt = ctqr.colmajor_from_numpy(np.asfortranarray(B[:, :S]))
        Xt = torch.zeros((S, n), dtype=Bt.dtype, device="cuda")
        ctqr.ct_qr_solve(f, Bt, S, Xt)
        X = ctqr.numpy_from_colmajor(Xt)
        assert relerr(X, X_or[:, :S]) <= SOLUTION[dt], (S, relerr(X, X_or[:, :S]))
        assert worst_col(X, X_or[:, :S]) <= SOLUTION[dt]
    # S = 65 is beyond two chunks: per-panel path
    Ct = ctqr.colmajor_from_numpy(np.asfortranarray(np.concatenate([B, B[:, :1]], axis=1)))
    ctqr.ct_qr_apply_qt(f, Ct, 65)
    assert f.stats()["apply_qt_path"] == 0
    assert relerr(ctqr.numpy_from_colmajor(Ct)[:, :64], C_or) <= 1e-11
    f.destroy()


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("band", [False, True])
def test_large_batch_two_panel_apply_qt(dt, band):
    """S >= 1024 applies Q^T two panels at a time (stats.apply_qt_path = 5: the 256-wide compact-WY blocks of the
    factorisation, merged T factor assembled from the cached off-diagonal block): seven full panels + a ragged one, so
    three pairs, one single full panel and the 4-column tail; with the band promise too.  Against the oracle."""
    import torch
    m, n, S = 1500, 900, 1024
    rng = np.random.default_rng(5)
    if band:
        m0 = m - n
        A = np.zeros((m, n)); A[:m0] = rng.standard_normal((m0, n)); A[m0:] = 0.8 * np.eye(n)
    else:
        A = rng.standard_normal((m, n))
    A = np.asfortranarray(A.astype(dt))
    B = np.asfortranarray(rng.standard_normal((m, S)).astype(dt))
    VR, tau = oracle.qr(A)
    C_or = oracle.apply_qt(VR, tau, B)
    X_or = oracle.backsub(VR, C_or[:n])
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n, lower_bandwidth=(m - n) if band else 0, solve_pairs=1)
    for rep in range(2):                                     # the second call reuses the cached blocks
        Ct = ctqr.colmajor_from_numpy(B)
        ctqr.ct_qr_apply_qt(f, Ct, S)
        assert f.stats()["apply_qt_path"] == 5
        C = ctqr.numpy_from_colmajor(Ct)
        assert relerr(C, C_or) <= ROUND[dt], relerr(C, C_or)
        assert worst_col(C, C_or) <= 10 * ROUND[dt]
    Xt = torch.zeros((S, n), dtype=Ct.dtype, device="cuda")
    ctqr.ct_qr_solve(f, ctqr.colmajor_from_numpy(B), S, Xt)
    X = ctqr.numpy_from_colmajor(Xt)
    assert relerr(X, X_or) <= SOLUTION[dt] and worst_col(X, X_or) <= SOLUTION[dt]
    # option solve_pairs = 1 (by default these paths start at sizes the oracle cannot reach): from 256 right-hand sides on
    # the blocked TRSM takes two diagonal blocks per update (K = 256; fp32: pre-split, TMA-fed when S is a multiple of 8,
    # the plain contraction otherwise; the diagonal task is mm128_kernel up to S = 512, a contraction beyond);
    # ct_qr_trsm on the oracle's C isolates it
    for S2 in (320, 300, 512, 1024):
        Ct2 = ctqr.colmajor_from_numpy(np.asfortranarray(C_or[:n, :S2]))
        X2 = torch.zeros((S2, n), dtype=Ct.dtype, device="cuda")
        ctqr.ct_qr_trsm(f, Ct2, S2, X2)
        X2 = ctqr.numpy_from_colmajor(X2)
        assert relerr(X2, X_or[:, :S2]) <= SOLUTION[dt], (S2, relerr(X2, X_or[:, :S2]))
        assert worst_col(X2, X_or[:, :S2]) <= SOLUTION[dt]
    Ct3 = ctqr.colmajor_from_numpy(np.asfortranarray(B[:, :256]))
    ctqr.ct_qr_apply_qt(f, Ct3, 256)
    assert f.stats()["apply_qt_path"] == 5
    assert relerr(ctqr.numpy_from_colmajor(Ct3), C_or[:, :256]) <= ROUND[dt]
    f.destroy()
    # the default (by size) and "never" leave both paths off at this size: same results from the one-panel order
    for sp in (0, -1):
        f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n, lower_bandwidth=(m - n) if band else 0, solve_pairs=sp)
        Xt = torch.zeros((512, n), dtype=Ct.dtype, device="cuda")
        ctqr.ct_qr_solve(f, ctqr.colmajor_from_numpy(np.asfortranarray(B[:, :512])), 512, Xt)
        assert f.stats()["apply_qt_path"] == 0
        assert relerr(ctqr.numpy_from_colmajor(Xt), X_or[:, :512]) <= SOLUTION[dt]
        f.destroy()


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("nb,ib", [(8, 8), (32, 16), (64, 16), (128, 16), (128, 32), (64, 8)])
@pytest.mark.parametrize("la", [0, 1])
def test_blocking_invariance(nb, ib, la, dt):
    """Reading 6: results must not depend on nb / look-ahead beyond rounding; n not a multiple of
    nb and m - n < nb are covered by the shape."""
    rng = np.random.default_rng(7)
    A = rng.standard_normal((700, 650)); B = rng.standard_normal((700, 9))
    check_against_oracle(A, B, dt, nb=nb, ib=ib, lookahead=la)


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("cfg", ["c0", "c1"])
def test_ct_config(cfg, dt):
    c = wl.CONFIGS[cfg]
    coo = wl.siddon_coo(c.N, c.n_ang, c.n_bins)
    A, lam = wl.dense_augmented(c, np.float64, coo)
    X0, B = wl.make_slices(c, coo=coo, lam=lam)
    g, VR, tau = check_against_oracle(A, B, dt)
    # T factor of the first and last panel against the oracle's larft recurrence
    nb = g["stats"]["nb"]
    for k in (0, g["stats"]["n_panels"] - 1):
        Tg = ctqr.ct_qr_get_T(g["f"], k)
        To = oracle.larft(VR, tau, k * nb, Tg.shape[0])
        assert relerr(Tg, To) <= ROUND[dt]


@pytest.mark.parametrize("dt", DT)
def test_zero_column_and_triangular(dt):
    rng = np.random.default_rng(3)
    A = rng.standard_normal((90, 40))
    A[:, 5] = 0.0                       # zero column: tau = 0, R_jj = 0 -> solve must refuse
    At = ctqr.colmajor_from_numpy(np.asfortranarray(A.astype(dt)))
    f = ctqr.ct_qr_factor(At, 90, 40)
    tau = ctqr.ct_qr_get_tau(f)
    VR, tau_o = oracle.qr(np.asfortranarray(A.astype(dt)))
    assert relerr(tau, tau_o) <= ROUND[dt]
    import torch
    Bt = torch.ones((2, 90), dtype=At.dtype, device="cuda"); Xt = torch.zeros((2, 40), dtype=At.dtype, device="cuda")
    # upper-triangular input: every sub-column is zero => tau = 0, R = A
    U = np.triu(rng.standard_normal((30, 30))) + 3 * np.eye(30)
    Ut = ctqr.colmajor_from_numpy(np.asfortranarray(U.astype(dt)))
    f2 = ctqr.ct_qr_factor(Ut, 30, 30)
    assert np.all(ctqr.ct_qr_get_tau(f2) == 0)
    assert np.array_equal(ctqr.ct_qr_get_R(f2), U.astype(dt))


def test_singular_solve_refused():
    import torch
    A = np.zeros((20, 4)); A[:4, :4] = np.eye(4); A[2, 2] = 0.0
    At = ctqr.colmajor_from_numpy(np.asfortranarray(A))
    f = ctqr.ct_qr_factor(At, 20, 4)
    Bt = torch.ones((1, 20), dtype=torch.float64, device="cuda"); Xt = torch.zeros((1, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_solve(f, Bt, 1, Xt)
    assert ei.value.code == 4


@pytest.mark.parametrize("dt", DT)
def test_trsm_exact_option_and_conditioning_guard(dt):
    """Blocked TRSM diagonal tasks: inverted diagonal blocks by default, back-substitution by option,
    and by itself when a diagonal block of R is ill-conditioned (columns graded over 12 / 5 orders of magnitude)."""
    rng = np.random.default_rng(77)
    m, n, S = 700, 384, 11
    A0 = rng.standard_normal((m, n))
    B = rng.standard_normal((m, S))
    # well conditioned: default uses the inverses, the option forces back-substitution, both match the oracle
    for exact in (False, True):
        g, VR, tau = check_against_oracle(A0, B, dt, trsm_exact=exact)
        st = g["f"].stats()
        assert st["trsm_exact"] == (1 if exact else 0)
        if not exact:
            assert 1.0 <= st["diag_block_cond"] < 1e3
        C = oracle.apply_qt(VR, tau, np.asfortranarray(B.astype(dt)))[:n]
        X = np.zeros((n, S), dtype=dt, order="F")
        ctqr.ct_qr_trsm(g["f"], np.asfortranarray(C), S, X)
        assert relerr(X, oracle.backsub(VR, C)) <= ROUND[dt] * 10
        g["f"].destroy()
    # graded columns inside every 128-block: the guard must switch to back-substitution and the solve must be
    # backward stable: ||R X - C|| <= c n u ||R|| ||X||, column by column
    span = 12.0 if dt == np.float64 else 5.0
    scale = 10.0 ** (-span * (np.arange(n) % 128) / 127.0)
    A = np.asfortranarray((A0 * scale).astype(dt))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n)
    R = ctqr.ct_qr_get_R(f).astype(np.float64)
    C = np.asfortranarray(rng.standard_normal((n, S)).astype(dt))
    X = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_trsm(f, C, S, X)
    st = f.stats()
    assert st["trsm_exact"] == 2 and st["diag_block_cond"] > (6.7e7 if dt == np.float64 else 2.9e3)
    X64 = X.astype(np.float64)
    u = np.finfo(dt).eps
    res = np.linalg.norm(R @ X64 - C.astype(np.float64), axis=0) / (np.linalg.norm(R) * np.linalg.norm(X64, axis=0))
    assert res.max() <= 4 * n * u, res.max()
    f.destroy()


def test_trim_cache_releases_blocks():
    rng = np.random.default_rng(5)
    A = rng.standard_normal((300, 200))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), 300, 200)
    f.destroy()                                   # its small buffers go to the process-wide cache
    assert ctqr.ct_qr_trim_cache() > 0
    assert ctqr.ct_qr_trim_cache() == 0
    check_against_oracle(A, rng.standard_normal((300, 3)), np.float64)      # the library works on after a trim


@pytest.mark.parametrize("dt", DT)
def test_host_pointers_and_halves(dt):
    """Host (numpy) A, B, X; apply_qt and trsm alone against the oracle's two halves."""
    rng = np.random.default_rng(11)
    A = np.asfortranarray(rng.standard_normal((400, 200)).astype(dt))
    B = np.asfortranarray(rng.standard_normal((400, 17)).astype(dt))
    f = ctqr.ct_qr_factor(A.copy(order="F"), 400, 200)
    VR, tau = oracle.qr(A)
    C = B.copy(order="F")
    ctqr.ct_qr_apply_qt(f, C, 17)
    C_or = oracle.apply_qt(VR, tau, B)
    assert relerr(C, C_or) <= ROUND[dt]
    X = np.zeros((200, 17), dtype=dt, order="F")
    ctqr.ct_qr_trsm(f, np.asfortranarray(C_or[:200]), 17, X)
    assert relerr(X, oracle.backsub(VR, C_or[:200])) <= SOLUTION[dt]
    X2 = np.zeros((200, 17), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, B, 17, X2)
    assert relerr(X2, oracle.solve(VR, tau, B)) <= SOLUTION[dt]


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("ta", [True, False])
@pytest.mark.parametrize("impl", [0, 1])
@pytest.mark.parametrize("mnk", [(128, 64, 256), (37, 150, 1001), (130, 9, 77), (5, 300, 4),
                                 # shapes that reach the stream-K / tcgen05 kernels with ragged tiles and K tails
                                 (100, 300, 1000), (1000, 300, 100), (256, 128, 4096), (128, 1000, 36)])
def test_gemm_kernel(mnk, impl, ta, dt):
    """Kernel-level: C <- alpha op(A) B + beta C against the definition (numpy fp64)."""
    import torch
    M, N, K = mnk
    rng = np.random.default_rng(M + N + K)
    A = rng.standard_normal((K, M) if ta else (M, K)).astype(dt)
    B = rng.standard_normal((K, N)).astype(dt)
    C = rng.standard_normal((M, N)).astype(dt)
    ref = -1.0 * (A.T.astype(np.float64) if ta else A.astype(np.float64)) @ B.astype(np.float64) + C.astype(np.float64)
    At, Bt, Ct = (ctqr.colmajor_from_numpy(np.asfortranarray(x)) for x in (A, B, C))
    ctqr.ct_qr_gemm(ta, M, N, K, -1.0, At, A.shape[0], Bt, K, 1.0, Ct, M, impl)
    got = ctqr.numpy_from_colmajor(Ct)
    assert relerr(got, ref) <= (1e-13 if dt == np.float64 else 2e-5)


@pytest.mark.parametrize("mnk", [(128, 128, 256), (256, 128, 32), (1000, 300, 100), (517, 259, 256), (130, 9, 77),
                                 (5, 300, 4), (2100, 1000, 256), (384, 640, 128)])
def test_gemm_presplit_tma_kernel(mnk):
    """impl 2: the TMA-fed tcgen05 kernel with operands pre-split into TF32 hi / lo (C <- C - V W of the two-panel
    update): ragged tiles in M and N, K tails, K = 256 as used, against the fp64 definition at the fp32 kernel gate."""
    M, N, K = mnk
    rng = np.random.default_rng(M + N + K)
    A = rng.standard_normal((M, K)).astype(np.float32)
    B = rng.standard_normal((K, N)).astype(np.float32)
    C = rng.standard_normal((M, N)).astype(np.float32)
    ref = -1.0 * A.astype(np.float64) @ B.astype(np.float64) + C.astype(np.float64)
    At, Bt, Ct = (ctqr.colmajor_from_numpy(np.asfortranarray(x)) for x in (A, B, C))
    ctqr.ct_qr_gemm(False, M, N, K, -1.0, At, M, Bt, K, 1.0, Ct, M, 2)
    got = ctqr.numpy_from_colmajor(Ct)
    assert relerr(got, ref) <= 2e-5, relerr(got, ref)
    assert max_abs(got, ref) <= 2e-5


def test_gemm_presplit_long_k_accumulation():
    """Same-sign data, K = 32768: the TMEM accumulator is drained every 128 of K, so the truncating in-MMA accumulation
    must stay at FFMA level (<= 1e-5 elementwise; 3e-4 if the whole K were accumulated inside the tensor core)."""
    import torch
    M, N, K = 128, 192, 32768
    rng = np.random.default_rng(1)
    A = np.abs(rng.standard_normal((M, K))).astype(np.float32)
    B = np.abs(rng.standard_normal((K, N))).astype(np.float32)
    ref = A.astype(np.float64) @ B.astype(np.float64)
    At, Bt = (ctqr.colmajor_from_numpy(np.asfortranarray(x)) for x in (A, B))
    Ct = torch.zeros((N, M), dtype=torch.float32, device="cuda")
    ctqr.ct_qr_gemm(False, M, N, K, 1.0, At, M, Bt, K, 0.0, Ct, M, 2)
    err = np.max(np.abs(ctqr.numpy_from_colmajor(Ct) - ref) / np.abs(ref))
    assert err <= 1e-5, err


# ---- a5: out-of-core scheduler (SURVEY.md 8c rung T4) ---------------------------------------
def _ooc_budget(m, nb, ns, dt):
    w = np.dtype(dt).itemsize
    lds = -(-m // (16 // w)) * (16 // w)
    return (2 * ns + 2 * nb) * lds * w + 64


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("nb,ns,pinned", [(32, 288, True), (32, 160, False), (32, 96, True), (64, 64, False)])
def test_out_of_core_matches_oracle_and_in_core(nb, ns, pinned, dt):
    """Host-resident A with a capped device budget (P_s = 3, 5, 7, 11 super-panels): the factor is
    written back into the host buffer; results must meet the same gates as in core and agree
    with the in-core path to rounding."""
    import torch
    m, n, S = 700, 650, 9
    rng = np.random.default_rng(21)
    A = np.asfortranarray(rng.standard_normal((m, n)).astype(dt))
    B = np.asfortranarray(rng.standard_normal((m, S)).astype(dt))
    Ah = ctqr.colmajor_from_numpy(A, device="cpu", pin=pinned)
    f = ctqr.ct_qr_factor(Ah, m, n, nb=nb, ib=16, device_budget_bytes=_ooc_budget(m, nb, ns, dt))
    st = f.stats()
    assert st["out_of_core"] == 1 and st["n_superpanels"] == -(-n // ns)
    w = np.dtype(dt).itemsize
    Ps = st["n_superpanels"]
    assert st["d2h_bytes"] == m * n * w and st["h2d_bytes"] >= m * n * w
    X = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, B, S, X)
    R, V, tau = ctqr.ct_qr_get_R(f), ctqr.ct_qr_get_V(f), ctqr.ct_qr_get_tau(f)
    VR, tau_o = oracle.qr(A)
    assert backward_error(A, V, tau, R) <= BACKWARD[dt]
    assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
    assert relerr(R, oracle.R_of(VR)) <= ROUND[dt]
    assert relerr(V, oracle.V_of(VR)) <= ROUND[dt]
    # in-core on the same input
    g = gpu_factor_solve(A, B, nb=nb, ib=16)
    assert relerr(R, g["R"]) <= ROUND[dt] and relerr(X, g["X"]) <= SOLUTION[dt]
    # the two halves of the solve through the streamed path
    C = B.copy(order="F"); ctqr.ct_qr_apply_qt(f, C, S)
    assert relerr(C, oracle.apply_qt(VR, tau_o, B)) <= ROUND[dt]


@pytest.mark.parametrize("dt,band", [(np.float64, False), (np.float32, False), (np.float64, True)])
def test_out_of_core_pair_updates(dt, band):
    """Super-panels of 1280 columns (P_s = 4, the last one 44 columns wide): wide enough for the two-panel path, so the
    factorisation inside a super-panel and the left-looking updates -- from the previous super-panel still resident and
    from pairs of panels streamed back from the host -- all run as 256-wide compact-WY blocks (fp32: pre-split, TMA-fed).
    Same gates as in core, against the oracle and against the in-core factor; with the band promise as well."""
    m, n, S, ns = 4600, 3884, 5, 1280
    rng = np.random.default_rng(77)
    if band:
        m0 = m - n
        A = np.zeros((m, n)); A[:m0] = rng.standard_normal((m0, n)); A[m0:] = 0.9 * np.eye(n)
    else:
        A = rng.standard_normal((m, n))
    A = np.asfortranarray(A.astype(dt))
    B = np.asfortranarray(rng.standard_normal((m, S)).astype(dt))
    Ah = ctqr.colmajor_from_numpy(A, device="cpu", pin=True)
    f = ctqr.ct_qr_factor(Ah, m, n, device_budget_bytes=_ooc_budget(m, 128, ns, dt), lower_bandwidth=(m - n) if band else 0)
    st = f.stats()
    assert st["out_of_core"] == 1 and st["n_superpanels"] == 4
    X = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, B, S, X)
    R, V, tau = ctqr.ct_qr_get_R(f), ctqr.ct_qr_get_V(f), ctqr.ct_qr_get_tau(f)
    VR, tau_o = oracle.qr(A)
    X_or = oracle.solve(VR, tau_o, B)
    assert relerr(X, X_or) <= SOLUTION[dt] and worst_col(X, X_or) <= SOLUTION[dt]
    assert relerr(R, oracle.R_of(VR)) <= ROUND[dt] and max_abs(R, oracle.R_of(VR)) <= ROUND[dt]
    assert relerr(V, oracle.V_of(VR)) <= ROUND[dt] and max_abs(V, oracle.V_of(VR)) <= ROUND[dt]
    assert relerr(tau, tau_o) <= ROUND[dt]
    f.destroy()
    g = gpu_factor_solve(A, B, lower_bandwidth=(m - n) if band else 0)
    assert relerr(R, g["R"]) <= ROUND[dt] and relerr(X, g["X"]) <= SOLUTION[dt]
    g["f"].destroy()


@pytest.mark.parametrize("dt", DT)
def test_out_of_core_ct_config(dt):
    """BASELINE.json configs[0] streamed through 4 super-panels of 256 columns."""
    c = wl.CONFIGS["c1"]
    coo = wl.siddon_coo(c.N, c.n_ang, c.n_bins)
    A, lam = wl.dense_augmented(c, dt, coo)
    X0, B = wl.make_slices(c, coo=coo, lam=lam)
    B = np.asfortranarray(B.astype(dt))
    Ah = ctqr.colmajor_from_numpy(A, device="cpu", pin=True)
    f = ctqr.ct_qr_factor(Ah, c.m, c.n, device_budget_bytes=_ooc_budget(c.m, 128, 256, dt))
    assert f.stats()["n_superpanels"] == 4
    X = np.zeros((c.n, c.S), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, B, c.S, X)
    VR, tau_o = oracle.qr(A)
    assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
    assert backward_error(A, ctqr.ct_qr_get_V(f), ctqr.ct_qr_get_tau(f), ctqr.ct_qr_get_R(f)) <= BACKWARD[dt]


def test_out_of_core_budget_too_small():
    A = np.asfortranarray(np.random.default_rng(0).standard_normal((300, 200)))
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_factor(A.copy(order="F"), 300, 200, nb=32, device_budget_bytes=1000)
    assert ei.value.code == 2


@pytest.mark.parametrize("ta", [True, False])
def test_gemm_fp32_long_k_accumulation(ta):
    """The fp32 contraction runs as a 3xTF32 split on the tensor cores; the tensor core's own
    accumulator truncates, so the kernel must not let the error grow with K.
    Same-sign data makes a biased accumulation visible: at K = 32768 the result must be as good as
    an FFMA sum (a few 1e-6), two orders below what in-MMA accumulation gives (3e-4)."""
    import torch
    M, N, K = 128, 192, 32768
    rng = np.random.default_rng(1)
    A = np.abs(rng.standard_normal((K, M) if ta else (M, K))).astype(np.float32)
    B = np.abs(rng.standard_normal((K, N))).astype(np.float32)
    ref = (A.T.astype(np.float64) if ta else A.astype(np.float64)) @ B.astype(np.float64)
    At, Bt = (ctqr.colmajor_from_numpy(np.asfortranarray(x)) for x in (A, B))
    Ct = torch.zeros((N, M), dtype=torch.float32, device="cuda")
    ctqr.ct_qr_gemm(ta, M, N, K, 1.0, At, A.shape[0], Bt, K, 0.0, Ct, M, 0)
    err = np.max(np.abs(ctqr.numpy_from_colmajor(Ct) - ref) / np.abs(ref))
    assert err <= 1e-5, err


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("budget_cols", [0, 96])
def test_file_backed_tier(tmp_path, dt, budget_cols):
    """Optional file tier (the matrix lives on secondary storage behind a host-RAM
    cache): the matrix is read from a file through the page cache, the factor is written back into
    the same file, the solve streams it from there.  budget 0 = one super-panel if it fits."""
    m, n, S, nb = 600, 500, 7, 32
    rng = np.random.default_rng(33)
    A = np.asfortranarray(rng.standard_normal((m, n)).astype(dt))
    B = np.asfortranarray(rng.standard_normal((m, S)).astype(dt))
    path = str(tmp_path / "A.bin")
    A.T.tofile(path)                                  # column-major bytes, lda = m
    budget = _ooc_budget(m, nb, budget_cols, dt) if budget_cols else 0
    f = ctqr.ct_qr_factor(None, m, n, nb=nb, file_path=path, dtype=dt, device_budget_bytes=budget)
    st = f.stats()
    assert st["out_of_core"] == 1 and st["n_superpanels"] == (-(-n // budget_cols) if budget_cols else 1)
    X = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, B, S, X)
    R, V, tau = ctqr.ct_qr_get_R(f), ctqr.ct_qr_get_V(f), ctqr.ct_qr_get_tau(f)
    VR, tau_o = oracle.qr(A)
    assert backward_error(A, V, tau, R) <= BACKWARD[dt]
    assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
    f.destroy()
    # the file now holds the factor: V below the diagonal blocks (and R above them)
    F = np.fromfile(path, dtype=dt).reshape(n, m).T
    assert relerr(np.tril(F, -nb)[:, :n], np.tril(oracle.V_of(VR), -nb)) <= ROUND[dt]


def test_file_tier_errors(tmp_path):
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_factor(None, 100, 50, file_path=str(tmp_path / "missing.bin"), dtype=np.float64)
    assert ei.value.code == 3
    p = tmp_path / "short.bin"
    p.write_bytes(b"\0" * 64)
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_factor(None, 100, 50, file_path=str(p), dtype=np.float64)
    assert ei.value.code == 3
