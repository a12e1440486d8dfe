"""Pins for the CPU oracle (SURVEY.md section 8c "What pins each part", rung T0).

Each test checks oracle/ against something other than itself: a hand-computed fixture, a
closed form, brute force by a different algorithm written here in plain numpy loops
(Gram-Schmidt, Cholesky, forward substitution), an invariant, or a LAPACK routine.
"""
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")
DT = [np.float64, np.float32]
EPS = {np.float64: 2.3e-16, np.float32: 6e-8}


def tol(dt, k=100.0):
    return k * EPS[dt]


def read_golden(path):
    out = {}
    with open(path) as f:
        lines = [l.strip() for l in f if l.strip() and not l.startswith("#")]
    i = 0
    while i < len(lines):
        key, r, c = lines[i].split()
        r, c = int(r), int(c)
        vals = [[float(x) for x in lines[i + 1 + k].split()] for k in range(r)]
        out[key] = np.array(vals)
        i += 1 + r
    return out


def rnd(m, n, seed, dt):
    return np.asfortranarray(np.random.default_rng(seed).standard_normal((m, n)).astype(dt))


# ---- brute-force helpers written independently of the oracle -----------------------------
def cgs2(A):
    """Classical Gram-Schmidt applied twice: positive-diagonal QR (fp64)."""
    A = np.asarray(A, dtype=np.float64)
    m, n = A.shape
    Q = np.zeros((m, n)); R = np.zeros((n, n))
    for j in range(n):
        v = A[:, j].copy()
        for _ in range(2):
            for i in range(j):
                h = float(Q[:, i] @ v)
                R[i, j] += h
                v -= h * Q[:, i]
        R[j, j] = np.sqrt(float(v @ v))
        Q[:, j] = v / R[j, j]
    return Q, R


def cholesky_upper(G):
    """Hand-written Cholesky G = U^T U (fp64)."""
    G = np.asarray(G, dtype=np.float64)
    n = G.shape[0]
    U = np.zeros((n, n))
    for j in range(n):
        s = G[j, j] - float(U[:j, j] @ U[:j, j])
        U[j, j] = np.sqrt(s)
        for k in range(j + 1, n):
            U[j, k] = (G[j, k] - float(U[:j, j] @ U[:j, k])) / U[j, j]
    return U


def householder_matrix(v, tau):
    return np.eye(len(v)) - tau * np.outer(v, v)


# ---- (i) hand-computed fixture ------------------------------------------------------------
@pytest.mark.parametrize("dt", DT)
def test_golden_3x2(dt):
    g = read_golden(os.path.join(GOLD, "householder_3x2.txt"))
    VR, tau = oracle.qr(g["A"].astype(dt))
    np.testing.assert_allclose(oracle.R_of(VR), g["R_lapack_signs"], atol=tol(dt))
    np.testing.assert_allclose(oracle.sign_normalise(oracle.R_of(VR)), g["R_positive_diag"], atol=tol(dt))
    np.testing.assert_allclose(tau, g["tau"].ravel(), atol=tol(dt))
    np.testing.assert_allclose([VR[1, 0], VR[2, 1]], g["v_below_diag"].ravel(), atol=tol(dt))
    assert VR[2, 0] == 0
    x = oracle.solve(VR, tau, g["b"].reshape(3, 1).astype(dt))
    np.testing.assert_allclose(x.ravel(), g["x"].ravel(), atol=tol(dt, 1e3))


# ---- (ii) special cases with closed forms --------------------------------------------------
@pytest.mark.parametrize("dt", DT)
def test_upper_triangular_input_is_fixed_point(dt):
    n = 9
    U = np.triu(rnd(n, n, 1, dt)) + 3 * np.eye(n, dtype=dt)
    A = np.vstack([U, np.zeros((4, n), dtype=dt)])
    VR, tau = oracle.qr(A)
    assert np.all(tau == 0)                       # every sub-column is exactly zero => H = I
    np.testing.assert_array_equal(oracle.R_of(VR), U)


@pytest.mark.parametrize("dt", DT)
def test_identity_over_mu_identity(dt):
    n, mu = 7, 0.25
    A = np.vstack([np.eye(n), mu * np.eye(n)]).astype(dt)
    VR, tau = oracle.qr(A)
    R = oracle.R_of(VR)
    np.testing.assert_allclose(np.abs(np.diag(R)), np.sqrt(1 + mu * mu), rtol=tol(dt))
    assert np.all(np.diag(R) < 0)                 # alpha = 1 >= 0 => beta = -norm
    np.testing.assert_allclose(R - np.diag(np.diag(R)), 0, atol=tol(dt))
    btop = np.arange(1, n + 1, dtype=dt)
    b = np.concatenate([btop, np.zeros(n, dtype=dt)]).reshape(-1, 1)
    x = oracle.solve(VR, tau, b)                  # Tikhonov shrink: x = b_top / (1 + mu^2)
    np.testing.assert_allclose(x.ravel(), btop / (1 + mu * mu), rtol=tol(dt, 1e3))


@pytest.mark.parametrize("dt", DT)
def test_zero_column_gives_tau_zero(dt):
    A = rnd(8, 4, 2, dt)
    A[:, 2] = 0                                   # an all-zero column stays zero under H_0 H_1
    VR, tau = oracle.qr(A)
    assert tau[2] == 0 and np.all(VR[:, 2] == 0)
    # a column that is zero below the diagonal when it is reached
    B = rnd(6, 3, 3, dt)
    B[1:, 0] = 0
    VR, tau = oracle.qr(B)
    assert tau[0] == 0 and VR[0, 0] == B[0, 0]
    np.testing.assert_array_equal(VR[:, 1:][0], B[0, 1:])   # H_0 = I leaves row 0 untouched


@pytest.mark.parametrize("dt", DT)
def test_tau_range_and_v_norm(dt):
    A = rnd(33, 17, 4, dt)
    VR, tau = oracle.qr(A)
    assert np.all((tau >= 1 - tol(dt)) & (tau <= 2 + tol(dt)))
    V = oracle.V_of(VR).astype(np.float64)
    np.testing.assert_allclose(tau * np.sum(V * V, axis=0), 2.0, rtol=tol(dt, 1e3))   # tau_j v_j^T v_j = 2


# ---- (iii) brute force: Gram-Schmidt -------------------------------------------------------
@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("shape", [(1, 1), (3, 2), (7, 4), (16, 16), (33, 17), (40, 40)])
def test_matches_gram_schmidt(dt, shape):
    m, n = shape
    A = rnd(m, n, 10 + m + n, dt)
    VR, tau = oracle.qr(A)
    _, Rg = cgs2(A)
    Rn = oracle.sign_normalise(oracle.R_of(VR).astype(np.float64))
    scale = np.linalg.norm(Rg)
    assert np.linalg.norm(Rn - Rg) / scale < tol(dt, 2e3)
    assert np.all(np.tril(oracle.R_of(VR), -1) == 0)


# ---- (iv) |diag R| = diag chol(A^T A); LAPACK as a library-routine pin -----------------------
@pytest.mark.parametrize("dt", DT)
def test_diag_matches_cholesky_and_lapack(dt):
    A = rnd(37, 19, 5, dt)
    VR, tau = oracle.qr(A)
    A64 = A.astype(np.float64)
    U = cholesky_upper(A64.T @ A64)
    np.testing.assert_allclose(np.abs(np.diag(VR[:19])), np.diag(U), rtol=tol(dt, 5e3))
    Rl = np.linalg.qr(A64, mode="r")
    np.testing.assert_allclose(oracle.sign_normalise(oracle.R_of(VR).astype(np.float64)),
                               oracle.sign_normalise(Rl), atol=tol(dt, 5e3) * np.linalg.norm(Rl))


# ---- (v) invariants ------------------------------------------------------------------------
@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("shape", [(3, 2), (16, 16), (33, 17), (64, 40)])
def test_orthogonality_and_backward_error(dt, shape):
    m, n = shape
    A = rnd(m, n, 20 + m, dt)
    VR, tau = oracle.qr(A)
    Q = oracle.form_q(VR, tau).astype(np.float64)
    R = oracle.R_of(VR).astype(np.float64)
    assert np.linalg.norm(Q.T @ Q - np.eye(n)) < tol(dt, 1e3)
    assert np.linalg.norm(A.astype(np.float64) - Q @ R) / np.linalg.norm(A) < tol(dt, 1e2)


@pytest.mark.parametrize("dt", DT)
def test_q_is_product_of_reflectors(dt):
    """Explicit H_0 H_1 ... built here with numpy equals what apply_q/apply_qt apply."""
    m, n = 9, 5
    A = rnd(m, n, 6, dt)
    VR, tau = oracle.qr(A)
    V = oracle.V_of(VR).astype(np.float64)
    Qfull = np.eye(m)
    for j in range(n):
        Qfull = Qfull @ householder_matrix(V[:, j], float(tau[j]))
    B = rnd(m, 3, 7, dt)
    np.testing.assert_allclose(oracle.apply_qt(VR, tau, B), Qfull.T @ B, atol=tol(dt, 1e3))
    np.testing.assert_allclose(oracle.apply_q(VR, tau, B), Qfull @ B, atol=tol(dt, 1e3))
    # Q^T A = [R; 0]
    QtA = oracle.apply_qt(VR, tau, A).astype(np.float64)
    np.testing.assert_allclose(QtA[:n], oracle.R_of(VR), atol=tol(dt, 1e3))
    np.testing.assert_allclose(QtA[n:], 0, atol=tol(dt, 1e3))


@pytest.mark.parametrize("dt", DT)
def test_apply_qt_preserves_norm_and_roundtrips(dt):
    A = rnd(40, 23, 8, dt)
    VR, tau = oracle.qr(A)
    B = rnd(40, 5, 9, dt)
    C = oracle.apply_qt(VR, tau, B)
    np.testing.assert_allclose(np.linalg.norm(C, axis=0), np.linalg.norm(B, axis=0), rtol=tol(dt, 1e2))
    np.testing.assert_allclose(oracle.apply_q(VR, tau, C), B, atol=tol(dt, 1e3))


# ---- T factor (a2) --------------------------------------------------------------------------
@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("j0,nb", [(0, 6), (3, 5), (8, 4)])
def test_larft_identities(dt, j0, nb):
    m, n = 30, 12
    A = rnd(m, n, 11, dt)
    VR, tau = oracle.qr(A)
    T = oracle.larft(VR, tau, j0, nb).astype(np.float64)
    V = oracle.V_of(VR).astype(np.float64)[:, j0:j0 + nb]
    t = tau[j0:j0 + nb].astype(np.float64)
    assert np.all(np.tril(T, -1) == 0)
    # T^{-1} = striu(V^T V) + diag(1/tau)
    Tinv = np.triu(V.T @ V, 1) + np.diag(1.0 / t)
    np.testing.assert_allclose(T @ Tinv, np.eye(nb), atol=tol(dt, 1e3))
    # I - V T V^T = H_{j0} ... H_{j0+nb-1}
    H = np.eye(m)
    for j in range(nb):
        H = H @ householder_matrix(V[:, j], t[j])
    np.testing.assert_allclose(np.eye(m) - V @ T @ V.T, H, atol=tol(dt, 1e3))


# ---- back-substitution ----------------------------------------------------------------------
@pytest.mark.parametrize("dt", DT)
def test_backsub_closed_forms(dt):
    n = 12
    C = rnd(n, 3, 12, dt)
    np.testing.assert_array_equal(oracle.backsub(np.eye(n, dtype=dt, order="F"), C), C)   # R = I
    # bidiagonal R = I + superdiag(-1): solution is the reversed cumulative sum of c
    R = np.eye(n) - np.diag(np.ones(n - 1), 1)
    c = np.arange(1, n + 1, dtype=np.float64).reshape(-1, 1)
    x = oracle.backsub(np.asfortranarray(R.astype(dt)), c.astype(dt))
    np.testing.assert_allclose(x.ravel(), np.cumsum(c[::-1])[::-1], rtol=tol(dt))
    # general: residual and comparison with forward substitution on the reversed system
    U = np.triu(rnd(n, n, 13, dt)) + 4 * np.eye(n, dtype=dt)
    X = oracle.backsub(np.asfortranarray(U), C).astype(np.float64)
    assert np.linalg.norm(U.astype(np.float64) @ X - C) / np.linalg.norm(C) < tol(dt, 1e2)
    L = U[::-1, ::-1].astype(np.float64); Cr = C[::-1].astype(np.float64)
    Y = np.zeros_like(Cr)
    for i in range(n):                             # forward substitution, written out
        Y[i] = (Cr[i] - L[i, :i] @ Y[:i]) / L[i, i]
    np.testing.assert_allclose(X, Y[::-1], rtol=tol(dt, 1e4), atol=tol(dt, 1e2))


@pytest.mark.parametrize("dt", DT)
def test_backsub_t_closed_forms_and_semi_normal_equations(dt):
    """The transposed substitution (R^T Y = C): identity, the bidiagonal closed form (now a running sum from the
    top), forward substitution written out, a transposed operand caught by an unsymmetric R, and the use it is
    made for -- R^{-1} R^{-T} (A^T b) is the least-squares solution (semi-normal equations) -- against lstsq."""
    n = 12
    C = rnd(n, 3, 21, dt)
    np.testing.assert_array_equal(oracle.backsub_t(np.eye(n, dtype=dt, order="F"), C), C)
    R = np.eye(n) - np.diag(np.ones(n - 1), 1)           # R^T = I - subdiag(1): y_j = c_j + y_{j-1}
    c = np.arange(1, n + 1, dtype=np.float64).reshape(-1, 1)
    y = oracle.backsub_t(np.asfortranarray(R.astype(dt)), c.astype(dt))
    np.testing.assert_allclose(y.ravel(), np.cumsum(c), rtol=tol(dt))
    U = np.triu(rnd(n, n, 22, dt)) + 4 * np.eye(n, dtype=dt)
    Y = oracle.backsub_t(np.asfortranarray(U), C).astype(np.float64)
    U64, C64 = U.astype(np.float64), C.astype(np.float64)
    Z = np.zeros_like(C64)
    for j in range(n):                                   # forward substitution with U^T, written out
        Z[j] = (C64[j] - U64[:j, j] @ Z[:j]) / U64[j, j]
    np.testing.assert_allclose(Y, Z, rtol=tol(dt, 1e4), atol=tol(dt, 1e2))
    assert np.linalg.norm(U64.T @ Y - C64) / np.linalg.norm(C64) < tol(dt, 1e2)
    assert np.linalg.norm(U64 @ Y - C64) / np.linalg.norm(C64) > 1e-2       # not the untransposed solve
    with pytest.raises(ZeroDivisionError):
        Us = np.triu(np.ones((4, 4))); Us[1, 1] = 0
        oracle.backsub_t(np.asfortranarray(Us), np.ones((4, 1)))
    # semi-normal equations on a full least-squares problem
    m, S = 40, 3
    A = rnd(m, n, 23, dt); B = rnd(m, S, 24, dt)
    VR, tau = oracle.qr(A)
    rhs = (A.astype(np.float64).T @ B.astype(np.float64)).astype(dt)
    X = oracle.backsub(VR, oracle.backsub_t(VR, rhs)).astype(np.float64)
    X_ls = np.linalg.lstsq(A.astype(np.float64), B.astype(np.float64), rcond=None)[0]
    assert np.linalg.norm(X - X_ls) / np.linalg.norm(X_ls) < tol(dt, 1e4)


def test_backsub_singular_raises():
    U = np.triu(np.ones((4, 4)))
    U[2, 2] = 0
    with pytest.raises(ZeroDivisionError):
        oracle.backsub(np.asfortranarray(U), np.ones((4, 1)))


# ---- whole solve ---------------------------------------------------------------------------
@pytest.mark.parametrize("dt", DT)
def test_exact_recovery_and_normal_equations(dt):
    m, n, S = 48, 20, 4
    A = rnd(m, n, 14, dt)
    X0 = rnd(n, S, 15, dt)
    A64 = A.astype(np.float64)
    VR, tau = oracle.qr(A)
    X = oracle.solve(VR, tau, (A64 @ X0.astype(np.float64)).astype(dt))
    assert np.linalg.norm(X - X0) / np.linalg.norm(X0) < tol(dt, 1e4)
    # noisy rhs: compare with the normal equations solved by the hand-written Cholesky
    B = rnd(m, S, 16, dt)
    X = oracle.solve(VR, tau, B).astype(np.float64)
    U = cholesky_upper(A64.T @ A64)
    rhs = A64.T @ B.astype(np.float64)
    Y = np.linalg.solve(U.T, rhs)
    Xn = np.linalg.solve(U, Y)
    assert np.linalg.norm(X - Xn) / np.linalg.norm(Xn) < tol(dt, 1e4)
    Xl = np.linalg.lstsq(A64, B.astype(np.float64), rcond=None)[0]
    assert np.linalg.norm(X - Xl) / np.linalg.norm(Xl) < tol(dt, 1e4)


@pytest.mark.parametrize("dt", DT)
def test_tiny_ct_case(dt):
    """N = 8 CT system (8 angles x 12 bins + 64 Tikhonov rows): the workload's shape."""
    from paper_2412_07631_b200 import workload as w
    cfg = w.CONFIGS["c0"]
    A, lam = w.dense_augmented(cfg, dtype=dt)
    X0, B = w.make_slices(cfg, consistent=True, lam=lam)
    VR, tau = oracle.qr(A)
    X = oracle.solve(VR, tau, B.astype(dt))
    assert np.linalg.norm(X - X0) / np.linalg.norm(X0) < tol(dt, 1e5)
    A64 = A.astype(np.float64)
    Q = oracle.form_q(VR, tau).astype(np.float64)
    assert np.linalg.norm(A64 - Q @ oracle.R_of(VR)) / np.linalg.norm(A64) < tol(dt, 1e2)
    # Tikhonov solution = argmin ||A x - b||^2 + lam ||x||^2 for the noisy rhs
    _, Bn = w.make_slices(cfg, lam=lam)
    Xn = oracle.solve(VR, tau, Bn.astype(dt)).astype(np.float64)
    A0 = A64[: cfg.m0]
    Xr = np.linalg.solve(A0.T @ A0 + (A64[cfg.m0, 0] ** 2) * np.eye(cfg.n), A0.T @ Bn[: cfg.m0])
    assert np.linalg.norm(Xn - Xr) / np.linalg.norm(Xr) < tol(dt, 1e5)


def test_fp32_oracle_really_computes_in_fp32():
    A = rnd(60, 30, 17, np.float32)
    VR32, _ = oracle.qr(A)
    VR64, _ = oracle.qr(A.astype(np.float64))
    d = np.linalg.norm(VR32.astype(np.float64) - VR64) / np.linalg.norm(VR64)
    assert VR32.dtype == np.float32 and 1e-9 < d < 1e-5


def test_argument_errors():
    with pytest.raises(ValueError):
        oracle.qr(np.zeros((2, 3)))                # m < n
    with pytest.raises(TypeError):
        oracle.qr(np.zeros((3, 2), dtype=np.int32))
