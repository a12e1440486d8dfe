"""fp32 factor + fp64 iterative refinement (Table 3: the
fp32 / fp64 quality gap the paper studies).  ct_qr_solve_refined reaches a result that has a plain definition -- the
fp64 least-squares solution of the fp64 system -- so the oracle is that definition: oracle.qr + oracle.solve in fp64.
Gate: the north_star fp64 solution gate, ||X - X_oracle64|| / ||X_oracle64|| <= 1e-9, from an fp32 factor within
three sweeps; the transposed triangular solve it is built on is compared with oracle.backsub_t on its own."""
import numpy as np
import pytest
import scipy.sparse as sp

import oracle
import paper_2412_07631_b200 as ctqr
from paper_2412_07631_b200 import workload as wl

pytestmark = pytest.mark.gpu

FP64_GATE = 1e-9


def relerr(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def worst_col(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return float(np.max(np.linalg.norm(a - b, axis=0) / np.linalg.norm(b, axis=0)))


@pytest.mark.parametrize("dt", [np.float64, np.float32])
@pytest.mark.parametrize("shape,nb,exact", [((700, 384), 0, False), ((700, 384), 0, True), ((517, 259), 0, False),
                                            ((300, 130), 32, False), ((60, 40), 0, False)])
def test_trsm_t_matches_the_oracle(shape, nb, exact, dt):
    m, n = shape
    rng = np.random.default_rng(m + 7 * n)
    A = np.asfortranarray(rng.standard_normal((m, n)).astype(dt))
    S = 11
    C = np.asfortranarray(rng.standard_normal((n, S)).astype(dt))
    VR, tau = oracle.qr(A)
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n, nb=nb, ib=16 if nb else 0, trsm_exact=exact)
    Y = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_trsm_t(f, C, S, Y)
    tol = 1e-10 if dt == np.float64 else 2e-3          # cond(R) of a random m x n matrix times the unit roundoff
    assert relerr(Y, oracle.backsub_t(VR, C)) <= tol
    # and the pair of solves is the normal-equations solve: R^{-1} R^{-T} (A^T b) = argmin ||A x - b||
    B = rng.standard_normal((m, S)).astype(dt)
    rhs = np.asfortranarray((A.astype(np.float64).T @ B.astype(np.float64)).astype(dt))
    X = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_trsm_t(f, rhs, S, Y)
    ctqr.ct_qr_trsm(f, Y, S, X)
    assert relerr(X, oracle.solve(VR, tau, np.asfortranarray(B))) <= (1e-9 if dt == np.float64 else 5e-2)
    f.destroy()


def ct_problem(name, S, consistent):
    c = wl.CONFIGS[name]
    coo = wl.siddon_coo(c.N, c.n_ang, c.n_bins)
    rows, cols, vals = coo
    A64, lam = wl.dense_augmented(c, np.float64, coo)
    X0, B = wl.make_slices(c, S=S, coo=coo, lam=lam, consistent=consistent)
    A0 = sp.coo_matrix((vals, (rows, cols)), shape=(c.m0, c.n)).tocsr()
    Acsr = sp.vstack([A0, np.sqrt(lam) * sp.identity(c.n, format="csr")]).tocsr()
    return c, A64, B, X0, Acsr


@pytest.mark.parametrize("consistent", [False, True], ids=["noisy", "consistent"])
@pytest.mark.parametrize("name", ["c0", "c1"])
def test_refined_fp32_factor_meets_the_fp64_gate(name, consistent):
    """BASELINE.json configs[0] (and the tiny c0): the fp32 factor alone is 1e-5 away from the fp64 oracle solution;
    three fp64 refinement sweeps bring every slice inside the fp64 gate."""
    c, A64, B, X0, Acsr = ct_problem(name, 8 if name == "c1" else 4, consistent)
    S = B.shape[1]
    VR, tau = oracle.qr(A64)
    X_or = oracle.solve(VR, tau, B)
    A32 = np.asfortranarray(A64.astype(np.float32))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A32), c.m, c.n)
    X = np.zeros((c.n, S), order="F")
    info0 = ctqr.ct_qr_solve_refined(f, np.asfortranarray(B), S, X, A_csr=Acsr, max_iters=0)
    e0 = relerr(X, X_or)
    assert info0["iters_done"] == 0 and 1e-8 < e0 <= 1e-3          # plain fp32 solve: the fp32 gate, not the fp64 one
    info = ctqr.ct_qr_solve_refined(f, np.asfortranarray(B), S, X, A_csr=Acsr, max_iters=3)
    assert info["iters_done"] == 3
    assert relerr(X, X_or) <= FP64_GATE and worst_col(X, X_or) <= FP64_GATE, (relerr(X, X_or), info)
    assert info["correction"][0] > 10 * info["correction"][2]       # the corrections shrink sweep by sweep
    # early stop on the correction norm
    info = ctqr.ct_qr_solve_refined(f, np.asfortranarray(B), S, X, A_csr=Acsr, max_iters=10, tol=1e-11)
    assert info["converged"] and info["iters_done"] <= 6
    assert relerr(X, X_or) <= FP64_GATE
    if consistent:                                                   # the paper's regime: exact recovery of the phantom
        assert relerr(X, X0) <= 1e-9
    # dense fp64 operator on the device: same result
    import torch
    Ad = ctqr.colmajor_from_numpy(A64)
    Xd = torch.zeros((S, c.n), dtype=torch.float64, device="cuda")
    Bd = ctqr.colmajor_from_numpy(B)
    ctqr.ct_qr_solve_refined(f, Bd, S, Xd, A_dense=Ad, max_iters=3)
    assert relerr(ctqr.numpy_from_colmajor(Xd), X_or) <= FP64_GATE
    f.destroy()


def test_refined_general_matrix_and_fp64_handle():
    """Not CT-shaped: a random sparse overdetermined system with an inconsistent right-hand side; and an fp64 handle,
    where the first correction is already at rounding level."""
    rng = np.random.default_rng(12)
    m, n, S = 900, 300, 5
    Acsr = (sp.random(m, n, density=0.05, random_state=3, format="csr") + sp.vstack([sp.identity(n), sp.csr_matrix((m - n, n))])).tocsr()
    A64 = np.asfortranarray(Acsr.toarray())
    B = np.asfortranarray(rng.standard_normal((m, S)))
    VR, tau = oracle.qr(A64)
    X_or = oracle.solve(VR, tau, B)
    X = np.zeros((n, S), order="F")
    f32 = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A64.astype(np.float32)), m, n)
    info = ctqr.ct_qr_solve_refined(f32, B, S, X, A_csr=Acsr, max_iters=4)
    assert relerr(X, X_or) <= FP64_GATE, (relerr(X, X_or), info)
    f32.destroy()
    f64 = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A64), m, n)
    info = ctqr.ct_qr_solve_refined(f64, B, S, X, A_csr=Acsr, max_iters=1)
    assert relerr(X, X_or) <= 1e-12 and info["correction"][0] <= 1e-11
    f64.destroy()


def test_refined_argument_errors():
    rng = np.random.default_rng(1)
    m, n = 60, 20
    A = np.asfortranarray(rng.standard_normal((m, n)))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A.astype(np.float32)), m, n)
    B = np.asfortranarray(rng.standard_normal((m, 2))); X = np.zeros((n, 2), order="F")
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_solve_refined(f, B, 2, X)                          # no operator
    assert ei.value.code == -4
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_solve_refined(f, B, 2, X, A_csr=sp.csr_matrix(np.ones((m + 1, n))))   # wrong shape
    assert ei.value.code == -2
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_solve_refined(f, B, 2, X, A_csr=sp.csr_matrix(A), max_iters=-1)
    assert ei.value.code == -11
    f.destroy()
