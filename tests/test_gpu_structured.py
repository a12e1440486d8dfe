"""Structure-aware factorisation: with opt->lower_bandwidth = kl the caller promises
A(i, j) == 0 for i - j > kl -- for the Tikhonov-augmented [A0; sqrt(lambda) I] of the configs, kl = m0.
Householder QR keeps that profile, so the library stops every panel and trailing update at row
kl + (last column of the block).  The skipped work is arithmetic on exact zeros: the factor must equal the
dense oracle's to rounding, the solve must meet the same gates, and a broken promise must be refused."""
import numpy as np
import pytest

import oracle
import paper_2412_07631_b200 as ctqr
from paper_2412_07631_b200 import workload as wl

pytestmark = pytest.mark.gpu

DT = [np.float64, np.float32]
SOLUTION = {np.float64: 1e-9, np.float32: 1e-3}
ROUND = {np.float64: 1e-11, np.float32: 5e-4}


def relerr(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (den if den > 0 else 1.0)


def banded_flops(m, n, kl):
    return sum(4.0 * (min(m, kl + j + 1) - j) * (n - j - 1) for j in range(n))


def check(A, B, dt, kl, **opts):
    m, n = A.shape
    S = B.shape[1]
    A = np.asfortranarray(A.astype(dt)); B = np.asfortranarray(B.astype(dt))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n, lower_bandwidth=kl, **opts)
    st = f.stats()
    assert st["lower_bandwidth"] == kl
    assert st["factor_flops_performed"] == pytest.approx(banded_flops(m, n, kl), rel=1e-12)
    assert st["factor_flops_performed"] < st["factor_flops"]
    X = np.zeros((n, S), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, B, S, X)
    VR, tau = oracle.qr(A)                              # the dense oracle: same factor, same convention
    assert relerr(ctqr.ct_qr_get_R(f), oracle.R_of(VR)) <= ROUND[dt]
    V = ctqr.ct_qr_get_V(f)
    assert relerr(V, oracle.V_of(VR)) <= ROUND[dt]
    assert relerr(ctqr.ct_qr_get_tau(f), tau) <= ROUND[dt]
    ii, jj = np.indices(V.shape)
    assert np.all(V[ii - jj > kl] == 0)                 # the profile survived: nothing was written below the band
    assert relerr(X, oracle.solve(VR, tau, B)) <= SOLUTION[dt]
    C = B.copy(order="F"); ctqr.ct_qr_apply_qt(f, C, S)
    assert relerr(C, oracle.apply_qt(VR, tau, B)) <= ROUND[dt]
    return f


def augmented(rng, m0, n, dt, density=0.3):
    A0 = rng.standard_normal((m0, n)) * (rng.random((m0, n)) < density)
    return np.vstack([A0, 0.37 * np.eye(n)]).astype(dt)


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("m0,n,nb,ib,la", [(40, 30, 8, 8, 1), (300, 260, 32, 16, 1), (300, 260, 32, 16, 0),
                                           (130, 517, 64, 16, 1), (1200, 1100, 0, 0, 1), (700, 1300, 0, 0, 1)])
def test_augmented_identity_block(m0, n, nb, ib, la, dt):
    """[A0; c I] with m0 above, below and far below n; nb = 128 cases take the two-panel (256-wide) driver."""
    rng = np.random.default_rng(m0 + n)
    A = augmented(rng, m0, n, dt)
    B = rng.standard_normal((m0 + n, 11))
    check(A, B, dt, kl=m0, nb=nb, ib=ib, lookahead=la)


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("kl", [1, 37, 128, 400])
def test_general_lower_band_profile(kl, dt):
    """Any matrix with A(i, j) = 0 for i - j > kl, not only an identity block (m = 900, n = 640)."""
    m, n = 900, 640
    rng = np.random.default_rng(kl)
    A = rng.standard_normal((m, n))
    ii, jj = np.indices(A.shape)
    A[ii - jj > kl] = 0
    A[jj > ii] *= 0.05                                  # a random dense upper triangle is exponentially ill-conditioned:
    A[ii == jj] += 3.0                                  # keep the narrow-band cases solvable in fp32
    check(A, rng.standard_normal((m, 5)), dt, kl=kl, nb=32, ib=16)
    check(A, rng.standard_normal((m, 5)), dt, kl=kl)


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("cfg", ["c1", "c2"])
def test_ct_config_structured(cfg, dt):
    """BASELINE.json configs[0], configs[1] with kl = n_ang * n_bins."""
    c = wl.CONFIGS[cfg]
    coo = wl.siddon_coo(c.N, c.n_ang, c.n_bins)
    A, lam = wl.dense_augmented(c, dt, coo)
    _, B = wl.make_slices(c, coo=coo, lam=lam)
    m0 = c.m - c.n
    f = check(A, B, dt, kl=m0)
    # c1: m0 = 1380 vs n = 1024 -> 2 m0 n^2 + ... against 2 m n^2 - 2 n^3 / 3
    st = f.stats()
    assert st["factor_flops_performed"] / st["factor_flops"] < 0.85


def test_broken_promise_is_refused_and_wide_band_is_dense():
    rng = np.random.default_rng(3)
    A = augmented(rng, 200, 150, np.float64)
    A[330, 17] = 1e-30                                  # below the band of kl = 200 (330 - 17 > 200)
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), 350, 150, lower_bandwidth=200)
    assert ei.value.code == -6 and "column 17" in str(ei.value)
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), 350, 150, lower_bandwidth=-1)
    assert ei.value.code == -6
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), 350, 150, lower_bandwidth=349)   # no zero is promised
    st = f.stats()
    assert st["lower_bandwidth"] == 0 and st["factor_flops_performed"] == st["factor_flops"]


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("nb,ns,pinned", [(32, 160, True), (64, 128, False)])
def test_out_of_core_uses_the_band(nb, ns, pinned, dt):
    """Host-resident [A0; c I] with a capped device budget (a5): the promise is checked per super-panel, the
    streamed reflector panels end at the band, so fewer bytes cross the host link than without the promise."""
    m0, n, S = 420, 650, 9
    m = m0 + n
    rng = np.random.default_rng(8)
    A = np.asfortranarray(augmented(rng, m0, n, dt))
    B = np.asfortranarray(rng.standard_normal((m, S)).astype(dt))
    w = np.dtype(dt).itemsize
    lds = -(-m // (16 // w)) * (16 // w)
    budget = (2 * ns + 2 * nb) * lds * w + 64
    VR, tau_o = oracle.qr(A)
    h2d = {}
    for kl in (0, m0):
        Ah = ctqr.colmajor_from_numpy(A, device="cpu", pin=pinned)
        f = ctqr.ct_qr_factor(Ah, m, n, nb=nb, ib=16, device_budget_bytes=budget, lower_bandwidth=kl)
        st = f.stats()
        assert st["out_of_core"] == 1 and st["n_superpanels"] == -(-n // ns) and st["lower_bandwidth"] == kl
        h2d[kl] = st["h2d_bytes"]
        X = np.zeros((n, S), dtype=dt, order="F")
        ctqr.ct_qr_solve(f, B, S, X)
        assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
        assert relerr(ctqr.ct_qr_get_R(f), oracle.R_of(VR)) <= ROUND[dt]
        assert relerr(ctqr.ct_qr_get_V(f), oracle.V_of(VR)) <= ROUND[dt]
        C = B.copy(order="F"); ctqr.ct_qr_apply_qt(f, C, S)
        assert relerr(C, oracle.apply_qt(VR, tau_o, B)) <= ROUND[dt]
        f.destroy()
    assert h2d[m0] < 0.95 * h2d[0]          # shorter streamed panels, minus the streamed pass that verifies the promise


def test_out_of_core_broken_promise_in_a_later_super_panel():
    m0, n, nb, ns = 300, 400, 32, 128
    rng = np.random.default_rng(9)
    A = np.asfortranarray(augmented(rng, m0, n, np.float64))
    A[m0 + n - 1, 300] = 0.5                            # column 300 lives in the third super-panel
    lds = m0 + n
    Ah = ctqr.colmajor_from_numpy(A, device="cpu", pin=True)
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_factor(Ah, m0 + n, n, nb=nb, ib=16, device_budget_bytes=(2 * ns + 2 * nb) * lds * 8 + 64,
                          lower_bandwidth=m0)
    assert ei.value.code == -6 and "column 300" in str(ei.value)
    # the promise is verified on the whole matrix before the first write-back: a refused input is left untouched
    assert np.array_equal(ctqr.numpy_from_colmajor(Ah), A)
