"""Factor persistence (the factorisation is computed once per
scanner geometry and reused for every later batch of slices): ct_qr_save / ct_qr_load through the C-ABI.

A loaded handle must hold bit-for-bit the factor that was saved (the file is a copy, no arithmetic),
and its solves must meet the same gates against the oracle as the solves of the factoring handle -- with
the factor read back into HBM, and with a device budget too small for it (file mapped, panels streamed)."""
import os

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


def factor_parts(f):
    P = f.stats()["n_panels"]
    return dict(R=ctqr.ct_qr_get_R(f), V=ctqr.ct_qr_get_V(f), tau=ctqr.ct_qr_get_tau(f),
                T=[ctqr.ct_qr_get_T(f, k) for k in range(P)])


def assert_same_factor(a, b):
    for k in ("R", "V", "tau"):
        assert np.array_equal(a[k], b[k]), k
    assert len(a["T"]) == len(b["T"]) and all(np.array_equal(x, y) for x, y in zip(a["T"], b["T"]))


def solve(f, B, dt):
    S = B.shape[1]
    X = np.zeros((f.n, S), dtype=dt, order="F")
    ctqr.ct_qr_solve(f, np.asfortranarray(B.astype(dt)), S, X)
    return X


def streamed_budget(m, nb, dt):
    # smaller than the factor, large enough to be a legal option value
    return 4 * nb * m * np.dtype(dt).itemsize


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("shape,nb,ib", [((517, 259), 0, 0), ((700, 650), 32, 16), ((1300, 1300), 0, 0), ((40, 7), 8, 8)])
def test_round_trip_in_core_and_streamed(tmp_path, shape, nb, ib, dt):
    m, n = shape
    rng = np.random.default_rng(77)
    A = np.asfortranarray(rng.standard_normal((m, n)).astype(dt))
    VR, tau_o = oracle.qr(A)
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m, n, nb=nb, ib=ib)
    nb_eff = f.stats()["nb"]
    ref = factor_parts(f)
    path = str(tmp_path / "factor.ctqr")
    ctqr.ct_qr_save(f, path)
    w = np.dtype(dt).itemsize
    ld = -(-m // (16 // w)) * (16 // w)
    P = -(-n // nb_eff)
    assert os.path.getsize(path) == 4096 + (ld * n + 2 * P * nb_eff * nb_eff + n) * w
    Bs = {S: np.asfortranarray(rng.standard_normal((m, S)).astype(dt)) for S in (1, 8, 19)}
    X_by_S = {S: solve(f, B, dt) for S, B in Bs.items()}
    f.destroy()                                        # the loaded handles below share nothing with it

    g = ctqr.ct_qr_load(path)                          # factor read back into HBM
    st = g.stats()
    assert (g.m, g.n, g.np_dtype) == (m, n, dt) and st["nb"] == nb_eff and st["out_of_core"] == 0
    assert st["factor_ms"] == 0.0
    assert_same_factor(ref, factor_parts(g))
    for S, B in Bs.items():
        X = solve(g, B, dt)
        assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
        assert relerr(X, X_by_S[S]) <= ROUND[dt]
    g.destroy()

    if n > 4 * nb_eff:                                 # budget below the factor: file mapped, panels streamed (a5)
        s = ctqr.ct_qr_load(path, device_budget_bytes=streamed_budget(m, nb_eff, dt))
        assert s.stats()["out_of_core"] == 1
        assert_same_factor(ref, factor_parts(s))
        for S, B in Bs.items():
            X = solve(s, B, dt)
            assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
            assert relerr(X, X_by_S[S]) <= ROUND[dt]
        C = Bs[19].copy(order="F"); ctqr.ct_qr_apply_qt(s, C, 19)
        assert relerr(C, oracle.apply_qt(VR, tau_o, Bs[19])) <= ROUND[dt]
        s.destroy()


@pytest.mark.parametrize("dt", DT)
def test_save_from_out_of_core_handle(tmp_path, dt):
    """A factor that was computed out of core (it lives in the caller's host buffer) saves to the same
    file, byte for byte, as the in-core factor of the same matrix would through get_V / get_R."""
    m, n, nb, S = 700, 650, 32, 9
    rng = np.random.default_rng(5)
    A = np.asfortranarray(rng.standard_normal((m, n)).astype(dt))
    B = np.asfortranarray(rng.standard_normal((m, S)).astype(dt))
    w = np.dtype(dt).itemsize
    lds = -(-m // (16 // w)) * (16 // w)
    Ah = ctqr.colmajor_from_numpy(A, device="cpu", pin=True)
    f = ctqr.ct_qr_factor(Ah, m, n, nb=nb, ib=16, device_budget_bytes=(2 * 160 + 2 * nb) * lds * w + 64)
    assert f.stats()["out_of_core"] == 1
    ref = factor_parts(f)
    path = str(tmp_path / "ooc.ctqr")
    ctqr.ct_qr_save(f, path)
    f.destroy()
    g = ctqr.ct_qr_load(path)
    assert g.stats()["out_of_core"] == 0
    assert_same_factor(ref, factor_parts(g))
    VR, tau_o = oracle.qr(A)
    assert relerr(solve(g, B, dt), oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]
    assert relerr(ref["V"], oracle.V_of(VR)) <= ROUND[dt]


@pytest.mark.parametrize("dt", DT)
def test_ct_config_factor_once_solve_later(tmp_path, dt):
    """BASELINE.json configs[0]: factor the geometry, save, and reconstruct the slices from the file in a
    'later session' -- in two batches, as the paper's service mode does."""
    c = wl.CONFIGS["c1"]
    coo = wl.siddon_coo(c.N, c.n_ang, c.n_bins)
    A, lam = wl.dense_augmented(c, dt, coo)
    X0, B = wl.make_slices(c, coo=coo, lam=lam)
    B = np.asfortranarray(B.astype(dt))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), c.m, c.n)
    path = str(tmp_path / "geom.ctqr")
    ctqr.ct_qr_save(f, path)
    f.destroy()
    g = ctqr.ct_qr_load(path)
    h = c.S // 2
    X = np.concatenate([solve(g, B[:, :h], dt), solve(g, B[:, h:], dt)], axis=1)
    VR, tau_o = oracle.qr(A)
    assert relerr(X, oracle.solve(VR, tau_o, B)) <= SOLUTION[dt]


def test_load_rejects_truncated_and_foreign_files(tmp_path):
    A = np.asfortranarray(np.random.default_rng(0).standard_normal((300, 200)))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), 300, 200)
    path = tmp_path / "f.ctqr"
    ctqr.ct_qr_save(f, str(path))
    data = path.read_bytes()
    (tmp_path / "cut.ctqr").write_bytes(data[:-8])
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_load(str(tmp_path / "cut.ctqr"))
    assert ei.value.code == 3
    bad = bytearray(data); bad[40] ^= 0xFF             # n in the header
    (tmp_path / "bad.ctqr").write_bytes(bytes(bad))
    with pytest.raises(ctqr.CtqrError) as ei:
        ctqr.ct_qr_load(str(tmp_path / "bad.ctqr"))
    assert ei.value.code == 3
    with pytest.raises(ctqr.CtqrError) as ei:          # unwritable destination: nothing is left behind
        ctqr.ct_qr_save(f, str(tmp_path / "no_such_dir" / "f.ctqr"))
    assert ei.value.code == 3


@pytest.mark.parametrize("dt", DT)
@pytest.mark.parametrize("streamed", [False, True])
def test_band_promise_travels_with_the_file(tmp_path, dt, streamed):
    """A factor computed under opt->lower_bandwidth keeps it across save / load: the reloaded handle reports it
    and its solves (which stop every panel at the band) still match the dense oracle."""
    m0, n, S = 500, 700, 10
    rng = np.random.default_rng(12)
    A0 = rng.standard_normal((m0, n)) * (rng.random((m0, n)) < 0.3)
    A = np.asfortranarray(np.vstack([A0, 0.4 * np.eye(n)]).astype(dt))
    B = np.asfortranarray(rng.standard_normal((m0 + n, S)).astype(dt))
    f = ctqr.ct_qr_factor(ctqr.colmajor_from_numpy(A), m0 + n, n, lower_bandwidth=m0)
    ref = factor_parts(f)
    path = str(tmp_path / "band.ctqr")
    ctqr.ct_qr_save(f, path)
    f.destroy()
    g = ctqr.ct_qr_load(path, device_budget_bytes=streamed_budget(m0 + n, 128, dt) if streamed else 0)
    st = g.stats()
    assert st["lower_bandwidth"] == m0 and st["out_of_core"] == int(streamed)
    assert_same_factor(ref, factor_parts(g))
    VR, tau_o = oracle.qr(A)
    for s_cols in (3, S):                               # fused small-S kernel (in core) and the per-panel path
        X = solve(g, B[:, :s_cols], dt)
        assert relerr(X, oracle.solve(VR, tau_o, B[:, :s_cols])) <= SOLUTION[dt]
