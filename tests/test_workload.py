"""Generator invariants (SURVEY.md section 8c pins for the Siddon generator, rung T1).
The generator is an input, not the method under test, but it is pinned all the same."""
import math

import numpy as np
import pytest

from paper_2412_07631_b200 import workload as w


@pytest.mark.parametrize("name", ["c0", "c1", "c2"])
def test_row_sums_equal_chord_lengths(name):
    cfg = w.CONFIGS[name]
    r, c, v = w.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    rs = np.bincount(r, weights=v, minlength=cfg.m0)
    np.testing.assert_allclose(rs, w.chord_length(cfg.N, cfg.n_ang, cfg.n_bins), atol=1e-12 * cfg.N)
    assert v.min() > 0 and v.max() <= math.sqrt(2) + 1e-12
    assert np.bincount(r, minlength=cfg.m0).max() <= 2 * cfg.N - 1 + 2   # + corner slivers
    assert c.min() >= 0 and c.max() < cfg.n


def test_config_shapes_match_baseline_json():
    exp = {"c1": (2404, 1024), "c2": (9556, 4096), "c3": (32764, 16384),
           "c4": (109096, 65536), "c5": (245376, 147456)}
    for k, (m, n) in exp.items():
        assert (w.CONFIGS[k].m, w.CONFIGS[k].n) == (m, n)
        assert w.CONFIGS[k].n_bins == math.ceil(math.sqrt(2) * w.CONFIGS[k].N)


def test_axis_aligned_rays_even_bins():
    """theta = 0 with an even number of bins: every in-image ray crosses N pixels of length 1."""
    N, n_ang, n_bins = 8, 4, 12
    r, c, v = w.siddon_coo(N, n_ang, n_bins)
    sel = r < n_bins                                 # angle 0
    np.testing.assert_allclose(v[sel], 1.0, atol=1e-14)
    cnt = np.bincount(r[sel], minlength=n_bins)
    assert set(cnt.tolist()) <= {0, N} and (cnt == N).sum() == N


def test_total_mass_per_angle_is_image_area():
    cfg = w.CONFIGS["c1"]
    r, c, v = w.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    per_angle = np.bincount(r // cfg.n_bins, weights=v, minlength=cfg.n_ang)
    assert np.all(np.abs(per_angle / cfg.n - 1) < 5e-3)


def test_rotation_symmetry_90_degrees():
    """A[a + n_ang/2, k, pixel (N-1-c, r)] = A[a, k, pixel (r, c)] (even n_bins)."""
    cfg = w.CONFIGS["c1"]
    N, nb, na = cfg.N, cfg.n_bins, cfg.n_ang
    A, _ = w.dense_augmented(cfg)
    A0 = A[: cfg.m0].reshape(na, nb, N, N)
    for a in (1, 3, 7):
        rot = np.rot90(A0[a], k=1, axes=(1, 2))      # (r, c) -> (N-1-c, r)
        np.testing.assert_allclose(A0[a + na // 2], rot, atol=1e-12)


def test_lambda_and_augmentation():
    cfg = w.CONFIGS["c0"]
    r, c, v = w.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    lam = w.tikhonov_lambda(v, cfg.n)
    A, lam2 = w.dense_augmented(cfg)
    assert lam == lam2 and A.shape == (cfg.m, cfg.n) and A.flags.f_contiguous
    np.testing.assert_allclose(lam, 1e-3 * np.sum(A[: cfg.m0] ** 2) / cfg.n, rtol=1e-13)
    np.testing.assert_allclose(A[cfg.m0:], math.sqrt(lam) * np.eye(cfg.n), atol=0)
    A32, _ = w.dense_augmented(cfg, dtype=np.float32)
    np.testing.assert_array_equal(A32, A.astype(np.float32))
    # survey probe values: lambda at c1
    r, c, v = w.siddon_coo(32, 30, 46)
    assert abs(w.tikhonov_lambda(v, 1024) - 0.02841) < 1e-5


def test_slices_are_seeded_and_shaped():
    cfg = w.CONFIGS["c0"]
    X0, B = w.make_slices(cfg)
    X1, B1 = w.make_slices(cfg)
    np.testing.assert_array_equal(B, B1)
    assert X0.shape == (cfg.n, cfg.S) and B.shape == (cfg.m, cfg.S)
    assert np.all(B[cfg.m0:] == 0) and X0.max() == 1.0 and X0.min() >= 0
    _, Bc = w.make_slices(cfg, consistent=True)
    A, lam = w.dense_augmented(cfg)
    np.testing.assert_allclose(A @ X0, Bc, atol=1e-12)


def test_poisson_noise_statistics():
    """Counts y ~ Poisson(I0 exp(-kappa p)): the log-transformed data is unbiased to O(1/y)."""
    cfg = w.CONFIGS["c1"]
    X0, Bn = w.make_slices(cfg, S=4)
    _, Bc = w.make_slices(cfg, S=4, noise=False)
    d = (Bn - Bc)[: cfg.m0]
    kappa = 4.0 / cfg.N
    var_pred = np.exp(kappa * Bc[: cfg.m0]) / cfg.I0 / kappa ** 2
    z = d / np.sqrt(var_pred)
    assert abs(z.mean()) < 0.05 and abs(z.std() - 1) < 0.05


def test_metrics_closed_forms():
    rng = np.random.default_rng(0)
    x = rng.uniform(size=(16, 16))
    assert w.ssim(x, x) == pytest.approx(1.0)
    assert w.psnr(x, x + 0.01) == pytest.approx(40.0)           # MSE = 1e-4, MAX = 1
    assert w.snr(x, x + 0.01) == pytest.approx(10 * math.log10(np.sum(x * x) / (256 * 1e-4)))
    assert w.ssim(x, 1 - x) < 0.5


# ---- fan-beam Joseph generator (the paper's own geometry, Table 1) ----------
def _fan_dense(N, n_det, n_views, fan_deg=30.0):
    r, c, v = w.joseph_fanbeam_coo(N, n_det, n_views, fan_deg)
    assert len(set(zip(r.tolist(), c.tolist()))) == len(r)            # no duplicate entries
    A = np.zeros((n_det * n_views, N * N))
    A[r, c] = v
    return A


def test_joseph_equals_the_hat_function_form_pixel_by_pixel():
    """Brute force on a tiny scanner, written pixel-driven instead of ray-driven: a_ij = (1 / |d_major|) *
    max(0, 1 - |coordinate of the ray on the sampling line through pixel j - pixel centre|)."""
    N, n_det, n_views, fan_deg = 6, 9, 7, 40.0
    A = _fan_dense(N, n_det, n_views, fan_deg)
    fan = math.radians(fan_deg)
    D = (N / math.sqrt(2)) / math.sin(fan / 2)
    B = np.zeros_like(A)
    for v in range(n_views):
        beta = 2 * math.pi * v / n_views
        sx, sy = D * math.cos(beta), D * math.sin(beta)
        for k in range(n_det):
            phi = beta + math.pi + (k - (n_det - 1) / 2) * fan / n_det
            dx, dy = math.cos(phi), math.sin(phi)
            for r in range(N):
                for c in range(N):
                    px, py = c + 0.5 - N / 2, N / 2 - r - 0.5        # pixel centre
                    if abs(dx) >= abs(dy):                           # sampling line x = px: distance along y
                        dist, L = abs(sy + (px - sx) * dy / dx - py), 1 / abs(dx)
                    else:                                            # sampling line y = py: distance along x
                        dist, L = abs(sx + (py - sy) * dx / dy - px), 1 / abs(dy)
                    B[v * n_det + k, r * N + c] = L * max(0.0, 1.0 - dist)
    np.testing.assert_allclose(A, B, atol=1e-12)


def test_joseph_central_ray_and_basic_invariants():
    N, n_det, n_views = 16, 33, 12
    A = _fan_dense(N, n_det, n_views)
    assert A.min() >= 0 and A.max() <= math.sqrt(2) + 1e-12 and (A != 0).sum(axis=1).max() <= 2 * N
    # view 0, central detector: the ray is the x axis; every column gives 1/2 to the two middle rows
    row = A[(n_det - 1) // 2].reshape(N, N)
    expect = np.zeros((N, N)); expect[N // 2 - 1] = 0.5; expect[N // 2] = 0.5
    np.testing.assert_allclose(row, expect, atol=1e-12)
    # row sums are the chord through the image up to the two end samples: |sum - chord| <= 2 / |d_major|
    fan = math.radians(30.0)
    D = (N / math.sqrt(2)) / math.sin(fan / 2)
    for v in (0, 1, 5):
        beta = 2 * math.pi * v / n_views
        sx, sy = D * math.cos(beta), D * math.sin(beta)
        for k in range(n_det):
            phi = beta + math.pi + (k - (n_det - 1) / 2) * fan / n_det
            dx, dy = math.cos(phi), math.sin(phi)
            lo, hi = -math.inf, math.inf
            for p0, d in ((sx, dx), (sy, dy)):
                if d != 0:
                    t1, t2 = (-N / 2 - p0) / d, (N / 2 - p0) / d
                    lo, hi = max(lo, min(t1, t2)), min(hi, max(t1, t2))
            chord = max(hi - lo, 0.0)
            assert abs(A[v * n_det + k].sum() - chord) <= 2.0 / max(abs(dx), abs(dy)) + 1e-9


def test_joseph_quarter_turn_symmetry():
    """A quarter turn of the source is a quarter turn of the image: A[v + n_views/4, k, rot(pixel)] = A[v, k, pixel]."""
    N, n_det, n_views = 12, 25, 8
    A = _fan_dense(N, n_det, n_views).reshape(n_views, n_det, N, N)
    for v in range(n_views):
        # rotating the scene by +90 degrees maps the point (x, y) to (-y, x): pixel (r, c) -> (N - 1 - c, r)
        rotated = np.rot90(A[v], k=1, axes=(1, 2))
        np.testing.assert_allclose(A[(v + n_views // 4) % n_views], rotated, atol=1e-12)


def test_fan_config_is_full_rank_like_the_papers():
    cfg = w.FAN_CONFIGS["fan32"]
    A = w.fanbeam_dense(cfg)
    assert A.shape == (cfg.m, cfg.n) == (1560, 1024)
    s = np.linalg.svd(A, compute_uv=False)
    assert s[-1] > 1e-2 and s[0] / s[-1] < 2e3
    X0, B = w.fanbeam_slices(cfg, S=2)
    np.testing.assert_allclose(A @ X0, B, atol=1e-10)
    assert X0.max() == 1.0 and B.min() >= 0
