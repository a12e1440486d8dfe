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
