"""Seeded synthetic CT workloads (inputs only -- none of the QR method's arithmetic lives here).

This module is the one piece shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_2412_07631_b200.binding``): it produces the system matrix A, the Tikhonov
augmentation, the phantoms and the noisy sinograms that both sides consume.  It imports
neither of them.

What the paper uses (Table 1, L208-232 Table 5): a fan-beam scanner matrix
built with Joseph's projector and sinograms simulated from the COVID-CT-MD / DICOM-CT-PD
data sets with Poisson noise (L210).  Those data sets are not available here; BASELINE.json
fixes the stand-in workloads (``configs``) reproduced below: parallel-beam Siddon
intersection lengths, random-ellipse phantoms, Poisson noise at I0 photons, and a
sqrt(lambda)*I block appended to A (lambda = 1e-3 * ||A||_F^2 / n).  DESIGN.md section
"Input recipe" states every convention.

Geometry conventions (readings 10-12):
  * pixel size 1, image square [-N/2, N/2]^2; pixel (r, c), r = 0 at the top, covers
    x in [c - N/2, c + 1 - N/2], y in [N/2 - r - 1, N/2 - r]; unknown index j = r*N + c
  * angle theta_a = a*pi/n_ang; detector axis u = (cos, sin); ray direction w = (-sin, cos)
  * bin k passes through s_k*u with s_k = k - (n_bins - 1)/2; ray (row) index i = a*n_bins + k
  * a segment belongs to the pixel that contains its midpoint (floor rule), segments whose
    midpoint falls outside the image or whose length is not positive are dropped.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

__all__ = [
    "CTConfig", "CONFIGS", "FanBeamConfig", "FAN_CONFIGS", "siddon_coo", "joseph_fanbeam_coo", "fanbeam_dense", "fanbeam_slices", "tikhonov_lambda", "dense_augmented", "dense_augmented_device",
    "ellipse_phantom", "make_slices", "chord_length", "psnr", "snr", "ssim", "shard_slices",
]


@dataclass(frozen=True)
class CTConfig:
    """One BASELINE.json config: N x N image, n_ang x n_bins rays, S slices, I0 photons."""
    name: str
    cfg_id: int
    N: int
    n_ang: int
    n_bins: int
    S: int
    I0: float

    @property
    def n(self) -> int:
        return self.N * self.N

    @property
    def m0(self) -> int:
        return self.n_ang * self.n_bins

    @property
    def m(self) -> int:
        return self.m0 + self.n

    def factor_flops(self) -> float:
        """2mn^2 - 2n^3/3 (BASELINE.json north_star)."""
        m, n = float(self.m), float(self.n)
        return 2.0 * m * n * n - 2.0 * n ** 3 / 3.0

    def solve_flops(self, S: int | None = None) -> float:
        """(4mn - n^2) * S: Q^T b costs 4mn - 2n^2, back-substitution n^2 per slice."""
        m, n = float(self.m), float(self.n)
        return (4.0 * m * n - n * n) * float(self.S if S is None else S)


# BASELINE.json "configs" (bins = ceil(sqrt(2)*N)); plus a tiny "c0" used only by tests.
CONFIGS = {
    "c0": CTConfig("c0", 0, 8, 8, 12, 4, 1e4),
    "c1": CTConfig("c1", 1, 32, 30, 46, 8, 1e4),
    "c2": CTConfig("c2", 2, 64, 60, 91, 64, 5e3),
    "c3": CTConfig("c3", 3, 128, 90, 182, 256, 5e3),
    "c4": CTConfig("c4", 4, 256, 120, 363, 512, 2e3),
    "c5": CTConfig("c5", 5, 384, 180, 544, 1024, 2e3),
}


def _angle_dirs(a: int, n_ang: int):
    """(u, w) for angle index a, exact at 0 and 90 degrees."""
    if a == 0:
        return (1.0, 0.0), (0.0, 1.0)
    if 2 * a == n_ang:
        return (0.0, 1.0), (-1.0, 0.0)
    th = a * math.pi / n_ang
    ct, st = math.cos(th), math.sin(th)
    return (ct, st), (-st, ct)


def siddon_coo(N: int, n_ang: int, n_bins: int):
    """Siddon ray/pixel intersection lengths of the un-augmented A as COO triplets.

    Returns (rows int64, cols int64, vals float64) with rows in [0, n_ang*n_bins) and
    cols in [0, N*N).  (row, col) pairs may repeat only for numerically zero slivers at
    pixel corners; consumers must accumulate duplicates.
    """
    half = N / 2.0
    grid = np.arange(N + 1, dtype=np.float64) - half          # grid line coordinates
    s = np.arange(n_bins, dtype=np.float64) - (n_bins - 1) / 2.0
    out_r, out_c, out_v = [], [], []
    for a in range(n_ang):
        (ux, uy), (wx, wy) = _angle_dirs(a, n_ang)
        ts = []
        if wx != 0.0:
            ts.append((grid[None, :] - s[:, None] * ux) / wx)
        if wy != 0.0:
            ts.append((grid[None, :] - s[:, None] * uy) / wy)
        t = np.sort(np.concatenate(ts, axis=1), axis=1)       # (n_bins, #crossings)
        seg = t[:, 1:] - t[:, :-1]
        tm = 0.5 * (t[:, 1:] + t[:, :-1])
        xm = s[:, None] * ux + tm * wx
        ym = s[:, None] * uy + tm * wy
        c = np.floor(xm + half).astype(np.int64)
        r = np.floor(half - ym).astype(np.int64)
        ok = (seg > 0.0) & (c >= 0) & (c < N) & (r >= 0) & (r < N)
        k_idx, _ = np.nonzero(ok)
        out_r.append(a * n_bins + k_idx)
        out_c.append(r[ok] * N + c[ok])
        out_v.append(seg[ok])
    return (np.concatenate(out_r).astype(np.int64),
            np.concatenate(out_c).astype(np.int64),
            np.concatenate(out_v))


def chord_length(N: int, n_ang: int, n_bins: int) -> np.ndarray:
    """Closed-form length of each ray inside the image square (used to pin the generator).

    Rays lying exactly on the boundary lines x = +N/2 or y = -N/2 count as missing, rays on
    x = -N/2 or y = +N/2 as inside (the midpoint/floor tie rule).
    """
    half = N / 2.0
    s = np.arange(n_bins, dtype=np.float64) - (n_bins - 1) / 2.0
    out = np.zeros((n_ang, n_bins))
    for a in range(n_ang):
        (ux, uy), (wx, wy) = _angle_dirs(a, n_ang)
        lo = np.full(n_bins, -np.inf)
        hi = np.full(n_bins, np.inf)
        for (p0, d) in ((s * ux, wx), (s * uy, wy)):
            if d == 0.0:
                continue
            t1 = (-half - p0) / d
            t2 = (half - p0) / d
            lo = np.maximum(lo, np.minimum(t1, t2))
            hi = np.minimum(hi, np.maximum(t1, t2))
        length = np.maximum(hi - lo, 0.0)
        if wx == 0.0:   # vertical ray at x = s
            length = np.where((s >= -half) & (s < half), length, 0.0)
        if wy == 0.0:   # horizontal ray at y = s
            length = np.where((s > -half) & (s <= half), length, 0.0)
        out[a] = length
    return out.reshape(-1)


# ----------------------------------------------------------------------------------------
# The paper's own geometry at reduced scale: fan beam, Joseph's projector
# (Table 1: 360 degree circular scan, source-to-isocentre 75 cm, source-to-
# detector 150 cm, fan angle 30 degrees, 1025 detectors, 512 x 512 pixels, 260 views; Table 5,
# L222-232, is the same with 65 cm / 33 degrees).  No Tikhonov block: like the paper, the number
# of views is chosen so that A has full column rank (L93-95).
#
# Readings (the paper gives the distances but not the pixel size, the detector shape or the
# details of the projector):
#   * pixel size 1 and the image square as in the Siddon conventions above; the fan covers the
#     circle circumscribed to the image, radius N / sqrt(2), so the source-to-isocentre distance is
#     D = (N / sqrt 2) / sin(fan / 2) pixels; the detector is an arc of n_det equal angles
#     (gamma_k = (k - (n_det - 1)/2) * fan / n_det), so the source-to-detector distance does not
#     enter the ray geometry;
#   * view v has the source at angle beta_v = 2 pi v / n_views, position D (cos beta, sin beta);
#     the ray of detector k leaves it in direction beta_v + pi + gamma_k; row index i = v n_det + k;
#   * Joseph's method: a ray with |dx| >= |dy| is sampled at every pixel-column centre, where the
#     image is interpolated linearly between the two nearest row centres, each sample weighted
#     by the path length per column 1 / |dx|; otherwise the same over rows.  Equivalently
#     a_ij = (1 / |dx|) * hat(row coordinate of the ray at column c(j) - r(j)), hat(t) = max(0, 1 - |t|);
#     samples whose neighbour lies outside the image keep only the inside weight.
# ----------------------------------------------------------------------------------------
@dataclass(frozen=True)
class FanBeamConfig:
    name: str
    N: int
    n_det: int
    n_views: int
    S: int
    fan_deg: float = 30.0

    @property
    def n(self) -> int:
        return self.N * self.N

    @property
    def m(self) -> int:
        return self.n_det * self.n_views


# Table 1 scaled down with the same proportions (detectors = 2 N + 1); the paper's 260 views for 512 x 512 are
# m / n = 1.017.  With the fan covering the circumscribed circle many outer rays only graze the corners, so at this
# scale full rank needs m / n of about 1.2 (19 views at N = 32: cond 2.7e4; 21: 2.9e3; 24: 7.9e2) -- the behaviour the
# paper reports in L93-95 and L240-242 (a few more views needed for a well-conditioned single-precision solve).
FAN_CONFIGS = {
    "fan32": FanBeamConfig("fan32", 32, 65, 24, 8),
    "fan64": FanBeamConfig("fan64", 64, 129, 48, 16),
    "fan128": FanBeamConfig("fan128", 128, 257, 96, 64),
}


def joseph_fanbeam_coo(N: int, n_det: int, n_views: int, fan_deg: float = 30.0):
    """Joseph-projector weights of the fan-beam scanner as COO triplets (rows int64 in [0, n_views * n_det),
    cols int64 in [0, N * N), vals float64); no duplicates."""
    half = N / 2.0
    fan = math.radians(fan_deg)
    D = (N / math.sqrt(2.0)) / math.sin(fan / 2.0)
    gam = (np.arange(n_det, dtype=np.float64) - (n_det - 1) / 2.0) * (fan / n_det)
    centres = (np.arange(N, dtype=np.float64) + 0.5) - half      # x of column c; y of row r is -centres[r]
    idx = np.arange(N, dtype=np.int64)
    out_r, out_c, out_v = [], [], []
    for v in range(n_views):
        beta = 2.0 * math.pi * v / n_views
        sx, sy = D * math.cos(beta), D * math.sin(beta)
        phi = beta + math.pi + gam
        dx, dy = np.cos(phi), np.sin(phi)
        hor = np.abs(dx) >= np.abs(dy)
        for sel, along_x in ((hor, True), (~hor, False)):
            ks = np.nonzero(sel)[0]
            if ks.size == 0:
                continue
            if along_x:      # sample at column centres x_c: y = sy + (x_c - sx) dy / dx, fractional row = N/2 - y - 1/2
                L = 1.0 / np.abs(dx[ks])
                t = half - (sy + (centres[None, :] - sx) * (dy[ks] / dx[ks])[:, None]) - 0.5
            else:            # sample at row centres y_r = -centres[r]: x = sx + (y_r - sy) dx / dy, fractional column = x + N/2 - 1/2
                L = 1.0 / np.abs(dy[ks])
                t = (sx + (-centres[None, :] - sy) * (dx[ks] / dy[ks])[:, None]) + half - 0.5
            i0 = np.floor(t).astype(np.int64)
            w1 = t - i0
            for other, w in ((i0, 1.0 - w1), (i0 + 1, w1)):
                ok = (other >= 0) & (other < N) & (w > 0.0)
                kk, jj = np.nonzero(ok)
                out_r.append(v * n_det + ks[kk])
                out_c.append(other[ok] * N + idx[jj] if along_x else idx[jj] * N + other[ok])
                out_v.append((L[:, None] * w)[ok])
    return (np.concatenate(out_r).astype(np.int64), np.concatenate(out_c).astype(np.int64), np.concatenate(out_v))


def fanbeam_dense(cfg: FanBeamConfig, dtype=np.float64, coo=None) -> np.ndarray:
    """Dense column-major A (m x n) of a fan-beam config, generated in fp64 and rounded once to ``dtype``."""
    rows, cols, vals = coo if coo is not None else joseph_fanbeam_coo(cfg.N, cfg.n_det, cfg.n_views, cfg.fan_deg)
    A = np.zeros((cfg.m, cfg.n), dtype=np.float64, order="F")
    A[rows, cols] = vals
    return np.asfortranarray(A.astype(dtype))


def fanbeam_slices(cfg: FanBeamConfig, S: int | None = None, coo=None, I0: float | None = None):
    """Phantoms X0 (n, S) and sinograms B = A X0 (m, S), fp64 Fortran order; seeds default_rng(7000 + N + slice).
    I0 = None: noiseless, consistent (the paper's full-dose regime, Tables 2-3); else Poisson noise at I0 photons
    with kappa = 4 / N as in make_slices (its low-dose regime, L208-212)."""
    import scipy.sparse as sp
    S = cfg.S if S is None else S
    rows, cols, vals = coo if coo is not None else joseph_fanbeam_coo(cfg.N, cfg.n_det, cfg.n_views, cfg.fan_deg)
    A = sp.coo_matrix((vals, (rows, cols)), shape=(cfg.m, cfg.n)).tocsr()
    X0 = np.zeros((cfg.n, S), order="F")
    B = np.zeros((cfg.m, S), order="F")
    kappa = 4.0 / cfg.N
    for sl in range(S):
        rng = np.random.default_rng(7000 + cfg.N + sl)
        x = ellipse_phantom(cfg.N, rng).reshape(-1)
        X0[:, sl] = x
        p = A @ x
        if I0 is None:
            B[:, sl] = p
        else:
            y = rng.poisson(I0 * np.exp(-kappa * p)).astype(np.float64)
            B[:, sl] = -np.log(np.maximum(y, 1.0) / I0) / kappa
    return X0, B


def tikhonov_lambda(vals: np.ndarray, n: int) -> float:
    """lambda = 1e-3 * ||A||_F^2 / n with ||A||_F of the un-augmented A (fp64)."""
    return 1e-3 * float(np.sum(vals.astype(np.float64) ** 2)) / float(n)


def dense_augmented(cfg: CTConfig, dtype=np.float64, coo=None):
    """Dense column-major A_aug = [A; sqrt(lambda) I] of shape (m, n) as a Fortran array.

    Generated in fp64 and rounded once to ``dtype``.  Returns (A, lam)."""
    rows, cols, vals = coo if coo is not None else siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    lam = tikhonov_lambda(vals, cfg.n)
    A = np.zeros((cfg.m, cfg.n), dtype=np.float64, order="F")
    np.add.at(A, (rows, cols), vals)
    A[cfg.m0 + np.arange(cfg.n), np.arange(cfg.n)] = math.sqrt(lam)
    return np.asfortranarray(A.astype(dtype)), lam


def dense_augmented_device(cfg: CTConfig, torch_dtype, coo=None, device="cuda", lda: int | None = None):
    """Same matrix as ``dense_augmented`` but scattered straight into device memory (the dense
    matrix of the larger configs is too big to stage through numpy).  Returns (At, lam) where
    ``At`` is a torch tensor of shape (n, lda) whose memory is the column-major m x n A_aug with
    leading dimension lda (default m).  Duplicates are accumulated in fp64 before the single
    rounding to ``torch_dtype``, like the host builder."""
    import torch
    rows, cols, vals = coo if coo is not None else siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    lam = tikhonov_lambda(vals, cfg.n)
    lda = cfg.m if lda is None else lda
    # accumulate duplicate (row, col) pairs on the host in fp64 (they are rare corner slivers)
    key = cols * np.int64(lda) + rows
    uk, inv = np.unique(key, return_inverse=True)
    acc = np.zeros(uk.shape[0], dtype=np.float64)
    np.add.at(acc, inv, vals)
    At = torch.zeros((cfg.n, lda), dtype=torch_dtype, device=device)
    flat = At.view(-1)
    flat[torch.from_numpy(uk).to(device)] = torch.from_numpy(acc).to(device).to(torch_dtype)
    d = torch.arange(cfg.n, device=device, dtype=torch.int64)
    flat[d * lda + cfg.m0 + d] = torch.tensor(math.sqrt(lam), dtype=torch.float64).to(torch_dtype).item()
    return At, lam


def ellipse_phantom(N: int, rng: np.random.Generator) -> np.ndarray:
    """Random-ellipse phantom (SURVEY.md 8c reading 13), values in [0, 1], max = 1."""
    K = int(rng.integers(5, 11))
    half = N / 2.0
    xs = (np.arange(N) + 0.5) - half                 # pixel-centre x for column c
    ys = half - (np.arange(N) + 0.5)                 # pixel-centre y for row r
    X, Y = np.meshgrid(xs, ys)
    img = np.zeros((N, N), dtype=np.float64)
    for _ in range(K):
        cx, cy = rng.uniform(-0.5, 0.5, size=2) * half
        ax, by = rng.uniform(0.05, 0.4, size=2) * half
        phi = rng.uniform(0.0, math.pi)
        rho = rng.uniform(0.1, 1.0)
        cp, sp = math.cos(phi), math.sin(phi)
        xr = (X - cx) * cp + (Y - cy) * sp
        yr = -(X - cx) * sp + (Y - cy) * cp
        img += rho * ((xr / ax) ** 2 + (yr / by) ** 2 <= 1.0)
    mx = img.max()
    if mx > 0:
        img /= mx
    return img


def make_slices(cfg: CTConfig, S: int | None = None, coo=None, noise: bool = True,
                consistent: bool = False, lam: float | None = None):
    """Phantoms X0 (n, S) and augmented right-hand sides B (m, S), both fp64 Fortran order.

    noise=True:  b = -ln(max(y,1)/I0)/kappa, y ~ Poisson(I0 exp(-kappa A x)), kappa = 4/N,
                 bottom n rows zero (SURVEY.md 8c reading 14).
    consistent=True: b_aug = A_aug x = [A x; sqrt(lambda) x] (reading 21; exact recovery).
    Seeds: numpy default_rng(1000*cfg_id + slice)."""
    import scipy.sparse as sp
    S = cfg.S if S is None else S
    rows, cols, vals = coo if coo is not None else siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    A0 = sp.coo_matrix((vals, (rows, cols)), shape=(cfg.m0, cfg.n)).tocsr()
    if lam is None:
        lam = tikhonov_lambda(vals, cfg.n)
    kappa = 4.0 / cfg.N
    X0 = np.zeros((cfg.n, S), order="F")
    B = np.zeros((cfg.m, S), order="F")
    for sl in range(S):
        rng = np.random.default_rng(1000 * cfg.cfg_id + sl)
        x = ellipse_phantom(cfg.N, rng).reshape(-1)
        X0[:, sl] = x
        p = A0 @ x
        if consistent:
            B[: cfg.m0, sl] = p
            B[cfg.m0:, sl] = math.sqrt(lam) * x
        elif noise:
            y = rng.poisson(cfg.I0 * np.exp(-kappa * p)).astype(np.float64)
            B[: cfg.m0, sl] = -np.log(np.maximum(y, 1.0) / cfg.I0) / kappa
        else:
            B[: cfg.m0, sl] = p
    return X0, B


def shard_slices(S: int, rank: int, world: int):
    """Contiguous, balanced share of S independent slices for `rank` of `world` (first S % world
    ranks get one more).  Returns (first slice, count).  The solve shards over right-hand sides with
    no exchange step."""
    base, extra = divmod(S, world)
    return rank * base + min(rank, extra), base + (1 if rank < extra else 0)


# ----------------------------------------------------------------------------------------
# Reported image-quality metrics (Eq. 4-7).  Reporting only.
# ----------------------------------------------------------------------------------------
def snr(ref: np.ndarray, img: np.ndarray) -> float:
    """Eq. 4: 10 log10( sum I0^2 / sum (I0 - I)^2 )."""
    ref = np.asarray(ref, dtype=np.float64); img = np.asarray(img, dtype=np.float64)
    den = float(np.sum((ref - img) ** 2))
    return float("inf") if den == 0 else 10.0 * math.log10(float(np.sum(ref ** 2)) / den)


def psnr(ref: np.ndarray, img: np.ndarray, vmax: float = 1.0) -> float:
    """Eq. 5-6: 10 log10(MAX^2 / MSE); MAX = 1 (normalised phantom)."""
    ref = np.asarray(ref, dtype=np.float64); img = np.asarray(img, dtype=np.float64)
    mse = float(np.mean((ref - img) ** 2))
    return float("inf") if mse == 0 else 10.0 * math.log10(vmax * vmax / mse)


def ssim(ref: np.ndarray, img: np.ndarray, L: float = 1.0, win: int = 7) -> float:
    """Eq. 7 averaged over all valid win x win windows, uniform weights,
    sample (N-1) variances, c1 = (0.01 L)^2, c2 = (0.03 L)^2 (SURVEY.md 8c reading 19)."""
    x = np.asarray(ref, dtype=np.float64); y = np.asarray(img, dtype=np.float64)
    c1, c2 = (0.01 * L) ** 2, (0.03 * L) ** 2
    npx = win * win

    def box(a):
        cs = np.cumsum(np.cumsum(np.pad(a, ((1, 0), (1, 0))), axis=0), axis=1)
        return cs[win:, win:] - cs[:-win, win:] - cs[win:, :-win] + cs[:-win, :-win]

    sx, sy = box(x), box(y)
    mx, my = sx / npx, sy / npx
    vx = (box(x * x) - sx * mx) / (npx - 1)
    vy = (box(y * y) - sy * my) / (npx - 1)
    cxy = (box(x * y) - sx * my) / (npx - 1)
    s = ((2 * mx * my + c1) * (2 * cxy + c2)) / ((mx * mx + my * my + c1) * (vx + vy + c2))
    return float(np.mean(s))
