"""Seeded synthetic inputs for parallel-beam FBP (shared by the tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic (no filter, no back-projection, no
interpolation).  It only synthesises what the paper calls the projections P_theta(t)
(rays ``x cos(theta) + y sin(theta) = t``) for phantoms made of
ellipses, using the textbook closed form of the Radon transform of an ellipse
(Kak & Slaney ch. 3 = ref [8]; restated in SURVEY.md section 8(c)), plus
the Lambert-Beer count model of PAPER.md:43-47 (eq. 1) for Poisson noise.

It depends on numpy only; it imports neither ``oracle/`` nor the CUDA binding, so both
sides can be fed the same bytes.

The paper's own workload (13 DTU / Visible-Human sinograms) is not
available; the five configurations of BASELINE.json stand in for it (recipe: DESIGN.md
section "Inputs").
"""
from __future__ import annotations

import hashlib
import math
from dataclasses import dataclass

import numpy as np

# ---------------------------------------------------------------------------------------
# Phantoms.  Columns: rho (additive density), A, B (semi-axes), x0, y0 (centre),
# alpha (rotation of the A axis from +x, radians).  Unit-square coordinates [-1, 1]^2.
# ---------------------------------------------------------------------------------------

#: SURVEY.md section 8(d): the survey's own 10-ellipse head-like stand-in ("HEAD10"):
#: a high-contrast shell with low-contrast interior features.  Image range 0...1.
HEAD10 = np.array(
    [
        (1.00, 0.80, 0.90, 0.00, 0.00, 0.0),
        (-0.75, 0.74, 0.84, 0.00, 0.00, 0.0),
        (-0.10, 0.25, 0.12, 0.30, 0.25, 0.6),
        (-0.10, 0.25, 0.12, -0.30, 0.25, -0.6),
        (0.05, 0.15, 0.15, 0.00, -0.35, 0.0),
        (0.05, 0.06, 0.10, 0.00, 0.05, 0.0),
        (0.02, 0.04, 0.04, -0.12, -0.60, 0.0),
        (0.02, 0.03, 0.03, 0.00, -0.60, 0.0),
        (0.02, 0.05, 0.025, 0.12, -0.60, 0.0),
        (0.10, 0.08, 0.05, 0.45, -0.20, 1.0),
    ],
    dtype=np.float64,
)


def random_ellipses(seed: int, n: int = 10) -> np.ndarray:
    """SURVEY.md section 8(d) generator for configs 3 and 4 (draw order is part of the recipe)."""
    rng = np.random.default_rng(seed)
    out = np.empty((n, 6), dtype=np.float64)
    for e in range(n):
        r = 0.7 * math.sqrt(rng.random())
        phi = 2.0 * math.pi * rng.random()
        a = rng.uniform(0.05, 0.4)
        b = rng.uniform(0.05, 0.4)
        alpha = rng.uniform(0.0, math.pi)
        rho = rng.uniform(-0.5, 1.0)
        out[e] = (rho, a, b, r * math.cos(phi), r * math.sin(phi), alpha)
    return out


def disk(radius_unit: float, rho: float = 1.0) -> np.ndarray:
    """A centred disk as a one-row ellipse table (pins P3 / P10 of SURVEY.md section 8(c))."""
    return np.array([(rho, radius_unit, radius_unit, 0.0, 0.0, 0.0)], dtype=np.float64)


# ---------------------------------------------------------------------------------------
# Geometry helpers (conventions G6-G8 of SURVEY.md section 8(c); they describe the INPUT
# sampling, the reconstruction itself lives in oracle/ and in the CUDA library).
# ---------------------------------------------------------------------------------------

def uniform_angles(n_angles: int, span: float = math.pi) -> np.ndarray:
    """theta_i = i*span/K, i = 0..K-1, end point excluded (G8)."""
    return np.arange(n_angles, dtype=np.float64) * (span / n_angles)


def detector_coords(n_det: int, det_spacing: float = 1.0) -> np.ndarray:
    """t_j = (j - (D-1)/2) * d  (G7: detector centred)."""
    return (np.arange(n_det, dtype=np.float64) - 0.5 * (n_det - 1)) * det_spacing


def default_n_det(image_n: int) -> int:
    """D = ceil(N*sqrt(2)) as in every BASELINE.json config (91, 363, 725, 2897)."""
    return int(math.ceil(image_n * math.sqrt(2.0)))


def ellipse_sinogram(
    ellipses: np.ndarray,
    angles: np.ndarray,
    n_det: int,
    det_spacing: float = 1.0,
    scale: float = 1.0,
) -> np.ndarray:
    """Analytic parallel-beam sinogram P[K][D] (fp64), point-sampled at bin centres (G15).

    ``scale`` maps phantom units to detector-length units (N/2 * pixel_size for a
    unit-square phantom shown on an N x N image): lengths, centres and therefore P scale
    with it.  Closed form per ellipse: P = 2 rho A B sqrt(a^2 - tau^2) / a^2 for
    |tau| <= a, with a^2 = A^2 cos^2(theta-alpha) + B^2 sin^2(theta-alpha) and
    tau = t - x0 cos(theta) - y0 sin(theta).
    """
    ellipses = np.atleast_2d(np.asarray(ellipses, dtype=np.float64))
    angles = np.asarray(angles, dtype=np.float64)
    t = detector_coords(n_det, det_spacing)[None, :]
    c = np.cos(angles)[:, None]
    s = np.sin(angles)[:, None]
    sino = np.zeros((angles.size, n_det), dtype=np.float64)
    for rho, a_ax, b_ax, x0, y0, alpha in ellipses:
        a_ax, b_ax, x0, y0 = a_ax * scale, b_ax * scale, x0 * scale, y0 * scale
        ca = np.cos(angles - alpha)[:, None]
        sa = np.sin(angles - alpha)[:, None]
        a2 = (a_ax * ca) ** 2 + (b_ax * sa) ** 2
        tau = t - x0 * c - y0 * s
        inside = a2 - tau * tau
        sino += np.where(inside > 0.0, 2.0 * rho * a_ax * b_ax * np.sqrt(np.maximum(inside, 0.0)) / a2, 0.0)
    return sino


def rasterise(ellipses: np.ndarray, image_n: int, pixel_size: float = 1.0, scale: float | None = None) -> np.ndarray:
    """Phantom sampled at pixel centres, image[r][c] with row <-> +y, column <-> +x (G6)."""
    ellipses = np.atleast_2d(np.asarray(ellipses, dtype=np.float64))
    if scale is None:
        scale = 0.5 * image_n * pixel_size
    ax = (np.arange(image_n, dtype=np.float64) - 0.5 * (image_n - 1)) * pixel_size
    x = ax[None, :]
    y = ax[:, None]
    img = np.zeros((image_n, image_n), dtype=np.float64)
    for rho, a_ax, b_ax, x0, y0, alpha in ellipses:
        dx = x - x0 * scale
        dy = y - y0 * scale
        xr = dx * math.cos(alpha) + dy * math.sin(alpha)
        yr = -dx * math.sin(alpha) + dy * math.cos(alpha)
        img += np.where((xr / (a_ax * scale)) ** 2 + (yr / (b_ax * scale)) ** 2 <= 1.0, rho, 0.0)
    return img


def region_masks(ellipses: np.ndarray, image_n: int, margin_px: float, pixel_size: float = 1.0):
    """For pin P11: (label image, interior mask).  A pixel is 'interior' when it is at least
    ``margin_px`` pixels (conservatively, measured through the ellipse level set) away from
    every ellipse boundary, so its true density is constant in a neighbourhood."""
    ellipses = np.atleast_2d(np.asarray(ellipses, dtype=np.float64))
    scale = 0.5 * image_n * pixel_size
    ax = (np.arange(image_n, dtype=np.float64) - 0.5 * (image_n - 1)) * pixel_size
    x = ax[None, :]
    y = ax[:, None]
    label = np.zeros((image_n, image_n), dtype=np.int64)
    interior = np.ones((image_n, image_n), dtype=bool)
    for e, (rho, a_ax, b_ax, x0, y0, alpha) in enumerate(ellipses):
        dx = x - x0 * scale
        dy = y - y0 * scale
        xr = dx * math.cos(alpha) + dy * math.sin(alpha)
        yr = -dx * math.sin(alpha) + dy * math.cos(alpha)
        a_px, b_px = a_ax * scale, b_ax * scale
        m = margin_px * pixel_size
        inside_shrunk = (xr / max(a_px - m, 1e-9)) ** 2 + (yr / max(b_px - m, 1e-9)) ** 2 <= 1.0
        outside_grown = (xr / (a_px + m)) ** 2 + (yr / (b_px + m)) ** 2 > 1.0
        inside = (xr / a_px) ** 2 + (yr / b_px) ** 2 <= 1.0
        label += inside.astype(np.int64) << e
        interior &= np.where(a_px > m and b_px > m, inside_shrunk, False) | outside_grown
    return label, interior


# ---------------------------------------------------------------------------------------
# Noise models
# ---------------------------------------------------------------------------------------

def poisson_noise(sino: np.ndarray, image_n: int, i0: float, seed: int) -> np.ndarray:
    """Lambert-Beer counts (eq. 1) with the unit convention G14 and the
    zero-count clamp G13 of SURVEY.md section 8(c):
    I ~ Poisson(I0 * exp(-P/(N/2))),  P_noisy = -(N/2) * ln(max(I, 1) / I0)."""
    rng = np.random.default_rng(seed)
    half = 0.5 * image_n
    counts = rng.poisson(i0 * np.exp(-sino / half)).astype(np.float64)
    return -half * np.log(np.maximum(counts, 1.0) / i0)


def gaussian_noise(sino: np.ndarray, rel_sigma: float, seed: int) -> np.ndarray:
    """Additive N(0, (rel_sigma * max P)^2) noise (config 4)."""
    rng = np.random.default_rng(seed)
    return sino + rng.normal(0.0, rel_sigma * float(np.max(sino)), size=sino.shape)


# ---------------------------------------------------------------------------------------
# The five BASELINE.json configurations
# ---------------------------------------------------------------------------------------

@dataclass(frozen=True)
class Config:
    name: str
    image_n: int
    n_angles: int
    n_det: int
    batch: int
    dtypes: tuple
    description: str


CONFIGS = {
    1: Config("cfg1", 64, 90, 91, 1, ("f32",), "HEAD10 analytic sinogram, noiseless"),
    2: Config("cfg2", 256, 180, 363, 1, ("f32",), "HEAD10, Poisson I0=1e5 (seed 2)"),
    3: Config("cfg3", 512, 360, 725, 1, ("f32", "f64"), "10 random ellipses (seed 3), noiseless -- headline"),
    4: Config("cfg4", 512, 720, 725, 64, ("f32",), "64 slices, random ellipses (seed 4000+s), Gaussian 1% (seed 4100+s)"),
    5: Config("cfg5", 2048, 1800, 2897, 1, ("f32", "f64"), "HEAD10, Poisson I0=1e6 (seed 5)"),
}


def config_angles(cfg_id: int) -> np.ndarray:
    return uniform_angles(CONFIGS[cfg_id].n_angles)


def config_slice(cfg_id: int, s: int = 0) -> np.ndarray:
    """fp64 sinogram [K][D] of slice ``s`` of a config (d = pixel = 1, theta_i = i*pi/K)."""
    cfg = CONFIGS[cfg_id]
    ang = uniform_angles(cfg.n_angles)
    half = 0.5 * cfg.image_n
    if cfg_id == 1:
        return ellipse_sinogram(HEAD10, ang, cfg.n_det, 1.0, half)
    if cfg_id == 2:
        return poisson_noise(ellipse_sinogram(HEAD10, ang, cfg.n_det, 1.0, half), cfg.image_n, 1e5, 2)
    if cfg_id == 3:
        return ellipse_sinogram(random_ellipses(3), ang, cfg.n_det, 1.0, half)
    if cfg_id == 4:
        clean = ellipse_sinogram(random_ellipses(4000 + s), ang, cfg.n_det, 1.0, half)
        return gaussian_noise(clean, 0.01, 4100 + s)
    if cfg_id == 5:
        return poisson_noise(ellipse_sinogram(HEAD10, ang, cfg.n_det, 1.0, half), cfg.image_n, 1e6, 5)
    raise KeyError(cfg_id)


def config_sinogram(cfg_id: int, n_slices: int | None = None) -> np.ndarray:
    """fp64 sinogram stack [B][K][D] (all slices of the config, or the first ``n_slices``)."""
    cfg = CONFIGS[cfg_id]
    b = cfg.batch if n_slices is None else n_slices
    return np.stack([config_slice(cfg_id, s) for s in range(b)], axis=0)


def random_sinogram(seed: int, batch: int, n_angles: int, n_det: int) -> np.ndarray:
    """Unstructured N(0,1) sinogram for linearity / adjoint / odd-shape parity cases."""
    return np.random.default_rng(seed).standard_normal((batch, n_angles, n_det))


def sha256(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


# ---------------------------------------------------------------------------------------
# Cone-beam inputs for the FDK row: analytic line integrals of balls.
# Geometry as include/fbp.h "fbp_fdk_reconstruct": source at -sad * e_s(beta), e_s = (-sin, cos, 0); flat virtual
# detector through the rotation axis spanned by e_a = (cos, sin, 0) and e_z, centred, spacings d_a and d_b.
# ---------------------------------------------------------------------------------------

def ball_cone_projections(balls, angles, sad, n_a, n_b, d_a=1.0, d_b=1.0) -> np.ndarray:
    """P[K][n_b][n_a] (fp64): sum over balls (rho, radius, x0, y0, z0) of rho * chord length of the ray from the
    source through the detector point (a_j, b_i); chord = 2 sqrt(radius^2 - dist^2), dist = distance from the
    ball's centre to the ray (closed form; point-sampled at the detector pixel centres)."""
    balls = np.atleast_2d(np.asarray(balls, dtype=np.float64))
    angles = np.asarray(angles, dtype=np.float64)
    a = detector_coords(n_a, d_a)[None, None, :]
    b = detector_coords(n_b, d_b)[None, :, None]
    cb, sb = np.cos(angles)[:, None, None], np.sin(angles)[:, None, None]
    # source S = -sad * e_s, detector point D = a e_a + b e_z, direction v = D - S
    sx, sy = sad * sb, -sad * cb
    vx, vy, vz = a * cb - sx, a * sb - sy, b + 0.0 * a
    vn = np.sqrt(vx * vx + vy * vy + vz * vz)
    vx, vy, vz = vx / vn, vy / vn, vz / vn
    out = np.zeros((angles.size, n_b, n_a), dtype=np.float64)
    for rho, rad, x0, y0, z0 in balls:
        wx, wy, wz = x0 - sx, y0 - sy, z0 + 0.0 * sx          # centre - source
        along = wx * vx + wy * vy + wz * vz
        dist2 = wx * wx + wy * wy + wz * wz - along * along
        out += rho * 2.0 * np.sqrt(np.maximum(rad * rad - dist2, 0.0))
    return out


# The cone-beam workload `bench.py --extras` times and tests/test_extras_sizes_gpu.py checks against the oracle: on a
# config's x-y grid and angle count (angles over 2 pi), 97 detector rows of the config's n_det bins, 64 slices of
# isotropic voxels, source distance 2 N, three balls (a large central one, two small off-centre ones, one of them
# negative) sized relative to the half-width of the image.
FDK_BENCH_ROWS, FDK_BENCH_SLICES = 97, 64


def fdk_bench_geometry(cfg_id: int):
    """(angles[K] over 2 pi, sad, n_rows, n_z) of the bench's cone-beam problem on config ``cfg_id``'s grid."""
    cfg = CONFIGS[cfg_id]
    return uniform_angles(cfg.n_angles, 2.0 * math.pi), 2.0 * cfg.image_n, FDK_BENCH_ROWS, FDK_BENCH_SLICES


def fdk_bench_projections(cfg_id: int) -> np.ndarray:
    """fp64 projections [K][97][n_det] of the three-ball phantom for ``fdk_bench_geometry(cfg_id)`` (analytic)."""
    cfg = CONFIGS[cfg_id]
    ang, sad, n_rows, _ = fdk_bench_geometry(cfg_id)
    h = 0.5 * cfg.image_n
    balls = [(1.0, 0.6 * h, 0.0, 0.0, 0.0), (0.5, 0.15 * h, 0.4 * h, -0.3 * h, 10.0), (-0.3, 0.12 * h, -0.15 * h, 0.2 * h, -8.0)]
    return ball_cone_projections(balls, ang, sad, cfg.n_det, n_rows)
