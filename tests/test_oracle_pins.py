"""Pins P1-P12: the CPU oracle against what the mathematics fixes.

None of these compares the oracle with itself or with the CUDA path.  Each pin names the
part of oracle/fbp_oracle.c it fixes and the plausible mistake it would catch.  The paper
 prints no worked numeric example, so there is no paper-value fixture; the
expected values are closed forms, library routines and brute force written here.
"""
import math

import numpy as np
import pytest
import scipy.linalg
import scipy.special

from paper_2109_02174_b200 import inputs as I

PI = math.pi


# --------------------------------------------------------------------------------------
# P1  taps: closed forms (O1).  Catches: wrong constant, wrong sign, even/odd swapped.
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_det,expected", [(91, 1.1257e-3), (725, 1.3995e-4), (2897, 3.4987e-5)])
def test_p1_tap_sum_closed_form(oracle, n_det, expected):
    h = oracle.taps(n_det)
    assert h.shape == (2 * n_det - 1,)
    # sum_{odd m} 1/m^2 = pi^2/8  =>  sum_m h[m] = (2/pi^2) * sum_{odd m >= M} 1/m^2,
    # M = first odd integer > D-1; the tail is trigamma(M/2)/4 (Hurwitz zeta), from scipy.
    first_odd = n_det if n_det % 2 == 1 else n_det + 1
    tail = float(scipy.special.polygamma(1, first_odd / 2.0)) / 4.0
    assert math.fsum(h) == pytest.approx(2.0 / PI**2 * tail, rel=1e-10)
    assert math.fsum(h) == pytest.approx(expected, rel=2e-4)  # the value printed in SURVEY.md P1


def test_p1_tap_values_and_symmetry(oracle):
    d = 33
    h = oracle.taps(d)
    c = d - 1
    assert h[c] == 0.25
    assert h[c + 1] == pytest.approx(-1.0 / PI**2, rel=1e-15)
    assert h[c + 3] == pytest.approx(-1.0 / (9.0 * PI**2), rel=1e-15)
    assert h[c + 7] == pytest.approx(-1.0 / (49.0 * PI**2), rel=1e-15)
    assert np.all(h[c + 2::2] == 0.0) and np.all(h[c - 2::-2] == 0.0)
    assert np.array_equal(h, h[::-1])


def test_p1_taps_are_the_band_limited_ramp(oracle):
    """DTFT of the taps is |f| on |f| <= 1/2 (Kak & Slaney ch. 3): sum_m h[m] e^{-2 pi i f m} -> |f|."""
    d = 4097
    h = oracle.taps(d)
    m = np.arange(-(d - 1), d)
    for f in (0.0, 0.05, 0.125, 0.25, 0.4, 0.5):
        val = float(np.sum(h * np.cos(2 * PI * f * m)))
        assert val == pytest.approx(abs(f), abs=2e-4)


# --------------------------------------------------------------------------------------
# P2  filter == library convolution == Toeplitz product (O2: alignment "same", 1/d).
#     Catches: off-by-one alignment, reversed kernel (harmless: symmetric), d vs 1/d.
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_det,d", [(13, 1.0), (12, 0.5), (91, 2.0), (64, 1.0)])
def test_p2_filter_is_numpy_convolve_and_toeplitz(oracle, n_det, d):
    rng = np.random.default_rng(100 + n_det)
    p = rng.standard_normal((3, n_det))
    m = np.arange(-(n_det - 1), n_det)
    h = np.where(m == 0, 0.25, np.where(m % 2 != 0, -1.0 / (PI**2 * np.where(m == 0, 1, m).astype(float) ** 2), 0.0))
    q = oracle.filter_sinogram(p, det_spacing=d)
    ref_conv = np.stack([np.convolve(row, h)[n_det - 1:2 * n_det - 1] / d for row in p])
    col = h[n_det - 1:]  # h[0..D-1]; symmetric Toeplitz T[n][k] = h[n-k]
    ref_toep = (scipy.linalg.toeplitz(col) @ p.T).T / d
    scale = np.abs(ref_conv).max()
    assert np.abs(q - ref_conv).max() <= 1e-13 * scale
    assert np.abs(q - ref_toep).max() <= 1e-13 * scale


def test_p2_filter_rows_subset_matches_full(oracle):
    p = np.random.default_rng(7).standard_normal((11, 37))
    ids = [0, 5, 10, 3]
    assert np.array_equal(oracle.filter_rows(p, ids, 0.7), oracle.filter_sinogram(p, 0.7)[ids])


# --------------------------------------------------------------------------------------
# P3  ramp-filtered projection of a centred disk (continuous result rho/pi inside,
#     (rho/pi)(1 - |t|/sqrt(t^2-R^2)) outside).  Fixes tap normalisation and the 1/d scale
#     (G2, G3).  Catches: a sampled-|omega| filter (wrong DC), missing 1/d, 1/d^2.
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize(
    "n_det,d,radius,tol_in",
    [(725, 1.0, 100.0, 3e-3), (725, 1.0, 200.3, 5e-4), (1449, 0.5, 100.0, 2e-3), (363, 2.0, 100.0, 1e-2),
     (2897, 1.0, 800.0, 2e-4)],
)
def test_p3_disk_projection_filtered_is_rho_over_pi(oracle, n_det, d, radius, tol_in):
    rho = 1.7
    t = I.detector_coords(n_det, d)
    p = 2.0 * rho * np.sqrt(np.maximum(radius**2 - t**2, 0.0))
    q = oracle.filter_sinogram(p[None, :], det_spacing=d)[0]
    inside = np.abs(t) < 0.8 * radius
    assert np.abs(q[inside] / rho - 1.0 / PI).max() < tol_in
    centre = q[(n_det - 1) // 2] / rho
    assert centre == pytest.approx(1.0 / PI, abs=0.1 * tol_in)  # discretisation error ~ (d/R)^2
    outside = (np.abs(t) > 1.3 * radius) & (np.abs(t) < 1.7 * radius)
    if outside.any():
        expect = (1.0 / PI) * (1.0 - np.abs(t[outside]) / np.sqrt(t[outside] ** 2 - radius**2))
        assert np.abs(q[outside] / rho - expect).max() < 10 * tol_in


# --------------------------------------------------------------------------------------
# P4  impulse at the detector centre at every angle -> centre pixel = pi/(4d), any K.
#     Fixes the pi/K weight (G1) and the centre alignment (G6, G7).
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [1, 7, 90])
@pytest.mark.parametrize("d", [1.0, 0.5, 2.0])
def test_p4_impulse_centre_pixel(oracle, k, d):
    n, n_det = 9, 13
    p = np.zeros((k, n_det))
    p[:, (n_det - 1) // 2] = 1.0
    f = oracle.reconstruct(p, I.uniform_angles(k), n, det_spacing=d, pixel_size=d)
    assert f[n // 2, n // 2] == pytest.approx(PI / (4.0 * d), rel=1e-14)
    assert PI / 4.0 == pytest.approx(0.7853981633974483, rel=1e-16)


# --------------------------------------------------------------------------------------
# P5  partition of unity: Q == 1 -> every pixel that stays on the detector equals pi.
#     Fixes the interpolation weights (O3).  Catches (1-w)/w swapped with a wrong sum, a
#     dropped neighbour, a wrong zero-extension.
# --------------------------------------------------------------------------------------
def test_p5_partition_of_unity(oracle):
    n, k, n_det = 8, 5, 13
    ang = I.uniform_angles(k)
    f = oracle.backproject(np.ones((k, n_det)), ang, n)
    assert np.abs(f - PI).max() < 1e-14
    # detector too short: corner pixels leave it, interior ones do not
    f_short = oracle.backproject(np.ones((k, 7)), ang, n)
    assert f_short[4, 4] == pytest.approx(PI, rel=1e-14) and f_short[0, 0] < PI - 0.1
    assert oracle.backproject(np.ones((k, n_det)), ang, n, scaled=False)[3, 4] == pytest.approx(k, rel=1e-15)


# --------------------------------------------------------------------------------------
# P6  one angle: theta = 0 -> every image row is numpy.interp of Q along x; theta = pi/2
#     -> every column along y.  Fixes geometry and the axis convention (column <-> +x,
#     row <-> +y, G6).  Catches: transposed image, flipped detector, cos/sin swapped.
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,n_det,d,pix", [(8, 13, 1.0, 1.0), (9, 14, 1.0, 1.0), (16, 40, 0.5, 0.75)])
def test_p6_single_angle_is_numpy_interp(oracle, n, n_det, d, pix):
    q = np.random.default_rng(n * 100 + n_det).standard_normal((1, n_det))
    coord = (np.arange(n) - 0.5 * (n - 1)) * pix / d + 0.5 * (n_det - 1)
    expect = np.interp(coord, np.arange(n_det), q[0], left=0.0, right=0.0) * PI
    f0 = oracle.backproject(q, np.array([0.0]), n, det_spacing=d, pixel_size=pix)
    assert np.abs(f0 - expect[None, :]).max() < 1e-13       # varies along columns (x)
    f90 = oracle.backproject(q, np.array([PI / 2]), n, det_spacing=d, pixel_size=pix)
    assert np.abs(f90 - expect[:, None]).max() < 1e-12      # varies along rows (y), +y = +row
    if n % 2 == 0 and n_det % 2 == 1 and d == pix:
        j = (coord - 0.5).astype(int)
        assert np.abs(f0[0] - PI * 0.5 * (q[0][j] + q[0][j + 1])).max() < 1e-13


def test_p6_angle_pi_flips_detector(oracle):
    """Q_{theta+pi}(t) = Q_theta(-t): back-projecting a row at pi equals the reversed row at 0."""
    n, n_det = 10, 17
    q = np.random.default_rng(5).standard_normal((1, n_det))
    a = oracle.backproject(q, np.array([PI]), n)
    b = oracle.backproject(q[:, ::-1].copy(), np.array([0.0]), n)
    assert np.abs(a - b).max() < 1e-12


# --------------------------------------------------------------------------------------
# P7  brute force on 8x8: an explicit dense weight matrix built by an independent loop.
# --------------------------------------------------------------------------------------
def _dense_weights(n, k, n_det, angles, d, pix):
    w_mat = np.zeros((n * n, k * n_det))
    for r in range(n):
        for c in range(n):
            for i in range(k):
                x = (c - (n - 1) / 2) * pix
                y = (r - (n - 1) / 2) * pix
                u = (x * math.cos(angles[i]) + y * math.sin(angles[i])) / d + (n_det - 1) / 2
                j = math.floor(u)
                frac = u - j
                if 0 <= j < n_det:
                    w_mat[r * n + c, i * n_det + j] += 1.0 - frac
                if 0 <= j + 1 < n_det:
                    w_mat[r * n + c, i * n_det + j + 1] += frac
    return w_mat


@pytest.mark.parametrize("n_det,d,pix", [(13, 1.0, 1.0), (9, 1.0, 1.0), (13, 0.8, 1.1)])
def test_p7_brute_force_8x8(oracle, n_det, d, pix):
    n, k = 8, 5
    ang = np.array([0.1, 0.9, 1.7, 2.2, 3.0])  # non-uniform on purpose
    q = np.random.default_rng(77).standard_normal((k, n_det))
    w_mat = _dense_weights(n, k, n_det, ang, d, pix)
    f = oracle.backproject(q, ang, n, det_spacing=d, pixel_size=pix, scaled=False)
    assert np.abs(f.ravel() - w_mat @ q.ravel()).max() < 1e-14
    fs = oracle.backproject(q, ang, n, det_spacing=d, pixel_size=pix, scaled=True)
    assert np.abs(fs.ravel() - (PI / k) * (w_mat @ q.ravel())).max() < 1e-14
    # the scatter projector is the transpose of the same matrix
    x = np.random.default_rng(78).standard_normal((n, n))
    rx = oracle.forward_scatter(x, ang, n_det, det_spacing=d, pixel_size=pix)
    assert np.abs(rx.ravel() - w_mat.T @ x.ravel()).max() < 1e-14
    if n_det == 13 and d == pix:
        assert np.allclose(w_mat.sum(axis=1), k, atol=1e-13)  # rows sum to K (P5)


# --------------------------------------------------------------------------------------
# P8  adjoint identity <R x, y> = <x, B y> with R the independent scatter code (O4).
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,k,n_det", [(8, 5, 13), (64, 90, 91), (33, 17, 40)])
def test_p8_adjoint_identity(oracle, n, k, n_det):
    rng = np.random.default_rng(n + k)
    ang = I.uniform_angles(k)
    x = rng.standard_normal((n, n))
    y = rng.standard_normal((k, n_det))
    lhs = float(np.vdot(oracle.forward_scatter(x, ang, n_det), y))
    rhs = float(np.vdot(x, oracle.backproject(y, ang, n, scaled=False)))
    assert abs(lhs - rhs) <= 1e-10 * max(abs(lhs), abs(rhs))
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(x) * np.linalg.norm(y) * math.sqrt(k)


# --------------------------------------------------------------------------------------
# P9  linearity of both steps.
# --------------------------------------------------------------------------------------
def test_p9_linearity(oracle):
    rng = np.random.default_rng(9)
    k, n_det, n = 12, 45, 31
    a, b = rng.standard_normal((2, k, n_det))
    al, be = 0.37, -2.5
    ang = I.uniform_angles(k)
    qa, qb, qab = (oracle.filter_sinogram(v, 1.3) for v in (a, b, al * a + be * b))
    assert np.abs(qab - (al * qa + be * qb)).max() <= 1e-13 * np.abs(qab).max()
    fa, fb, fab = (oracle.backproject(v, ang, n) for v in (a, b, al * a + be * b))
    assert np.abs(fab - (al * fa + be * fb)).max() <= 1e-13 * np.abs(fab).max()


# --------------------------------------------------------------------------------------
# P10  uniform disk, whole chain including every scale factor.
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,k,n_det,bound_half,bound_08",
                         [(64, 90, 91, 1e-2, 2.5e-2), (256, 180, 363, 2e-3, 4e-3), (512, 360, 725, 1e-3, 1.5e-3)])
def test_p10_uniform_disk_reconstruction(oracle, n, k, n_det, bound_half, bound_08):
    ang = I.uniform_angles(k)
    radius = 0.5 * (n / 2)
    sino = I.ellipse_sinogram(I.disk(0.5), ang, n_det, 1.0, n / 2)
    f = oracle.reconstruct(sino, ang, n)
    ax = np.arange(n) - 0.5 * (n - 1)
    rr = np.hypot(ax[None, :], ax[:, None])
    assert np.abs(f[rr < 0.5 * radius] - 1.0).max() < bound_half
    assert np.abs(f[rr < 0.8 * radius] - 1.0).max() < bound_08
    assert abs(f[rr < 0.5 * radius].mean() - 1.0) < 0.5 * bound_half
    assert np.abs(f[rr > 1.3 * radius]).mean() < 0.02  # outside the disk: ~0


# --------------------------------------------------------------------------------------
# P11  analytic ellipse sinograms: region interiors recover the true density.
#      HEAD10 is not symmetric, so a flipped axis or a wrong rotation sign fails here.
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n,k", [("head10", 256, 180), ("rand3", 256, 360)])
def test_p11_ellipse_phantom_regions(oracle, name, n, k):
    ell = I.HEAD10 if name == "head10" else I.random_ellipses(3)
    n_det = I.default_n_det(n)
    ang = I.uniform_angles(k)
    f = oracle.reconstruct(I.ellipse_sinogram(ell, ang, n_det, 1.0, n / 2), ang, n)
    truth = I.rasterise(ell, n)
    label, interior = I.region_masks(ell, n, margin_px=3.0)
    dr = truth.max() - truth.min()
    checked = 0
    for lab in np.unique(label[interior]):
        sel = interior & (label == lab)
        if sel.sum() < 30:
            continue
        assert np.ptp(truth[sel]) == 0.0
        assert abs(f[sel].mean() - truth[sel][0]) < 0.01 * dr, (lab, f[sel].mean(), truth[sel][0])
        checked += 1
    assert checked >= 5


def test_p11_off_centre_disk_lands_where_the_generator_put_it(oracle):
    """Orientation / sign pin: a small disk at (x0, y0) = (+0.5, +0.25) must be reconstructed
    at column c_N + x0*N/2 and row c_N + y0*N/2 (column <-> +x, row <-> +y).  A transposed
    image, a flipped detector or a wrong sign of sin(theta) moves it to another quadrant."""
    n, k = 128, 120
    n_det = I.default_n_det(n)
    ang = I.uniform_angles(k)
    ell = np.array([(1.0, 0.08, 0.08, 0.5, 0.25, 0.0)])
    f = oracle.reconstruct(I.ellipse_sinogram(ell, ang, n_det, 1.0, n / 2), ang, n)
    ax = np.arange(n) - 0.5 * (n - 1)
    blob = np.where(f > 0.5, f, 0.0)
    col = float((blob * ax[None, :]).sum() / blob.sum())
    row = float((blob * ax[:, None]).sum() / blob.sum())
    assert col == pytest.approx(0.5 * n / 2, abs=0.05)
    assert row == pytest.approx(0.25 * n / 2, abs=0.05)
    assert blob.sum() == pytest.approx(PI * (0.08 * n / 2) ** 2, rel=0.10)  # ~ area * density (edge pixels thresholded away)


# --------------------------------------------------------------------------------------
# P12  symmetries.
# --------------------------------------------------------------------------------------
def test_p12_symmetries(oracle):
    n, k, n_det = 32, 16, 47
    row = np.random.default_rng(12).standard_normal(n_det)
    row = row + row[::-1]                       # even in t
    q = np.tile(row, (k, 1))                    # identical at all angles
    f = oracle.backproject(q, I.uniform_angles(k), n)
    assert np.abs(f - f[::-1, ::-1]).max() < 1e-13        # (x,y) -> (-x,-y)
    assert np.abs(f - np.rot90(f)).max() < 1e-13          # K even: 90 degree rotation
    # 2 pi worth of angles with Q_{theta+pi}(t) = Q_theta(-t) doubles the [0,pi) sum
    k2 = 10
    qa = np.random.default_rng(13).standard_normal((k2, n_det))
    ang_pi = I.uniform_angles(k2)
    full = np.concatenate([qa, qa[:, ::-1]])
    ang_2pi = np.concatenate([ang_pi, ang_pi + PI])
    fa = oracle.backproject(qa, ang_pi, n, scaled=False)
    fb = oracle.backproject(full, ang_2pi, n, scaled=False)
    assert np.abs(fb - 2 * fa).max() < 1e-12


def test_batch_slices_are_independent(oracle):
    rng = np.random.default_rng(21)
    p = rng.standard_normal((3, 6, 19))
    ang = I.uniform_angles(6)
    f = oracle.reconstruct(p, ang, 11)
    for s in range(3):
        assert np.array_equal(f[s], oracle.reconstruct(p[s], ang, 11))
    assert np.array_equal(oracle.reconstruct(p, ang, 11, threads=1), f)  # threads do not change bits
    pix = oracle.backproject_pixels(oracle.filter_sinogram(p[1]), ang, 11, [0, 10, 4], [3, 10, 4])
    assert np.array_equal(pix, f[1][[0, 10, 4], [3, 10, 4]])
