"""Pins for oracle/fbp_oracle_fdk.c (cone-beam FDK, the paper's announced continuation).
None compares the oracle with itself or with the CUDA path: the parallel limit reduces FDK to the 2-D oracle
(itself pinned by P1-P12), the ball tests use analytic cone-beam line integrals, the matrix test an independent loop."""
import math

import numpy as np
import pytest

from paper_2109_02174_b200 import inputs as I

PI = math.pi


def test_c3_preweight_closed_form(oracle):
    n_a, n_b, sad = 9, 5, 4.0
    p = np.ones((2, n_b, n_a))
    w = oracle.fdk_weight(p, 1.0, 2.0, sad)
    assert w[0, 2, 4] == pytest.approx(1.0, rel=1e-15)                       # a = b = 0
    assert w[1, 2, 8] == pytest.approx(1.0 / math.sqrt(2.0), rel=1e-15)      # a = 4 = sad, b = 0
    assert w[0, 4, 4] == pytest.approx(1.0 / math.sqrt(2.0), rel=1e-15)      # b = 2 * 2 = sad, a = 0
    assert w[0, 0, 0] == pytest.approx(sad / math.sqrt(sad**2 + 16.0 + 16.0), rel=1e-15)
    assert np.array_equal(w[0], w[1])


def test_parallel_limit_is_the_2d_oracle_row_by_row(oracle):
    """sad -> infinity: a' -> t, b' -> z, weight -> 1, so every detector row is an independent 2-D problem with the K
    angles spread over 2 pi and the pi/K weight of the 2-D method.  Pins t = x cos + y sin (same sign and axes as
    PAPER.md:55), the column interpolation, the angular weight and the row <-> z association."""
    n, k, n_a, n_b = 12, 10, 19, 4
    ang = I.uniform_angles(k, 2 * PI)
    q = np.random.default_rng(5).normal(size=(k, n_b, n_a))
    f = oracle.fdk_backproject(q, ang, 1e10, n, n_b, d_a=1.0, d_b=0.7, pixel_size=1.0, voxel_z=0.7)
    for i in range(n_b):
        want = oracle.backproject(q[:, i, :], ang, n)
        assert np.allclose(f[i], want, rtol=1e-7, atol=1e-8), i
    # twice as many slices on half the spacing: the new in-between slices are the mean of their two neighbours' rows
    f2 = oracle.fdk_backproject(q, ang, 1e10, n, 2 * n_b - 1, d_a=1.0, d_b=0.7, pixel_size=1.0, voxel_z=0.35)
    assert np.allclose(f2[::2], f, rtol=1e-7, atol=1e-8)
    assert np.allclose(f2[1::2], 0.5 * (f[:-1] + f[1:]), rtol=1e-7, atol=1e-8)
    # other spacings: d_a != pixel
    f3 = oracle.fdk_backproject(q, ang, 1e10, n, n_b, d_a=0.5, d_b=1.0, pixel_size=0.25, voxel_z=1.0)
    for i in range(n_b):
        assert np.allclose(f3[i], oracle.backproject(q[:, i, :], ang, n, 0.5, 0.25), rtol=1e-7, atol=1e-8)


@pytest.mark.parametrize("centre", [(0.0, 0.0, 0.0), (14.0, -9.0, 0.0), (-8.0, 15.0, 0.0)])
def test_midplane_ball_from_analytic_cone_data(oracle, centre):
    """Fan-beam FBP is exact in the mid-plane up to discretisation: a ball of density 1 must come back as 1 in the
    interior of its mid-plane section, where the generator put it.  sad = 2.2 N/2 makes the magnification vary by
    +-27 % across the field, so (sad/U) instead of (sad/U)^2, a flipped sign of s, or a missing pre-weight show as
    several per cent (tried: each fails this test)."""
    n, k, n_z = 64, 240, 3
    sad, rad = 70.0, 9.0
    n_a, n_b = 161, 9
    ang = I.uniform_angles(k, 2 * PI)
    proj = I.ball_cone_projections([(1.0, rad, *centre)], ang, sad, n_a, n_b)
    f = oracle.fdk_reconstruct(proj, ang, sad, n, n_z)
    c = (n - 1) / 2
    yy, xx = np.mgrid[0:n, 0:n]
    r = np.hypot(xx - c - centre[0], yy - c - centre[1])
    # "outside": away from the ball but inside 0.8 N/2 of the axis (nearer the source orbit, where U is small and the
    # weight (sad/U)^2 reaches 6, angular sampling streaks of a few per cent are the method's, not an error)
    inside, outside = r < 0.6 * rad, (r > rad + 4) & (np.hypot(xx - c, yy - c) < 0.8 * n / 2)
    assert abs(f[1][inside].mean() - 1.0) < 6e-3
    assert np.abs(f[1][inside] - 1.0).max() < 2.5e-2
    assert np.abs(f[1][outside]).max() < 6e-2                    # streaks off the ball's edge (240 views, point-sampled data)
    # a ball centred on the mid-plane is symmetric in z
    assert np.allclose(f[0], f[2], rtol=1e-12, atol=1e-13)


def test_ball_above_the_midplane_small_cone_angle(oracle):
    """Off the mid-plane FDK is approximate; at a cone angle of ~3 degrees a ball centred at z0 still comes back with
    its density at its centre (2 %), in the slice where the generator put it (row <-> z, sign of z)."""
    n, k, n_z = 32, 120, 9
    sad, rad, z0 = 400.0, 6.0, 3.0
    ang = I.uniform_angles(k, 2 * PI)
    proj = I.ball_cone_projections([(1.0, rad, 0.0, 0.0, z0)], ang, sad, 61, 33)
    f = oracle.fdk_reconstruct(proj, ang, sad, n, n_z)          # z_k = k - 4
    c = (n - 1) / 2
    centre_val = f[7][15:17, 15:17].mean()                      # z = +3
    assert abs(centre_val - 1.0) < 2e-2
    assert abs(f[1][15:17, 15:17].mean()) < 0.2                 # z = -3: |z - z0| = 6 = rad, the ball's pole
    assert f[7].sum() > 5 * abs(f[1].sum())


def test_dense_matrix_brute_force(oracle):
    """B q = W q with W (n_z N^2 x K n_b n_a) built by an independent loop from C5's formulas."""
    n, n_z, k, n_a, n_b = 4, 3, 5, 9, 5
    sad, d_a, d_b, pix, vz = 11.0, 0.8, 1.1, 1.0, 0.9
    ang = np.sort(np.random.default_rng(2).uniform(0, 2 * PI, k))
    q = np.random.default_rng(3).normal(size=(k, n_b, n_a))
    w_mat = np.zeros((n_z * n * n, k * n_b * n_a))
    for kz in range(n_z):
        for r in range(n):
            for c in range(n):
                x, y, z = (c - (n - 1) / 2) * pix, (r - (n - 1) / 2) * pix, (kz - (n_z - 1) / 2) * vz
                for m in range(k):
                    t = x * math.cos(ang[m]) + y * math.sin(ang[m])
                    s = -x * math.sin(ang[m]) + y * math.cos(ang[m])
                    mag = sad / (sad + s)
                    ua, ub = mag * t / d_a + (n_a - 1) / 2, mag * z / d_b + (n_b - 1) / 2
                    ja, ib = math.floor(ua), math.floor(ub)
                    for di, wi in ((0, 1 - (ub - ib)), (1, ub - ib)):
                        for dj, wj in ((0, 1 - (ua - ja)), (1, ua - ja)):
                            if 0 <= ib + di < n_b and 0 <= ja + dj < n_a:
                                w_mat[(kz * n + r) * n + c, (m * n_b + ib + di) * n_a + ja + dj] += mag * mag * wi * wj * PI / k
    want = (w_mat @ q.ravel()).reshape(n_z, n, n)
    got = oracle.fdk_backproject(q, ang, sad, n, n_z, d_a, d_b, pix, vz)
    assert np.allclose(got, want, rtol=1e-13, atol=1e-14)


def test_linearity_and_threads(oracle):
    n, k = 10, 7
    ang = I.uniform_angles(k, 2 * PI)
    rng = np.random.default_rng(9)
    pa, pb = rng.normal(size=(k, 5, 17)), rng.normal(size=(k, 5, 17))
    fa = oracle.fdk_reconstruct(pa, ang, 30.0, n, 4)
    fb = oracle.fdk_reconstruct(pb, ang, 30.0, n, 4)
    fab = oracle.fdk_reconstruct(2.0 * pa - 0.5 * pb, ang, 30.0, n, 4)
    assert np.allclose(fab, 2.0 * fa - 0.5 * fb, rtol=1e-12, atol=1e-13)
    assert np.array_equal(oracle.fdk_reconstruct(pa, ang, 30.0, n, 4, threads=1), fa)
