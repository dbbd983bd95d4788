"""GPU parity for cone-beam FDK (fbp_fdk_reconstruct) against
oracle/fbp_oracle_fdk.c on the same seeded inputs.  Tolerances as for the 2-D images (BASELINE.json):
fp64 1e-12 of max|f|; fp32 max-abs <= 1e-4 DR and RMSE <= 1e-5 DR, DR over the whole volume."""
import math

import numpy as np
import pytest

from paper_2109_02174_b200 import inputs as I

pytestmark = pytest.mark.gpu


def _npdt(dt):
    return np.float32 if dt == "f32" else np.float64


def _dev(a, dt):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=_npdt(dt))).cuda()


def _check(gpu, ref, dt, what):
    err = np.abs(np.asarray(gpu, dtype=np.float64) - ref)
    if dt == "f64":
        assert err.max() / np.abs(ref).max() <= 1e-12, (what, err.max() / np.abs(ref).max())
    else:
        dr = ref.max() - ref.min()
        if dr == 0.0:                      # a one-voxel volume: fall back to its magnitude
            dr = max(float(np.abs(ref).max()), 1e-30)
        assert err.max() / dr <= 1e-4 and math.sqrt(float(np.mean(err * err))) / dr <= 1e-5, (what, err.max() / dr)


CASES = [  # (N, K, n_a, n_b, n_z, d_a, d_b, pix, vz, sad, angle kind)
    (24, 36, 61, 17, 11, 1.0, 1.0, 1.0, 1.0, 60.0, "uniform"),       # n_z not a multiple of the z register tile
    (33, 25, 80, 9, 8, 0.5, 0.75, 0.5, 0.6, 40.0, "random"),          # N odd, n_a even, unequal spacings, any angles
    (16, 12, 20, 5, 19, 1.0, 2.0, 1.0, 1.0, 14.0, "uniform"),         # detector too small: rays miss it on both axes
    (1, 3, 2, 1, 1, 1.0, 1.0, 1.0, 1.0, 5.0, "uniform"),
]


@pytest.mark.parametrize("kind", [pytest.param(2, id="fft"), pytest.param(1, id="direct")])
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("case", CASES)
def test_fdk_matches_oracle_on_random_projections(fbp, oracle, case, dt, kind):
    import torch
    n, k, n_a, n_b, n_z, d_a, d_b, pix, vz, sad, akind = case
    rng = np.random.default_rng(100 + n + k)
    ang = I.uniform_angles(k, 2 * math.pi) if akind == "uniform" else np.sort(rng.uniform(-1.0, 7.0, k))
    proj = rng.normal(size=(k, n_b, n_a)).astype(_npdt(dt))
    ref = oracle.fdk_reconstruct(proj.astype(np.float64), ang, sad, n, n_z, d_a, d_b, pix, vz)
    with fbp.Plan(list(ang), n_a, n, det_spacing=d_a, pixel_size=pix, dtype=dt, options={"filter_kind": kind}) as plan:
        got = plan.fdk_reconstruct(_dev(proj, dt), sad, n_z, row_spacing=d_b, voxel_z=vz)
        again = plan.fdk_reconstruct(_dev(proj, dt), sad, n_z, row_spacing=d_b, voxel_z=vz)
        assert torch.equal(got, again)                                  # bit-identical repeats
    _check(got.cpu().numpy(), ref, dt, case)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_fdk_ball_phantom_128(fbp, oracle, dt):
    """128^3-class problem from analytic cone-beam data of three balls: parity with the oracle on the whole volume,
    and the physics: the mid-plane section of the central ball comes back with its density."""
    n, k, n_a, n_b, n_z, sad = 128, 180, 255, 97, 48, 300.0
    ang = I.uniform_angles(k, 2 * math.pi)
    balls = [(1.0, 30.0, 0.0, 0.0, 0.0), (0.5, 10.0, 25.0, -20.0, 8.0), (-0.3, 8.0, -10.0, 12.0, -5.0)]
    proj = I.ball_cone_projections(balls, ang, sad, n_a, n_b).astype(_npdt(dt))
    ref = oracle.fdk_reconstruct(proj.astype(np.float64), ang, sad, n, n_z)
    with fbp.Plan(list(ang), n_a, n, dtype=dt) as plan:
        got = plan.fdk_reconstruct(_dev(proj, dt), sad, n_z).cpu().numpy()
    _check(got, ref, dt, "balls")
    mid = 0.5 * (got[23] + got[24]).astype(np.float64)                      # z = -0.5 and +0.5
    c = (n - 1) / 2
    yy, xx = np.mgrid[0:n, 0:n]
    core = np.hypot(xx - c - 5, yy - c - 15) < 5                            # inside the big ball, away from the small ones
    assert abs(mid[core].mean() - 1.0) < 2e-2


def test_fdk_window_and_errors(fbp, oracle):
    import torch
    n, k, n_a, n_b, n_z, sad = 20, 16, 41, 7, 5, 50.0
    ang = I.uniform_angles(k, 2 * math.pi)
    proj = np.random.default_rng(4).normal(size=(k, n_b, n_a))
    w = oracle.fdk_weight(proj, 1.0, 1.0, sad)
    q = oracle.filter_sinogram_window(w.reshape(k * n_b, n_a), "hann").reshape(k, n_b, n_a)
    ref = oracle.fdk_backproject(q, ang, sad, n, n_z)
    with fbp.Plan(list(ang), n_a, n, dtype="f64") as plan:
        plan.set_window("hann")
        got = plan.fdk_reconstruct(_dev(proj, "f64"), sad, n_z)
        _check(got.cpu().numpy(), ref, "f64", "hann")
        vol = torch.full((n_z, n, n), 7.0, dtype=torch.float64, device="cuda")
        d_proj = _dev(proj, "f64")
        for args in ((0, vol, n_b, 1.0, sad, n_z, 1.0), (d_proj, 0, n_b, 1.0, sad, n_z, 1.0), (d_proj, vol, 0, 1.0, sad, n_z, 1.0),
                     (d_proj, vol, n_b, 0.0, sad, n_z, 1.0), (d_proj, vol, n_b, 1.0, 10.0, n_z, 1.0),      # sad inside the image
                     (d_proj, vol, n_b, 1.0, float("nan"), n_z, 1.0), (d_proj, vol, n_b, 1.0, sad, 0, 1.0),
                     (d_proj, vol, n_b, 1.0, sad, n_z, -1.0)):
            with pytest.raises(fbp.FbpError) as ei:
                fbp.fbp_fdk_reconstruct(plan.handle, *args)
            assert ei.value.status == fbp.FBP_EINVAL
        torch.cuda.synchronize()
        assert bool((vol == 7.0).all())


@pytest.mark.parametrize("pixel_size", [0.5, 0.0])
def test_fdk_default_voxel_height_is_the_pixel_size(fbp, oracle, pixel_size):
    """voxel_z left out means isotropic voxels on both sides: the plan's pixel size (pixel_size <= 0: the detector
    spacing, as fbp_create resolves it), whatever the detector's row spacing is."""
    n, k, n_a, n_b, n_z, d_a, d_b, sad = 20, 18, 47, 9, 7, 0.75, 1.5, 40.0
    ang = I.uniform_angles(k, 2 * math.pi)
    proj = np.random.default_rng(9).normal(size=(k, n_b, n_a))
    pix = pixel_size if pixel_size > 0 else d_a
    ref = oracle.fdk_reconstruct(proj, ang, sad, n, n_z, d_a, d_b, pix)                 # oracle default: voxel_z = pix
    with fbp.Plan(list(ang), n_a, n, det_spacing=d_a, pixel_size=pixel_size, dtype="f64") as plan:
        assert plan.pixel_size == pix
        got = plan.fdk_reconstruct(_dev(proj, "f64"), sad, n_z, row_spacing=d_b)
    _check(got.cpu().numpy(), ref, "f64", "default voxel_z")
    other = oracle.fdk_reconstruct(proj, ang, sad, n, n_z, d_a, d_b, pix, d_b)          # the old default would give this volume
    assert np.abs(other - ref).max() > 1e-3 * np.abs(ref).max()
