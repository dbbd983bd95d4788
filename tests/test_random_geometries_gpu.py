"""Randomised geometries (fixed seeds): fbp_reconstruct, fbp_project and fbp_fdk_reconstruct against the oracle on a few
hundred small problems whose sizes, spacings, angle sets and dtypes are drawn at random -- odd and even N and D, K = 1,
detectors far too short or too long, pixel_size != det_spacing either way, angles over [0, pi), [0, 2 pi), arbitrary
sorted reals and exact multiples of pi/2, batches 1..3.  They walk through the corners a hand-written case list misses:
chunks of the fp64 back-projector that can and cannot be walked in one launch, staged projector windows clamped at
either end of the padded line, partially live bin blocks, cone-beam samples clamped on both detector axes.
Tolerances are BASELINE.json's; a result whose largest value is itself at rounding level (a detector that the image
only grazes) is compared absolutely instead."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _ok(got, ref, dt):
    err = float(np.abs(got - ref).max())
    mx = float(np.abs(ref).max())
    if mx < 1e-9:                                   # nothing but rounding reaches the output: absolute comparison
        return err <= 1e-12, err
    if dt == "f64":
        return err <= 1e-12 * mx, err / mx
    dr = float(ref.max() - ref.min()) or mx
    return err <= 1e-4 * dr and math.sqrt(float(np.mean((got - ref) ** 2))) <= 1e-5 * dr, err / dr


@pytest.mark.parametrize("seed", [11, 12])
def test_random_2d_geometries(fbp, oracle, seed):
    import torch
    rng = np.random.default_rng(seed)
    for case in range(120):
        n, k, dd = int(rng.integers(1, 140)), int(rng.integers(1, 70)), int(rng.integers(2, 260))
        d = float(rng.choice([1.0, 0.5, 2.0, 0.8, 1.37]))
        pix = float(rng.choice([1.0, 0.5, 2.0, 1.0, 1.21]))
        kind = int(rng.integers(0, 4))
        if kind == 0:
            ang = np.pi * np.arange(k) / k
        elif kind == 1:
            ang = 2 * np.pi * np.arange(k) / k
        elif kind == 2:
            ang = np.sort(rng.uniform(-4.0, 8.0, k))
        else:
            ang = np.arange(k) * (np.pi / 2)
        b = int(rng.integers(1, 4))
        dt = "f64" if rng.random() < 0.6 else "f32"
        npdt = np.float64 if dt == "f64" else np.float32
        sino = rng.standard_normal((b, k, dd)).astype(npdt)
        img = rng.standard_normal((b, n, n)).astype(npdt)
        try:
            plan = fbp.Plan(list(ang), dd, n, det_spacing=d, pixel_size=pix, dtype=dt, max_batch=b)
        except fbp.FbpError as e:
            assert e.status == fbp.FBP_EUNSUPPORTED, (case, e)      # a tile's staged segment would not fit shared memory
            continue
        with plan:
            rec = plan.reconstruct(torch.from_numpy(sino).cuda()).cpu().numpy().astype(np.float64)
            prj = plan.project(torch.from_numpy(img).cuda()).cpu().numpy().astype(np.float64)
        what = dict(case=case, n=n, k=k, dd=dd, d=d, pix=pix, kind=kind, b=b, dt=dt)
        for s in range(b):
            ok, e = _ok(rec[s], oracle.reconstruct(sino[s].astype(np.float64), ang, n, d, pix), dt)
            assert ok, ("reconstruct", what, s, e)
            ok, e = _ok(prj[s], oracle.forward_scatter(img[s].astype(np.float64), ang, dd, d, pix), dt)
            assert ok, ("project", what, s, e)


def test_random_cone_beam_geometries(fbp, oracle):
    import torch
    rng = np.random.default_rng(21)
    for case in range(100):
        n, k = int(rng.integers(1, 40)), int(rng.integers(1, 30))
        n_a, n_b, n_z = int(rng.integers(2, 90)), int(rng.integers(1, 24)), int(rng.integers(1, 24))
        d_a, d_b = float(rng.choice([1.0, 0.5, 2.0, 0.7])), float(rng.choice([1.0, 0.5, 2.0, 1.3]))
        pix, vz = float(rng.choice([1.0, 0.5, 1.7])), float(rng.choice([1.0, 0.4, 2.5]))
        sad = float(0.5 * (n - 1) * math.sqrt(2.0) * pix * rng.uniform(1.05, 6.0) + 0.1)
        ang = 2 * np.pi * np.arange(k) / k if rng.random() < 0.5 else np.sort(rng.uniform(-1.0, 7.0, k))
        dt = "f64" if rng.random() < 0.6 else "f32"
        npdt = np.float64 if dt == "f64" else np.float32
        proj = rng.standard_normal((k, n_b, n_a)).astype(npdt)
        ref = oracle.fdk_reconstruct(proj.astype(np.float64), ang, sad, n, n_z, d_a, d_b, pix, vz)
        with fbp.Plan(list(ang), n_a, n, det_spacing=d_a, pixel_size=pix, dtype=dt) as plan:
            got = plan.fdk_reconstruct(torch.from_numpy(proj).cuda(), sad, n_z, row_spacing=d_b, voxel_z=vz)
        got = got.cpu().numpy().astype(np.float64)
        err, mx = float(np.abs(got - ref).max()), float(np.abs(ref).max())
        # a volume that only the fringe of a one-row detector reaches is a difference of nearly equal numbers: compare
        # with the size of the data (1) instead of the size of the result
        ok = err <= 1e-12 * max(mx, 1e-3) if dt == "f64" else _ok(got, ref, dt)[0]
        assert ok, (dict(case=case, n=n, k=k, n_a=n_a, n_b=n_b, n_z=n_z, d_a=d_a, d_b=d_b, pix=pix, vz=vz, sad=sad, dt=dt), err, mx)
