"""Parity at exactly the problem sizes `bench.py --extras` reports numbers for (a number on a configuration no test
compares with the oracle is a claim, not a measurement):

  fbp_project           config 5 (2048^2, 1800 x 2897), 1 slice, and config 4 (512^2, 720 x 725), 8 slices
  fbp_fdk_reconstruct   64 x 512^2 voxels from 360 projections of 97 x 725 (config 3's grid), whole volume
  fbp_metrics           a 64 x 512^2 pair (the config-4 output stack)
  fbp_interpolate_stack 64 -> 256 slices of 512^2

each in the launch configuration the library chooses for that size (no options), on seeded inputs
(paper_2109_02174_b200/inputs.py; the cone-beam data are the very arrays bench.py times).  PAPER.md:228-235 (FDK),
PAPER.md:85-97 (eq. 3-4), PAPER.md:19 (stack interpolation); SURVEY.md 8(f).  Tolerances as everywhere else:
fp64 1e-12 of max|ref|; fp32 max-abs <= 1e-4 DR and RMSE <= 1e-5 DR."""
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
        assert err.max() / dr <= 1e-4 and math.sqrt(float(np.mean(err * err))) / dr <= 1e-5, (what, err.max() / dr)


def _phantom_stack(cfg_id, b, seed):
    """b seeded images of the config's size: a rasterised ellipse phantom plus 2 % noise (so no pixel is exactly 0),
    rounded to fp32 so that the fp32 and the fp64 plan see the same values."""
    n = I.CONFIGS[cfg_id].image_n
    rng = np.random.default_rng(seed)
    out = np.stack([I.rasterise(I.random_ellipses(seed + s), n) for s in range(b)])
    return (out + 0.02 * rng.standard_normal(out.shape)).astype(np.float32)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_project_config5_sampled_angles(fbp, oracle, dt):
    cfg = I.CONFIGS[5]
    ang = I.config_angles(5)
    img = _phantom_stack(5, 1, 50)
    sel = np.arange(7, cfg.n_angles, 100)                                  # 18 of the 1800 angles, every bin of each
    want = oracle.forward_scatter(img[0].astype(np.float64), ang[sel], cfg.n_det)
    with fbp.Plan(list(ang), cfg.n_det, cfg.image_n, dtype=dt) as plan:
        got = plan.project(_dev(img, dt))[0][sel].cpu().numpy()
    _check(got, want, dt, "project cfg5")


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_project_config4_eight_slices_sampled_angles(fbp, oracle, dt):
    cfg = I.CONFIGS[4]
    ang = I.config_angles(4)
    img = _phantom_stack(4, 8, 40)
    sel = np.arange(3, cfg.n_angles, 60)                                   # 12 of the 720 angles, in all 8 slices
    want = np.stack([oracle.forward_scatter(img[s].astype(np.float64), ang[sel], cfg.n_det) for s in range(8)])
    with fbp.Plan(list(ang), cfg.n_det, cfg.image_n, dtype=dt, max_batch=cfg.batch) as plan:
        got = plan.project(_dev(img, dt))[:, sel].cpu().numpy()
    for s in range(8):
        _check(got[s], want[s], dt, "project cfg4 slice %d" % s)


@pytest.fixture(scope="module")
def fdk_bench_case(oracle):
    """The bench's cone-beam problem on config 3's grid and its oracle volume (all 64 x 512^2 voxels; about six
    billion voxel-angle updates: tens of seconds on the host cores, computed once for both dtypes)."""
    ang, sad, n_rows, n_z = I.fdk_bench_geometry(3)
    proj = I.fdk_bench_projections(3).astype(np.float32)                   # fp32-representable: both plans read the same values
    ref = oracle.fdk_reconstruct(proj.astype(np.float64), ang, sad, I.CONFIGS[3].image_n, n_z)
    return ang, sad, n_rows, n_z, proj, ref


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_fdk_at_the_bench_size_whole_volume(fbp, fdk_bench_case, dt):
    import torch
    ang, sad, n_rows, n_z, proj, ref = fdk_bench_case
    cfg = I.CONFIGS[3]
    assert proj.shape == (cfg.n_angles, n_rows, cfg.n_det) and ref.shape == (n_z, cfg.image_n, cfg.image_n)
    with fbp.Plan(list(ang), cfg.n_det, cfg.image_n, dtype=dt) as plan:
        d_proj = _dev(proj, dt)
        got = plan.fdk_reconstruct(d_proj, sad, n_z)
        again = plan.fdk_reconstruct(d_proj, sad, n_z)
        assert torch.equal(got, again)
    got = got.cpu().numpy()
    _check(got, ref, dt, "FDK 64 x 512^2")
    mid = 0.5 * (got[31] + got[32]).astype(np.float64)                    # z = -0.5 and +0.5: the central ball's density
    c = (cfg.image_n - 1) / 2
    yy, xx = np.mgrid[0:cfg.image_n, 0:cfg.image_n]
    core = np.hypot(xx - c + 60, yy - c + 60) < 20                        # inside the big ball, clear of the small ones
    assert abs(mid[core].mean() - 1.0) < 2e-2


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_metrics_on_a_config4_sized_stack(fbp, oracle, dt):
    cfg = I.CONFIGS[4]
    rng = np.random.default_rng(44)
    x = rng.uniform(-0.2, 1.1, (cfg.batch, cfg.image_n, cfg.image_n)).astype(_npdt(dt))
    y = (x + rng.normal(0, 0.01, x.shape)).astype(_npdt(dt))
    with fbp.Plan(list(I.uniform_angles(4)), 8, 4, dtype=dt) as plan:
        got = plan.metrics(_dev(x, dt), _dev(y, dt), 1.0)
    want = oracle.metrics(x.astype(np.float64), y.astype(np.float64), 1.0)
    for k, v in want.items():
        assert got[k] == pytest.approx(v, rel=1e-11, abs=1e-18), k


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_stack_interpolation_64_to_256_slices_of_512(fbp, oracle, dt):
    cfg = I.CONFIGS[4]
    stack = np.random.default_rng(46).normal(size=(cfg.batch, cfg.image_n, cfg.image_n)).astype(_npdt(dt))
    want = oracle.interpolate_stack(stack.astype(np.float64), 4 * cfg.batch)
    with fbp.Plan(list(I.uniform_angles(4)), 2 * cfg.image_n, cfg.image_n, dtype=dt) as plan:
        got = plan.interpolate_stack(_dev(stack, dt), 4 * cfg.batch).cpu().numpy()
    eps = np.finfo(_npdt(dt)).eps                                          # bound as tests/test_next_gpu.py derives it
    assert np.abs(got.astype(np.float64) - want).max() <= 3 * eps * np.abs(stack).max()
