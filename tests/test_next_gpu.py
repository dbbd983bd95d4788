"""GPU parity for the rows SURVEY.md 8(f) marks "next": metrics (PSNR/SSIM), apodised filters,
per-angle weights -- each against oracle/fbp_oracle_ext.c on the same seeded inputs."""
import math

import numpy as np
import pytest

from paper_2109_02174_b200 import inputs as I

pytestmark = pytest.mark.gpu


def _np_dtype(dt):
    return np.float32 if dt == "f32" else np.float64


def _dev(a, dt):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=_np_dtype(dt))).cuda()


# fp64 sums on both sides; the GPU adds in a different (fixed) order and multiplies by 1/n: a few ulp
# of the largest partial sum.  1e-11 relative leaves room for the cancellation in 2 s_xy + C2.
METRIC_RTOL = 1e-11


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("shape", [(1,), (7,), (255, 257), (3, 512, 512), (2048, 2048)])
def test_metrics_match_oracle(fbp, oracle, dt, shape):
    import torch
    rng = np.random.default_rng(sum(shape))
    x = rng.uniform(-0.2, 1.1, shape).astype(_np_dtype(dt))
    y = (x + rng.normal(0, 0.01, shape)).astype(_np_dtype(dt))
    with fbp.Plan(list(I.uniform_angles(4)), 8, 4, dtype=dt) as plan:
        got = plan.metrics(_dev(x, dt), _dev(y, dt), 1.0)
        again = plan.metrics(_dev(x, dt), _dev(y, dt), 1.0)
        same = plan.metrics(_dev(x, dt), _dev(x, dt), 1.0)
        custom = plan.metrics(_dev(x, dt), _dev(y, dt), 2.0, c1=0.5, c2=0.25)
    want = oracle.metrics(x.astype(np.float64), y.astype(np.float64), 1.0)
    for k, v in want.items():
        assert got[k] == pytest.approx(v, rel=METRIC_RTOL, abs=1e-18), k
    assert got == again                                         # bit-identical across runs
    assert same["mse"] == 0.0 and math.isinf(same["psnr"]) and same["psnr"] > 0
    assert same["ssim"] == pytest.approx(1.0, abs=1e-14)
    want2 = oracle.metrics(x.astype(np.float64), y.astype(np.float64), 2.0, 0.5, 0.25)
    assert custom["ssim"] == pytest.approx(want2["ssim"], rel=METRIC_RTOL)
    assert custom["psnr"] == pytest.approx(want2["psnr"], rel=METRIC_RTOL)


def test_metrics_of_a_reconstruction_against_the_oracle_image(fbp, oracle):
    """The paper's use of the metrics (Tables 1-4): compare two reconstructions of the same slice.
    GPU fp32 vs oracle fp64 at config 2: PSNR is finite and large, SSIM ~ 1; run-to-run: inf / 1."""
    import torch
    cfg = I.CONFIGS[2]
    sino = I.config_sinogram(2).astype(np.float32)
    ref = oracle.reconstruct(sino.astype(np.float64), I.config_angles(2), cfg.image_n)
    with fbp.Plan(list(I.config_angles(2)), cfg.n_det, cfg.image_n, dtype="f32") as plan:
        a = plan.reconstruct(_dev(sino, "f32"))
        b = plan.reconstruct(_dev(sino, "f32"))
        r = torch.from_numpy(ref.astype(np.float32)).cuda()
        mx = float(ref.max())
        run_to_run = plan.metrics(a, b, mx)
        vs_ref = plan.metrics(a, r, mx)
    assert math.isinf(run_to_run["psnr"]) and run_to_run["ssim"] == pytest.approx(1.0, abs=1e-14)
    assert vs_ref["psnr"] > 100.0 and vs_ref["ssim"] > 0.999999


def test_metrics_error_paths(fbp):
    import torch
    with fbp.Plan(list(I.uniform_angles(4)), 8, 4, dtype="f32") as plan:
        x = torch.zeros(16, device="cuda")
        out = torch.full((8,), 7.0, dtype=torch.float64, device="cuda")
        for args in ((0, x, 16, 1.0), (x, 0, 16, 1.0), (x, x, 0, 1.0), (x, x, 16, 0.0), (x, x, 16, float("nan"))):
            with pytest.raises(fbp.FbpError) as ei:
                fbp.fbp_metrics(plan.handle, args[0], args[1], args[2], args[3], -1.0, -1.0, out)
            assert ei.value.status == fbp.FBP_EINVAL
        with pytest.raises(fbp.FbpError):
            fbp.fbp_metrics(plan.handle, x, x, 16, 1.0, -1.0, -1.0, 0)
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())
