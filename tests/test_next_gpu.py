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


# ---- apodised windows (fbp_set_window) and per-angle weights (fbp_set_angle_weights) ----------
F64_TOL, F32_MAXABS, F32_RMSE = 1e-12, 1e-4, 1e-5


def _check_image(gpu, ref, dt, what):
    err = np.abs(np.asarray(gpu, dtype=np.float64) - ref)
    if dt == "f64":
        assert err.max() / np.abs(ref).max() <= F64_TOL, what
    else:
        dr = ref.max() - ref.min()
        if dr == 0.0:                      # a constant reference (1-pixel images): fall back to its magnitude
            dr = max(float(np.abs(ref).max()), 1e-30)
        assert err.max() / dr <= F32_MAXABS and math.sqrt(float(np.mean(err * err))) / dr <= F32_RMSE, what


def _check_filter(gpu, ref, dt, p_max, d, window, what):
    err = np.abs(np.asarray(gpu, dtype=np.float64) - ref).max()
    if dt == "f64":
        assert err / np.abs(ref).max() <= F64_TOL, what
    else:
        # n-term recursive fp32 sum, sum |h_W| <= 1/2 + 1/4 for every window here
        n_det = ref.shape[-1]
        assert err <= math.sqrt(n_det + 1) * 2.0 ** -24 * 0.75 * p_max / d, (what, err)


WINDOW_CASES = [  # (N, K, D, d, batch)
    (64, 90, 91, 1.0, 1),          # config 1 geometry
    (33, 7, 48, 0.5, 2),           # D even, N odd
    (130, 31, 185, 1.0, 1),
    (256, 24, 363, 1.0, 1),        # config 2 row length
    (40, 12, 725, 2.0, 1),         # config 3 row length
    (64, 5, 2897, 1.0, 1),         # config 5 row length: several filter units per row
]


@pytest.mark.parametrize("kind", [pytest.param(2, id="fft"), pytest.param(1, id="direct")])
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("window", ["shepp-logan", "cosine", "hamming", "hann"])
@pytest.mark.parametrize("case", WINDOW_CASES)
def test_windowed_filter_and_reconstruction_match_oracle(fbp, oracle, case, window, dt, kind):
    import torch
    n, k, dd, d, b = case
    ang = I.uniform_angles(k)
    sino = I.random_sinogram(21 + dd, b, k, dd).astype(_np_dtype(dt))
    ref_q = oracle.filter_sinogram_window(sino.astype(np.float64), window, d)
    ref_f = oracle.backproject(ref_q, ang, n, d)
    with fbp.Plan(list(ang), dd, n, det_spacing=d, dtype=dt, max_batch=b, options={"filter_kind": kind}) as plan:
        assert plan.info()["filter_kind"] == kind
        plan.set_window(window)
        ds = _dev(sino, dt)
        q = plan.filter(ds)
        f = plan.reconstruct(ds)
        f2 = plan.backproject(q)
        torch.cuda.synchronize()
        assert torch.equal(f, f2)                                 # reconstruct == backproject(filter)
        _check_filter(q.cpu().numpy(), ref_q, dt, np.abs(sino).max(), d, window, (case, window))
        _check_image(f.cpu().numpy(), ref_f, dt, (case, window))
        plan.set_window("ramlak")                                  # and back: the default path again
        f0 = plan.reconstruct(ds).cpu().numpy()
    _check_image(f0, oracle.reconstruct(sino.astype(np.float64), ang, n, d), dt, (case, "ramlak again"))


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_windowed_cfg3_full_image(fbp, oracle, dt):
    cfg = I.CONFIGS[3]
    ang = I.config_angles(3)
    sino = I.config_sinogram(3).astype(_np_dtype(dt))
    ref = oracle.backproject(oracle.filter_sinogram_window(sino.astype(np.float64), "hann"), ang, cfg.image_n)
    with fbp.Plan(list(ang), cfg.n_det, cfg.image_n, dtype=dt) as plan:
        plan.set_window("hann")
        a = plan.reconstruct(_dev(sino, dt))
        b = plan.reconstruct(_dev(sino, dt))
        assert bool((a == b).all())
    _check_image(a.cpu().numpy(), ref, dt, "cfg3 hann")


@pytest.mark.parametrize("b", [2, 9])
@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_angle_weights_match_oracle(fbp, oracle, dt, b):
    """Non-uniform angles with trapezoid weights; NULL restores pi/K.
    b = 9 takes the batch pipeline (filter and back-projection of slice groups on plan-owned streams)."""
    n, k, dd = 70, 41, 101
    rng = np.random.default_rng(17)
    ang = np.sort(rng.uniform(0.0, math.pi, k))
    edges = np.concatenate([[ang[-1] - math.pi], ang, [ang[0] + math.pi]])
    w = 0.5 * (edges[2:] - edges[:-2])                              # half the gap to each neighbour, periodic in pi
    assert w.sum() == pytest.approx(math.pi)
    q = I.random_sinogram(3, b, k, dd).astype(_np_dtype(dt))
    sino = I.random_sinogram(4, b, k, dd).astype(_np_dtype(dt))
    with fbp.Plan(list(ang), dd, n, dtype=dt, max_batch=b) as plan:
        plan.set_angle_weights(list(w))
        f_bp = plan.backproject(_dev(q, dt)).cpu().numpy()
        f_rc = plan.reconstruct(_dev(sino, dt)).cpu().numpy()
        plan.set_angle_weights(None)
        f_uni = plan.backproject(_dev(q, dt)).cpu().numpy()
    _check_image(f_bp, oracle.backproject_weighted(q.astype(np.float64), ang, w, n), dt, "weighted bp")
    ref_q = oracle.filter_sinogram(sino.astype(np.float64))
    _check_image(f_rc, oracle.backproject_weighted(ref_q, ang, w, n), dt, "weighted reconstruct")
    _check_image(f_uni, oracle.backproject(q.astype(np.float64), ang, n), dt, "uniform again")


def test_window_and_weight_error_paths(fbp):
    with fbp.Plan(list(I.uniform_angles(8)), 16, 8, dtype="f32") as plan:
        with pytest.raises(fbp.FbpError) as ei:
            fbp.fbp_set_window(plan.handle, 9)
        assert ei.value.status == fbp.FBP_EINVAL
        with pytest.raises(fbp.FbpError):
            fbp.fbp_set_angle_weights(plan.handle, [1.0] * 7 + [float("inf")], 8)
        with pytest.raises(ValueError):
            fbp.fbp_set_angle_weights(plan.handle, [1.0] * 7, 8)          # the C side would read 8 doubles
        with pytest.raises(ValueError):
            plan.set_angle_weights([1.0] * 3)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_metrics_unaligned_views_and_ragged_tails(fbp, oracle, dt):
    """Pointers that are not 16-byte aligned take the scalar path; lengths that are not a multiple of the
    vector width leave a tail: both must give the oracle's numbers."""
    rng = np.random.default_rng(99)
    x = rng.uniform(0, 1, 100003).astype(_np_dtype(dt))
    y = rng.uniform(0, 1, 100003).astype(_np_dtype(dt))
    dx, dy = _dev(x, dt), _dev(y, dt)
    with fbp.Plan(list(I.uniform_angles(4)), 8, 4, dtype=dt) as plan:
        for lo, hi in ((0, 100003), (1, 100003), (1, 99999), (3, 4)):
            got = plan.metrics(dx[lo:hi], dy[lo:hi], 1.0)
            want = oracle.metrics(x[lo:hi].astype(np.float64), y[lo:hi].astype(np.float64), 1.0)
            for k in ("mse", "psnr", "ssim", "var_x", "cov_xy"):
                assert got[k] == pytest.approx(want[k], rel=METRIC_RTOL, abs=1e-18), (lo, hi, k)


# ---- slice stack -> volume (fbp_interpolate_stack) -----------------------------------------------
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("n,n_in,n_out", [(64, 5, 9), (33, 3, 10), (7, 1, 4), (130, 8, 8), (512, 16, 61), (5, 2, 1)])
def test_stack_interpolation_matches_oracle(fbp, oracle, dt, n, n_in, n_out):
    """(1-t) a + t b in the working precision against the fp64 oracle: one rounding of t, one product, one
    fma => |err| <= 3 ulp of the larger operand (written out: 3 * eps * max|stack|)."""
    import torch
    rng = np.random.default_rng(n + n_in + n_out)
    stack = rng.normal(size=(n_in, n, n)).astype(_np_dtype(dt))
    want = oracle.interpolate_stack(stack.astype(np.float64), n_out)
    with fbp.Plan(list(I.uniform_angles(4)), 2 * n, n, dtype=dt) as plan:
        got = plan.interpolate_stack(_dev(stack, dt), n_out)
        again = plan.interpolate_stack(_dev(stack, dt), n_out)
        assert torch.equal(got, again)
    eps = np.finfo(_np_dtype(dt)).eps
    assert np.abs(got.cpu().numpy().astype(np.float64) - want).max() <= 3 * eps * np.abs(stack).max()
    if n_out == n_in:
        assert np.array_equal(got.cpu().numpy(), stack)             # same grid: t = 0 exactly, identity


def test_stack_interpolation_of_reconstructed_slices_and_errors(fbp, oracle):
    """The paper's use: reconstruct a stack (config-1 geometry, 6 noisy slices), then interpolate it to a volume."""
    import torch
    cfg = I.CONFIGS[1]
    clean = I.config_slice(1)
    sino = np.stack([I.gaussian_noise(clean * (1.0 + 0.05 * s), 0.01, 4100 + s) for s in range(6)]).astype(np.float32)
    ang = I.config_angles(1)
    ref = oracle.interpolate_stack(oracle.reconstruct(sino.astype(np.float64), ang, cfg.image_n), 16)
    with fbp.Plan(list(ang), cfg.n_det, cfg.image_n, dtype="f32", max_batch=6) as plan:
        vol = plan.interpolate_stack(plan.reconstruct(_dev(sino, "f32")), 16)
        _check_image(vol.cpu().numpy(), ref, "f32", "interpolated volume")
        st = torch.zeros(2, 64, 64, device="cuda")
        out = torch.full((3, 64, 64), 7.0, device="cuda")
        for args in ((0, 2, out, 3), (st, 0, out, 3), (st, 2, 0, 3), (st, 2, out, 0), (st, 2, st, 2)):
            with pytest.raises(fbp.FbpError) as ei:
                fbp.fbp_interpolate_stack(plan.handle, *args)
            assert ei.value.status == fbp.FBP_EINVAL
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())


def test_selfcheck_driver(fbp):
    import selfcheck                     # tests/selfcheck.py (the tests directory is on sys.path under pytest)
    assert selfcheck.main() == 0


# ---- matched forward projector R = B^T (fbp_project) ------------------------------------------------
PROJ_CASES = [  # (N, K, D, d, pix, angle kind, batch)
    (64, 90, 91, 1.0, None, "uniform", 1),
    (33, 9, 48, 1.0, None, "uniform", 2),
    (1, 3, 2, 1.0, None, "uniform", 1),
    (65, 37, 93, 0.5, 0.5, "uniform", 1),
    (40, 23, 70, 2.0, 1.0, "random", 2),          # pixel < bin: longer runs per line
    (50, 16, 40, 1.0, 1.0, "full", 1),            # detector shorter than the image: pixels fall off it
    (96, 12, 150, 0.7, 1.3, "random", 1),         # pixel > bin
    (256, 8, 363, 1.0, None, "axes", 1),          # exactly 0, pi/2, pi, ... : cos or sin = 0 and both majors
    (48, 7, 300, 3.0, 1.0, "random", 1),          # bins 3 pixels wide: wide windows, short staged blocks, 2 bin blocks
    (200, 5, 1100, 0.25, 1.0, "random", 1),       # pixels 4 bins wide: 5 bin blocks, most of them off the image
]


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("case", PROJ_CASES)
def test_forward_projector_matches_oracle_scatter(fbp, oracle, case, dt):
    import torch
    n, k, dd, d, pix, kind, b = case
    rng = np.random.default_rng(500 + n + k)
    if kind == "uniform":
        ang = I.uniform_angles(k)
    elif kind == "full":
        ang = I.uniform_angles(k, 2 * math.pi)
    elif kind == "axes":
        ang = np.arange(k) * (math.pi / 2)
    else:
        ang = np.sort(rng.uniform(-1.0, 4.0, size=k))
    img = rng.normal(size=(b, n, n)).astype(_np_dtype(dt))
    want = np.stack([oracle.forward_scatter(img[s].astype(np.float64), ang, dd, d, pix) for s in range(b)])
    with fbp.Plan(list(ang), dd, n, det_spacing=d, pixel_size=0.0 if pix is None else pix, dtype=dt, max_batch=b) as plan:
        got = plan.project(_dev(img, dt))
        again = plan.project(_dev(img, dt))
        assert torch.equal(got, again)
    _check_image(got.cpu().numpy(), want, dt, ("project", case))


def test_forward_projector_is_the_adjoint_of_the_backprojector_on_the_gpu(fbp):
    """<R x, y> = <x, B y> with both operators from the library (fp64), B = fbp_backproject / (pi/K)."""
    import torch
    n, k, dd = 70, 33, 101
    ang = np.sort(np.random.default_rng(2).uniform(0, math.pi, k))
    x = torch.from_numpy(np.random.default_rng(3).normal(size=(1, n, n))).cuda()
    y = torch.from_numpy(np.random.default_rng(4).normal(size=(1, k, dd))).cuda()
    with fbp.Plan(list(ang), dd, n, dtype="f64") as plan:
        rx = plan.project(x)
        by = plan.backproject(y) * (k / math.pi)
    lhs, rhs = float((rx * y).sum()), float((x * by).sum())
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs), float(rx.abs().max() * y.abs().sum()) * 1e-3)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_forward_projector_cfg3_sampled_rows(fbp, oracle, dt):
    """Config 3 size (512^2, 360 x 725) in the launch configuration bench.py --extras times; every 40th angle
    checked in full against the oracle, plus analytic sanity: projecting the rasterised phantom approximates
    the analytic sinogram (the generator's conventions agree with the projector's)."""
    cfg = I.CONFIGS[3]
    ang = I.config_angles(3)
    phantom = I.rasterise(I.random_ellipses(3), cfg.image_n).astype(_np_dtype(dt))
    sel = np.arange(0, cfg.n_angles, 40)
    want = oracle.forward_scatter(phantom.astype(np.float64), ang[sel], cfg.n_det)
    with fbp.Plan(list(ang), cfg.n_det, cfg.image_n, dtype=dt) as plan:
        got = plan.project(_dev(phantom[None], dt))[0].cpu().numpy()
    _check_image(got[sel], want, dt, "cfg3 project")
    analytic = I.config_sinogram(3)[0]
    assert np.abs(got - analytic).mean() <= 0.02 * np.abs(analytic).max()
