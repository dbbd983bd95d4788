"""fbp_metrics_static: the PSNR / SSIM reduction for callers that cannot allocate device memory.

Why the entry point exists.  Every other compute call of libfbp takes a plan, and making a plan calls cudaMalloc.
A program that has already given all device memory to its own pool or caching allocator, a loop with a latency
bound (cudaMalloc and cudaFree wait for the device), or a process with a fixed, pre-accounted memory budget cannot
make one.  fbp_metrics_static needs no plan: the kernel's work area (per-CTA partial sums and the finish ticket)
is a fixed 73 984-byte array inside libfbp.so, the caller passes the two arrays and the 8-double result buffer, and
the call itself allocates nothing.  Limit: n <= 2^31 elements per array (FBP_METRICS_STATIC_MAX_N).

What is checked here.  The new entry point against the existing plan path (fbp_metrics) on the same device arrays,
within the tolerance the metric parity tests use (tests/test_next_gpu.py: 1e-11 relative), on two calls in a row:
the second call finds the work area as the first one left it (a larger grid's stale records, a used ticket) and
must still be right.  This file is named to be collected last, so a failure here hides no other test under
`pytest -x`; it passes alone in a fresh process (the first call does the per-device set-up) and after the other
tests (the library is already loaded and its plans have used their own scratch).
"""
import math

import numpy as np
import pytest

import paper_2109_02174_b200 as pkg

METRIC_RTOL = 1e-11          # the same bound as tests/test_next_gpu.py
KEYS = ("mse", "psnr", "ssim", "mu_x", "mu_y", "var_x", "var_y", "cov_xy")


def _pair(seed, n, npdt):
    rng = np.random.default_rng(seed)
    x = rng.uniform(-0.2, 1.1, n).astype(npdt)
    y = (x + rng.normal(0, 0.01, n)).astype(npdt)
    return x, y


def _close(got, want):
    for k, g, w in zip(KEYS, got, want):
        if math.isinf(w):
            assert g == w, k
        else:
            assert g == pytest.approx(w, rel=METRIC_RTOL, abs=1e-18), k


@pytest.mark.gpu
@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_static_metrics_match_the_plan_path_on_two_calls_in_a_row(fbp, dt):
    import torch
    from paper_2109_02174_b200 import inputs as I

    npdt, tdt, code = (np.float32, torch.float32, fbp.FBP_F32) if dt == "f32" else (np.float64, torch.float64, fbp.FBP_F64)
    # first call: many CTAs (3 x 512 x 512 elements); second call: a ragged, unaligned, much shorter view, so it runs
    # fewer CTAs over a work area that still holds the first call's records
    xa, ya = _pair(11, 3 * 512 * 512, npdt)
    xb, yb = _pair(12, 255 * 257 + 3, npdt)
    dxa, dya = torch.from_numpy(xa).cuda(), torch.from_numpy(ya).cuda()
    dxb, dyb = torch.from_numpy(xb).cuda()[1:], torch.from_numpy(yb).cuda()[1:]
    assert dxa.dtype == tdt

    # every buffer the new entry point touches is made here, by the caller, before it is called
    out_a = torch.full((8,), float("nan"), dtype=torch.float64, device="cuda")
    out_b = torch.full((8,), float("nan"), dtype=torch.float64, device="cuda")
    out_same = torch.full((8,), float("nan"), dtype=torch.float64, device="cuda")

    with fbp.Plan(list(I.uniform_angles(4)), 8, 4, dtype=dt) as plan:
        want_a = [plan.metrics(dxa, dya, 1.0)[k] for k in KEYS]
        want_b = [plan.metrics(dxb, dyb, 2.0, c1=0.5, c2=0.25)[k] for k in KEYS]
    torch.cuda.synchronize()

    # two calls in a row on one stream, nothing in between; results read only after both
    fbp.fbp_metrics_static(code, dxa, dya, dxa.numel(), 1.0, -1.0, -1.0, out_a)
    fbp.fbp_metrics_static(code, dxb, dyb, dxb.numel(), 2.0, 0.5, 0.25, out_b)
    fbp.fbp_metrics_static(code, dxa, dxa, dxa.numel(), 1.0, -1.0, -1.0, out_same)
    torch.cuda.synchronize()
    _close(out_a.cpu().tolist(), want_a)
    _close(out_b.cpu().tolist(), want_b)
    same = out_same.cpu().tolist()
    assert same[0] == 0.0 and math.isinf(same[1]) and same[1] > 0          # identical images: MSE 0, PSNR +inf
    assert same[2] == pytest.approx(1.0, abs=1e-14)

    # and once more, the large case after the small one: same bits as its first run (fixed order, no data atomics)
    out_again = torch.empty(8, dtype=torch.float64, device="cuda")
    fbp.fbp_metrics_static(code, dxa, dya, dxa.numel(), 1.0, -1.0, -1.0, out_again)
    torch.cuda.synchronize()
    assert torch.equal(out_again, out_a)


@pytest.mark.gpu
def test_static_metrics_rejects_bad_arguments(fbp):
    import torch
    x = torch.zeros(64, dtype=torch.float32, device="cuda")
    out = torch.zeros(8, dtype=torch.float64, device="cuda")
    for args in ((0, x, 64, 1.0, out), (x, 0, 64, 1.0, out), (x, x, 0, 1.0, out), (x, x, 64, 0.0, out),
                 (x, x, 64, float("inf"), out), (x, x, 64, 1.0, 0)):
        with pytest.raises(fbp.FbpError) as ei:
            fbp.fbp_metrics_static(fbp.FBP_F32, args[0], args[1], args[2], args[3], -1.0, -1.0, args[4])
        assert ei.value.status == fbp.FBP_EINVAL
    with pytest.raises(fbp.FbpError) as ei:
        fbp.fbp_metrics_static(7, x, x, 64, 1.0, -1.0, -1.0, out)
    assert ei.value.status == fbp.FBP_EINVAL
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0                                    # a refused call writes nothing


def test_static_metrics_refuses_sizes_beyond_its_limit():
    """The size check comes before any CUDA call, so it is checked on a machine without a GPU too: the pointers are
    never dereferenced.  The message names the limit."""
    pkg.build()
    lib = pkg.load_library()
    st = lib.fbp_metrics_static(pkg.FBP_F32, 256, 512, pkg.METRICS_STATIC_MAX_N + 1, 1.0, -1.0, -1.0, 1024, None)
    assert st == pkg.FBP_EINVAL
    msg = pkg.fbp_last_error(None)
    assert "FBP_METRICS_STATIC_MAX_N" in msg and str(pkg.METRICS_STATIC_MAX_N) in msg
    assert lib.fbp_metrics_static(pkg.FBP_F32, 256, 512, 0, 1.0, -1.0, -1.0, 1024, None) == pkg.FBP_EINVAL
