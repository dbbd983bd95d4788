"""tests/golden/: closed-form fixtures (each with its citation) against the oracle, and the
oracle-written fixture (tests/golden/make_golden.py) against the oracle and the CUDA path."""
import json
import math
import os

import numpy as np
import pytest

from paper_2109_02174_b200 import inputs as I

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _load(name):
    with open(os.path.join(GOLDEN, name)) as fh:
        return json.load(fh)


def test_closed_form_tap_sums(oracle):
    g = _load("closed_forms.json")["tap_sum"]
    for n_det, val in g["values"].items():
        assert math.fsum(oracle.taps(int(n_det))) == pytest.approx(val, rel=g["rel_tol"])


def test_closed_form_impulse_and_unity(oracle):
    g = _load("closed_forms.json")
    n, d = 9, 13
    for k in (7, 90):
        p = np.zeros((1, k, d))
        p[0, :, (d - 1) // 2] = 1.0
        f = oracle.reconstruct(p, I.uniform_angles(k), n)
        assert f[0, n // 2, n // 2] == pytest.approx(g["impulse_centre_pixel"]["value_d1"], rel=1e-14)
    q = np.ones((1, 5, 13))
    f = oracle.backproject(q, I.uniform_angles(5), 8)
    assert np.allclose(f, g["partition_of_unity"]["value"], rtol=g["partition_of_unity"]["rel_tol"], atol=0)


def test_closed_form_disk_filtered_centre(oracle):
    g = _load("closed_forms.json")["disk_filtered_interior"]
    for case in g["cases"]:
        n_det, rad = case["n_det"], case["radius"]
        t = I.detector_coords(n_det)
        p = 2.0 * np.sqrt(np.maximum(rad * rad - t * t, 0.0))
        q = oracle.filter_sinogram(p[None, None, :])
        assert q[0, 0, (n_det - 1) // 2] == pytest.approx(g["value_rho1"], abs=case["abs_tol_centre"])


def test_input_recipe_and_oracle_reproduce_the_stored_values(oracle):
    g = _load("oracle_cfg1.json")
    sino32 = I.config_sinogram(1).astype(np.float32)
    assert I.sha256(sino32) == g["input_sha256_f32"]
    sino = sino32.astype(np.float64)
    f = oracle.reconstruct(sino, I.config_angles(1), 64)
    q = oracle.filter_sinogram(sino)
    for r, c, v in g["image_samples"]:
        assert f[0, r, c] == pytest.approx(v, rel=1e-13, abs=1e-15)
    for i, n, v in g["filtered_samples"]:
        assert q[0, i, n] == pytest.approx(v, rel=1e-13, abs=1e-15)


@pytest.mark.gpu
@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_gpu_matches_the_stored_oracle_values(fbp, dt):
    import torch
    g = _load("oracle_cfg1.json")
    npdt = np.float32 if dt == "f32" else np.float64
    sino = I.config_sinogram(1).astype(np.float32).astype(npdt)     # the stored values are for the fp32-rounded input
    with fbp.Plan(list(I.config_angles(1)), 91, 64, dtype=dt) as plan:
        ds = torch.from_numpy(sino).cuda()
        f = plan.reconstruct(ds).cpu().numpy().astype(np.float64)
        q = plan.filter(ds).cpu().numpy().astype(np.float64)
    dr = g["image_max"] - g["image_min"]
    tol_f = 1e-4 * dr if dt == "f32" else 1e-12 * max(abs(g["image_max"]), abs(g["image_min"]))
    for r, c, v in g["image_samples"]:
        assert abs(f[0, r, c] - v) <= tol_f, (r, c)
    p_max = float(np.abs(sino).max())
    tol_q = math.sqrt(91 / 2 + 1) * 2.0 ** -24 * 0.5 * p_max if dt == "f32" else 1e-12 * p_max
    for i, n, v in g["filtered_samples"]:
        assert abs(q[0, i, n] - v) <= tol_q, (i, n)
