"""Pins for oracle/fbp_oracle_ext.c (the rows SURVEY.md 8(f) marks "next"): apodised filter taps,
per-angle weights, PSNR / SSIM.  None compares the oracle with itself or with the CUDA path."""
import math

import numpy as np
import pytest
import scipy.integrate

from paper_2109_02174_b200 import inputs as I

PI = math.pi
WINDOW_FUNCS = {
    "ramlak": lambda f: 1.0,
    "shepp-logan": lambda f: np.sinc(f),                       # sin(pi f)/(pi f)
    "cosine": lambda f: math.cos(PI * f),
    "hamming": lambda f: 0.54 + 0.46 * math.cos(2 * PI * f),
    "hann": lambda f: 0.5 + 0.5 * math.cos(2 * PI * f),
}


@pytest.mark.parametrize("name", list(WINDOW_FUNCS))
def test_w1_taps_are_the_defining_integral(oracle, name):
    """h_W[m] = 2 int_0^{1/2} f W(f) cos(2 pi f m) df by adaptive quadrature (scipy), m = 0..12 and a far tap.
    Catches: a wrong closed form, a wrong window constant, a sign or factor-2 slip."""
    d = 64
    h = oracle.window_taps(d, name)
    w = WINDOW_FUNCS[name]
    for m in list(range(0, 13)) + [37, 63]:
        val, _ = scipy.integrate.quad(lambda f: 2.0 * f * w(f) * math.cos(2 * PI * f * m), 0.0, 0.5,
                                      epsabs=1e-14, epsrel=1e-13, limit=400)
        assert h[d - 1 + m] == pytest.approx(val, abs=5e-13), (name, m)
        assert h[d - 1 - m] == h[d - 1 + m]


@pytest.mark.parametrize("name", list(WINDOW_FUNCS))
def test_w1_dtft_of_taps_is_the_apodised_ramp(oracle, name):
    d = 4097
    h = oracle.window_taps(d, name)
    m = np.arange(-(d - 1), d)
    for f in (0.0, 0.07, 0.2, 0.33, 0.5):
        val = float(np.sum(h * np.cos(2 * PI * f * m)))
        assert val == pytest.approx(abs(f) * WINDOW_FUNCS[name](f), abs=3e-4), (name, f)


def test_w1_window_0_is_the_core_ramlak_and_known_values(oracle):
    assert np.array_equal(oracle.window_taps(33, "ramlak"), oracle.taps(33))
    h = oracle.window_taps(9, "shepp-logan")
    assert h[8] == pytest.approx(2.0 / PI**2, rel=1e-15)               # m = 0: -2/(pi^2 (0 - 1))
    assert h[9] == pytest.approx(-2.0 / (3.0 * PI**2), rel=1e-15)      # m = 1
    hn = oracle.window_taps(9, "hann")
    assert hn[8] == pytest.approx(0.125 - 0.5 / PI**2, rel=1e-14)      # 0.5/4 + 0.25 * 2 * (-1/pi^2)
    assert hn[10] == pytest.approx(0.25 * (-1 / PI**2 - 1 / (9 * PI**2)), rel=1e-14)   # m = 2: neighbours 1 and 3


@pytest.mark.parametrize("name", ["shepp-logan", "hann"])
def test_w1_filter_is_numpy_convolve(oracle, name):
    d, k = 45, 3
    p = I.random_sinogram(11, 1, k, d)[0]
    h = oracle.window_taps(d, name)
    q = oracle.filter_sinogram_window(p, name, det_spacing=0.5)
    for i in range(k):
        want = np.convolve(p[i], h)[d - 1:2 * d - 1] / 0.5
        assert np.allclose(q[i], want, rtol=1e-13, atol=1e-14)


def test_w2_weights_reduce_to_uniform_and_are_linear(oracle):
    n, k, d = 17, 9, 27
    ang = np.sort(np.random.default_rng(3).uniform(0, PI, k))
    q = I.random_sinogram(4, 2, k, d)
    uni = oracle.backproject_weighted(q, ang, np.full(k, PI / k), n)
    assert np.allclose(uni, oracle.backproject(q, ang, n), rtol=1e-13, atol=1e-14)
    # a one-hot weight vector isolates one angle: the sum over one-hots with weights w is the weighted result
    w = np.random.default_rng(5).uniform(0.1, 1.0, k)
    parts = sum(w[i] * oracle.backproject_weighted(q, ang, np.eye(k)[i], n) for i in range(k))
    assert np.allclose(oracle.backproject_weighted(q, ang, w, n), parts, rtol=1e-12, atol=1e-13)
    # single angle 0 with weight w0: image rows are w0 * interp of the row (axis convention as P6)
    one = oracle.backproject_weighted(q[0, :1], np.zeros(1), np.array([0.37]), n)
    x = np.arange(n) - (n - 1) / 2 + (d - 1) / 2
    assert np.allclose(one[5], 0.37 * np.interp(x, np.arange(d), q[0, 0]), rtol=1e-13)


def test_w2_weight_i_belongs_to_angle_i(oracle):
    """Pins the weight <-> angle ASSOCIATION (eq. 2 weighted) against code that is not the
    weighted routine: (a) one-hot weight e_i == the core back-projector (pinned by P4-P7, P12) applied to the
    sinogram with every row but i zeroed, times K/pi; (b) random non-uniform weights == the dense brute-force
    matrix of P7 (independent triple loop, 8x8) with the columns of angle i scaled by w_i.
    A mis-indexed weight (weights[K-1-i], weights[(i+1)%K]) fails both."""
    n, k, d = 13, 7, 21
    ang = np.sort(np.random.default_rng(31).uniform(0, PI, k))          # non-uniform: no angle symmetry to hide behind
    q = I.random_sinogram(41, 1, k, d)[0]
    for i in range(k):
        only_i = np.zeros_like(q)
        only_i[i] = q[i]
        want = oracle.backproject(only_i, ang, n) * (k / PI)
        got = oracle.backproject_weighted(q, ang, np.eye(k)[i], n)
        assert np.allclose(got, want, rtol=1e-13, atol=1e-15), i
        assert np.abs(want).max() > 0
    # dense W (n^2 x K D) by an independent triple loop, columns of angle i scaled by w_i
    n, k, d, dd, pix = 8, 5, 13, 1.0, 1.0
    ang = np.sort(np.random.default_rng(32).uniform(0, PI, k))
    w = np.random.default_rng(33).uniform(0.2, 2.0, k)
    q = I.random_sinogram(42, 1, k, d)[0]
    w_mat = np.zeros((n * n, k * d))
    for r in range(n):
        for c in range(n):
            for i in range(k):
                u = ((c - (n - 1) / 2) * pix * math.cos(ang[i]) + (r - (n - 1) / 2) * pix * math.sin(ang[i])) / dd + (d - 1) / 2
                j = math.floor(u)
                if 0 <= j < d:
                    w_mat[r * n + c, i * d + j] += (1.0 - (u - j)) * w[i]
                if 0 <= j + 1 < d:
                    w_mat[r * n + c, i * d + j + 1] += (u - j) * w[i]
    want = (w_mat @ q.ravel()).reshape(n, n)
    assert np.allclose(oracle.backproject_weighted(q, ang, w, n), want, rtol=1e-13, atol=1e-14)
    # and the batch axis keeps slices apart
    q2 = I.random_sinogram(43, 2, k, d)
    both = oracle.backproject_weighted(q2, ang, w, n)
    assert np.allclose(both[1], (w_mat @ q2[1].ravel()).reshape(n, n), rtol=1e-13, atol=1e-14)


def test_m1_psnr_ssim_closed_forms(oracle):
    rng = np.random.default_rng(8)
    x = rng.uniform(0, 1, (31, 29))
    same = oracle.metrics(x, x, 1.0)
    assert same["mse"] == 0.0 and math.isinf(same["psnr"]) and same["ssim"] == pytest.approx(1.0, abs=1e-15)
    # constant offset c: MSE = c^2, PSNR = 20 log10(MAX/c); variances and covariance unchanged
    c = 0.05
    off = oracle.metrics(x, x + c, 1.0)
    assert off["mse"] == pytest.approx(c * c, rel=1e-12)
    assert off["psnr"] == pytest.approx(20 * math.log10(1.0 / c), rel=1e-12)
    mu, var = x.mean(), x.var()
    c1, c2 = 1e-4, 9e-4
    want = (2 * mu * (mu + c) + c1) * (2 * var + c2) / ((mu**2 + (mu + c)**2 + c1) * (2 * var + c2))
    assert off["ssim"] == pytest.approx(want, rel=1e-12)
    # scaling y = a x: s_xy = a var, s_y^2 = a^2 var
    a = 0.8
    sc = oracle.metrics(x, a * x, 1.0)
    want = (2 * a * mu * mu + c1) * (2 * a * var + c2) / ((mu * mu * (1 + a * a) + c1) * (var * (1 + a * a) + c2))
    assert sc["ssim"] == pytest.approx(want, rel=1e-12)
    # numpy restatement on unrelated images
    y = rng.uniform(0, 1, x.shape)
    m = oracle.metrics(x, y, 1.0)
    assert m["mse"] == pytest.approx(np.mean((x - y) ** 2), rel=1e-13)
    assert m["cov_xy"] == pytest.approx(np.mean((x - x.mean()) * (y - y.mean())), rel=1e-12)
    assert m["var_y"] == pytest.approx(y.var(), rel=1e-13)


def test_s1_stack_interpolation_is_numpy_interp_along_z(oracle):
    """Pins: numpy.interp per pixel column (library routine), endpoints, midpoints, exactness on a linear ramp."""
    rng = np.random.default_rng(12)
    stack = rng.normal(size=(5, 3, 4))
    for n_out in (1, 2, 5, 9, 14):
        got = oracle.interpolate_stack(stack, n_out)
        z = np.linspace(0.0, 4.0, n_out) if n_out > 1 else np.zeros(1)
        for r in range(3):
            for c in range(4):
                assert np.allclose(got[:, r, c], np.interp(z, np.arange(5), stack[:, r, c]), rtol=1e-14, atol=1e-15)
    assert np.array_equal(oracle.interpolate_stack(stack, 5), stack)                    # same grid: identity
    nine = oracle.interpolate_stack(stack, 9)
    assert np.array_equal(nine[::2], stack) and np.allclose(nine[1::2], 0.5 * (stack[:-1] + stack[1:]), rtol=1e-15)
    ramp = np.arange(4.0)[:, None, None] * np.ones((1, 2, 2)) * 3.0 + 1.0              # linear in z: reproduced exactly
    assert np.allclose(oracle.interpolate_stack(ramp, 10)[:, 0, 0], 1.0 + 3.0 * np.linspace(0, 3, 10), rtol=1e-15)
    assert np.array_equal(oracle.interpolate_stack(stack[:1], 3), np.repeat(stack[:1], 3, axis=0))
