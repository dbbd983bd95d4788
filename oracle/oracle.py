"""ctypes front-end of the C oracle (``fbp_oracle.c``).  Test infrastructure only.

Argument marshalling only: every number is computed in ``fbp_oracle.c``.  ``build()``
compiles it with ``gcc -O2 -fopenmp`` (no -ffast-math) into ``oracle/libfbp_oracle.so``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fbp_oracle.c")
_SRC_EXT = os.path.join(_HERE, "fbp_oracle_ext.c")
_SRC_FDK = os.path.join(_HERE, "fbp_oracle_fdk.c")
_LIB = os.path.join(_HERE, "libfbp_oracle.so")
_lock = threading.Lock()
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile the oracle if the shared object is missing or older than its source."""
    with _lock:
        stale = (force or not os.path.exists(_LIB)
                 or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_EXT), os.path.getmtime(_SRC_FDK)))
        if stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, _SRC_EXT, _SRC_FDK, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.fbp_oracle_max_threads.restype = ctypes.c_int
        lib.fbp_oracle_taps.argtypes = [ctypes.c_int, _dp]
        lib.fbp_oracle_filter.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_double, ctypes.c_int]
        lib.fbp_oracle_backproject.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp,
                                               ctypes.c_double, ctypes.c_int, ctypes.c_double,
                                               ctypes.c_int, ctypes.c_int]
        lib.fbp_oracle_backproject_pixels.argtypes = [_dp, _ip, _ip, ctypes.c_long, _dp, ctypes.c_int,
                                                      ctypes.c_int, _dp, ctypes.c_double, ctypes.c_int,
                                                      ctypes.c_double, ctypes.c_int]
        lib.fbp_oracle_filter_rows.argtypes = [_dp, _ip, ctypes.c_long, _dp, ctypes.c_int,
                                               ctypes.c_double, ctypes.c_int]
        lib.fbp_oracle_forward_scatter.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, _dp,
                                                   ctypes.c_double, ctypes.c_int, ctypes.c_double]
        lib.fbp_oracle_reconstruct.argtypes = [_dp, _dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                               _dp, ctypes.c_double, ctypes.c_int, ctypes.c_double,
                                               ctypes.c_int]
        lib.fbp_oracle_window_taps.argtypes = [ctypes.c_int, ctypes.c_int, _dp]
        lib.fbp_oracle_window_taps.restype = None
        lib.fbp_oracle_filter_window.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                 ctypes.c_double, ctypes.c_int, ctypes.c_int]
        lib.fbp_oracle_filter_window.restype = None
        lib.fbp_oracle_backproject_weighted.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, _dp,
                                                        ctypes.c_double, ctypes.c_int, ctypes.c_double, ctypes.c_int]
        lib.fbp_oracle_backproject_weighted.restype = None
        lib.fbp_oracle_metrics.argtypes = [_dp, _dp, ctypes.c_long, ctypes.c_double, ctypes.c_double,
                                           ctypes.c_double, _dp]
        lib.fbp_oracle_metrics.restype = None
        lib.fbp_oracle_interpolate_stack.argtypes = [_dp, ctypes.c_int, _dp, ctypes.c_int, ctypes.c_long]
        lib.fbp_oracle_interpolate_stack.restype = None
        lib.fbp_oracle_fdk_weight.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                              ctypes.c_double, ctypes.c_double]
        lib.fbp_oracle_fdk_weight.restype = None
        lib.fbp_oracle_fdk_backproject.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, ctypes.c_double,
                                                   ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_double,
                                                   ctypes.c_int, ctypes.c_double, ctypes.c_int]
        lib.fbp_oracle_fdk_backproject.restype = None
        for fn in ("fbp_oracle_taps", "fbp_oracle_filter", "fbp_oracle_backproject",
                   "fbp_oracle_backproject_pixels", "fbp_oracle_filter_rows",
                   "fbp_oracle_forward_scatter", "fbp_oracle_reconstruct"):
            getattr(lib, fn).restype = None
        _lib = lib
    return _lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _stack3(a) -> np.ndarray:
    a = _f64(a)
    if a.ndim == 2:
        a = a[None]
    if a.ndim != 3:
        raise ValueError("expected [K][D] or [B][K][D]")
    return a


def max_threads() -> int:
    return int(_load().fbp_oracle_max_threads())


def taps(n_det: int) -> np.ndarray:
    """h[m], m = -(D-1)..D-1, returned as an array of 2D-1 values (index m + D-1)."""
    h = np.empty(2 * n_det - 1, dtype=np.float64)
    _load().fbp_oracle_taps(int(n_det), _p(h))
    return h


def filter_sinogram(sino, det_spacing: float = 1.0, threads: int = 0) -> np.ndarray:
    """Q = (1/d) h * P along the last axis; input [K][D] or [B][K][D], output same shape."""
    p = _f64(sino)
    p3 = _stack3(p)
    q = np.empty_like(p3)
    b, k, d = p3.shape
    _load().fbp_oracle_filter(_p(p3), _p(q), b, k, d, float(det_spacing), int(threads))
    return q.reshape(p.shape)


def filter_rows(sino2d, row_ids, det_spacing: float = 1.0, threads: int = 0) -> np.ndarray:
    """Filter only the listed rows of a [R][D] array; returns [len(row_ids)][D]."""
    p = _f64(sino2d)
    assert p.ndim == 2
    ids = _i32(row_ids)
    q = np.empty((ids.size, p.shape[1]), dtype=np.float64)
    _load().fbp_oracle_filter_rows(_p(p), ids.ctypes.data_as(_ip), ids.size, _p(q), p.shape[1],
                                   float(det_spacing), int(threads))
    return q


def backproject(filtered, angles, image_n: int, det_spacing: float = 1.0, pixel_size: float | None = None,
                scaled: bool = True, threads: int = 0) -> np.ndarray:
    """f = (pi/K) sum_i interp(Q_i, u_i) (scaled) or the bare sum B (scaled=False)."""
    q = _f64(filtered)
    q3 = _stack3(q)
    ang = _f64(angles)
    b, k, d = q3.shape
    assert ang.shape == (k,)
    pix = float(det_spacing if pixel_size is None else pixel_size)
    f = np.empty((b, image_n, image_n), dtype=np.float64)
    _load().fbp_oracle_backproject(_p(q3), _p(f), b, k, d, _p(ang), float(det_spacing), int(image_n), pix,
                                   1 if scaled else 0, int(threads))
    return f[0] if q.ndim == 2 else f


def backproject_pixels(filtered2d, angles, image_n: int, rows, cols, det_spacing: float = 1.0,
                       pixel_size: float | None = None, threads: int = 0) -> np.ndarray:
    """Scaled back-projection of the listed pixels of ONE slice [K][D]."""
    q = _f64(filtered2d)
    assert q.ndim == 2
    ang = _f64(angles)
    rr, cc = _i32(rows), _i32(cols)
    assert rr.shape == cc.shape and ang.shape == (q.shape[0],)
    pix = float(det_spacing if pixel_size is None else pixel_size)
    out = np.empty(rr.size, dtype=np.float64)
    _load().fbp_oracle_backproject_pixels(_p(q), rr.ctypes.data_as(_ip), cc.ctypes.data_as(_ip), rr.size,
                                          _p(out), q.shape[0], q.shape[1], _p(ang), float(det_spacing),
                                          int(image_n), pix, int(threads))
    return out


def forward_scatter(image2d, angles, n_det: int, det_spacing: float = 1.0,
                    pixel_size: float | None = None) -> np.ndarray:
    """R x = B^T x as an independent scatter (adjoint pin P8); one slice [N][N] -> [K][D]."""
    x = _f64(image2d)
    assert x.ndim == 2 and x.shape[0] == x.shape[1]
    ang = _f64(angles)
    pix = float(det_spacing if pixel_size is None else pixel_size)
    y = np.empty((ang.size, n_det), dtype=np.float64)
    _load().fbp_oracle_forward_scatter(_p(x), _p(y), ang.size, int(n_det), _p(ang), float(det_spacing),
                                       x.shape[0], pix)
    return y


def reconstruct(sino, angles, image_n: int, det_spacing: float = 1.0, pixel_size: float | None = None,
                threads: int = 0) -> np.ndarray:
    """Filter then back-project (eq. 2)."""
    p = _f64(sino)
    p3 = _stack3(p)
    ang = _f64(angles)
    b, k, d = p3.shape
    assert ang.shape == (k,)
    pix = float(det_spacing if pixel_size is None else pixel_size)
    work = np.empty_like(p3)
    f = np.empty((b, image_n, image_n), dtype=np.float64)
    _load().fbp_oracle_reconstruct(_p(p3), _p(work), _p(f), b, k, d, _p(ang), float(det_spacing),
                                   int(image_n), pix, int(threads))
    return f[0] if p.ndim == 2 else f


# ---- rows SURVEY.md 8(f) marks "next" (fbp_oracle_ext.c) --------------------------------------
WINDOWS = {"ramlak": 0, "shepp-logan": 1, "cosine": 2, "hamming": 3, "hann": 4}


def window_taps(n_det: int, window) -> np.ndarray:
    """h_W[m], m = -(D-1)..D-1, of the apodised ramp |f| W(f) (W1 of fbp_oracle_ext.c)."""
    lib = _load()
    out = np.empty(2 * n_det - 1, dtype=np.float64)
    lib.fbp_oracle_window_taps(int(n_det), int(WINDOWS.get(window, window)), _p(out))
    return out


def filter_sinogram_window(sino, window, det_spacing: float = 1.0, threads: int = 0) -> np.ndarray:
    lib = _load()
    p = _stack3(sino)
    q = np.empty_like(p)
    lib.fbp_oracle_filter_window(_p(p), _p(q), p.shape[0], p.shape[1], p.shape[2], float(det_spacing),
                                 int(WINDOWS.get(window, window)), int(threads))
    return q.reshape(np.shape(sino))


def backproject_weighted(filtered, angles, weights, image_n: int, det_spacing: float = 1.0,
                         pixel_size: float | None = None, threads: int = 0) -> np.ndarray:
    """f = sum_i w_i lerp(Q_i, u_i): eq. 2 with caller-supplied per-angle weights (W2)."""
    lib = _load()
    q = _stack3(filtered)
    ang, wts = _f64(angles), _f64(weights)
    assert ang.shape == wts.shape == (q.shape[1],)
    pix = float(det_spacing if pixel_size is None else pixel_size)
    f = np.empty((q.shape[0], image_n, image_n), dtype=np.float64)
    lib.fbp_oracle_backproject_weighted(_p(q), _p(f), q.shape[0], q.shape[1], q.shape[2], _p(ang), _p(wts),
                                        float(det_spacing), int(image_n), pix, int(threads))
    return f if np.ndim(filtered) == 3 else f[0]


def metrics(x, y, max_val: float, c1: float | None = None, c2: float | None = None) -> dict:
    """MSE, PSNR (eq. 3) and global-statistics SSIM (eq. 4) of one image pair (M1)."""
    lib = _load()
    a, b = _f64(x).ravel(), _f64(y).ravel()
    assert a.shape == b.shape
    c1 = (0.01 * max_val) ** 2 if c1 is None else c1
    c2 = (0.03 * max_val) ** 2 if c2 is None else c2
    out = np.empty(8, dtype=np.float64)
    lib.fbp_oracle_metrics(_p(a), _p(b), a.size, float(max_val), float(c1), float(c2), _p(out))
    keys = ("mse", "psnr", "ssim", "mu_x", "mu_y", "var_x", "var_y", "cov_xy")
    return dict(zip(keys, (float(v) for v in out)))


def interpolate_stack(stack, n_out: int) -> np.ndarray:
    """Linear interpolation along the stack axis to n_out slices (S1 of fbp_oracle_ext.c)."""
    lib = _load()
    a = _f64(stack)
    assert a.ndim == 3
    out = np.empty((int(n_out),) + a.shape[1:], dtype=np.float64)
    lib.fbp_oracle_interpolate_stack(_p(a), a.shape[0], _p(out), int(n_out), a.shape[1] * a.shape[2])
    return out


# ---- cone-beam FDK (fbp_oracle_fdk.c) -----------------------------------------------------------
def fdk_weight(proj, d_a: float, d_b: float, sad: float) -> np.ndarray:
    """C3: cosine pre-weight sad / sqrt(sad^2 + a^2 + b^2) of projections [K][n_b][n_a]."""
    lib = _load()
    p = _f64(proj)
    assert p.ndim == 3
    out = np.empty_like(p)
    lib.fbp_oracle_fdk_weight(_p(p), _p(out), p.shape[0], p.shape[1], p.shape[2], float(d_a), float(d_b), float(sad))
    return out


def fdk_backproject(filtered, angles, sad: float, image_n: int, n_z: int, d_a: float = 1.0, d_b: float = 1.0,
                    pixel_size: float | None = None, voxel_z: float | None = None, threads: int = 0) -> np.ndarray:
    """C5: volume [n_z][N][N] from filtered, weighted projections [K][n_b][n_a]."""
    lib = _load()
    q = _f64(filtered)
    ang = _f64(angles)
    assert q.ndim == 3 and ang.shape == (q.shape[0],)
    pix = float(d_a if pixel_size is None else pixel_size)
    vz = float(pix if voxel_z is None else voxel_z)
    f = np.empty((int(n_z), int(image_n), int(image_n)), dtype=np.float64)
    lib.fbp_oracle_fdk_backproject(_p(q), _p(f), q.shape[0], q.shape[1], q.shape[2], _p(ang), float(d_a), float(d_b),
                                   float(sad), int(image_n), pix, int(n_z), vz, int(threads))
    return f


def fdk_reconstruct(proj, angles, sad: float, image_n: int, n_z: int, d_a: float = 1.0, d_b: float = 1.0,
                    pixel_size: float | None = None, voxel_z: float | None = None, threads: int = 0) -> np.ndarray:
    """FDK end to end: pre-weight (C3), Ram-Lak row filter (C4 = O2 of fbp_oracle.c on every detector row),
    weighted cone-beam back-projection (C5)."""
    w = fdk_weight(proj, d_a, d_b, sad)
    k, nb, na = w.shape
    q = filter_sinogram(w.reshape(k * nb, na), d_a, threads).reshape(k, nb, na)
    return fdk_backproject(q, angles, sad, image_n, n_z, d_a, d_b, pixel_size, voxel_z, threads)
