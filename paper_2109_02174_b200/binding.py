"""ctypes binding of libfbp (include/fbp.h): argument marshalling only.

Every step of the path (filter, then back-projection) runs in the CUDA
kernels of ``csrc/``.  There is no CPU fallback: if ``libfbp.so`` is missing or fails to
load, ``load_library`` raises.  torch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

FBP_F32, FBP_F64 = 0, 1
FBP_OK, FBP_EINVAL, FBP_ENOMEM, FBP_ECUDA, FBP_EUNSUPPORTED = 0, 1, 2, 3, 4
STATUS_NAMES = {0: "FBP_OK", 1: "FBP_EINVAL", 2: "FBP_ENOMEM", 3: "FBP_ECUDA", 4: "FBP_EUNSUPPORTED"}

EXPORTS = (
    "fbp_create", "fbp_create_tuned", "fbp_filter", "fbp_backproject", "fbp_reconstruct", "fbp_reconstruct_host",
    "fbp_destroy", "fbp_last_error", "fbp_plan_info", "fbp_set_profiling", "fbp_get_kernel_ms",
    "fbp_set_trace", "fbp_metrics", "fbp_set_window", "fbp_set_angle_weights", "fbp_interpolate_stack", "fbp_project", "fbp_fdk_reconstruct",
    "fbp_metrics_static", "fbp_measure_issue_rate",
)

PLAN_INFO_FIELDS = (
    "bp_tile_w", "bp_tile_h", "bp_pixels_per_thread", "bp_angle_splits", "bp_angles_per_chunk",
    "bp_segment_len", "bp_ctas_per_slice", "bp_threads", "bp_smem_bytes",
    "filter_outputs_per_thread", "filter_threads", "filter_input_slices", "filter_smem_bytes",
    "kernels_per_reconstruct", "filter_units_per_row", "device_sms", "filter_ctas", "filter_kind",
    "fft_length",
)

# keys of fbp_create_tuned (include/fbp.h, fbp_option)
OPTIONS = {
    "bp_variant": 1, "bp_splits": 2, "bp_chunk": 3, "filter_r": 4, "filter_sb": 5, "filter_kind": 6,
    "pipeline": 7, "pipe_group": 8, "pipe_min_batch": 9, "pdl": 10, "host_zero_copy": 11, "bp_even": 13,
}

_lib = None


class FbpError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), message))
        self.status = status


def load_library(path: str | None = None) -> ctypes.CDLL:
    """Load libfbp.so (built in-tree by ``build.build()``); raise if it is not there."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or _build.LIB          # an A/B build of the library is loaded by passing its path: nothing else picks the file
    if not os.path.exists(path):
        raise FileNotFoundError(
            "%s not found: build it with `python -m paper_2109_02174_b200.build` "
            "(there is no CPU fallback)" % path)
    lib = ctypes.CDLL(path)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    lib.fbp_create.argtypes = [ctypes.POINTER(vp), ci, ci, ctypes.POINTER(cd), cd, ci, cd, ci, ci, ci]
    lib.fbp_create.restype = ci
    lib.fbp_create_tuned.argtypes = [ctypes.POINTER(vp), ci, ci, ctypes.POINTER(cd), cd, ci, cd, ci, ci, ci,
                                     ctypes.POINTER(ci), ci]
    lib.fbp_create_tuned.restype = ci
    for name in ("fbp_filter", "fbp_backproject", "fbp_reconstruct", "fbp_reconstruct_host", "fbp_project"):
        fn = getattr(lib, name)
        fn.argtypes = [vp, vp, vp, ci, vp]
        fn.restype = ci
    lib.fbp_metrics.argtypes = [vp, vp, vp, ctypes.c_longlong, cd, cd, cd, vp, vp]
    lib.fbp_metrics.restype = ci
    lib.fbp_metrics_static.argtypes = [ci, vp, vp, ctypes.c_longlong, cd, cd, cd, vp, vp]
    lib.fbp_metrics_static.restype = ci
    lib.fbp_measure_issue_rate.argtypes = [ci, ctypes.POINTER(cd)]
    lib.fbp_measure_issue_rate.restype = ci
    lib.fbp_set_window.argtypes = [vp, ci]
    lib.fbp_set_window.restype = ci
    lib.fbp_set_angle_weights.argtypes = [vp, ctypes.POINTER(cd)]
    lib.fbp_set_angle_weights.restype = ci
    lib.fbp_interpolate_stack.argtypes = [vp, vp, ci, vp, ci, vp]
    lib.fbp_interpolate_stack.restype = ci
    lib.fbp_fdk_reconstruct.argtypes = [vp, vp, vp, ci, cd, cd, ci, cd, vp]
    lib.fbp_fdk_reconstruct.restype = ci
    lib.fbp_destroy.argtypes = [vp]
    lib.fbp_destroy.restype = None
    lib.fbp_last_error.argtypes = [vp]
    lib.fbp_last_error.restype = ctypes.c_char_p
    lib.fbp_plan_info.argtypes = [vp, ctypes.POINTER(ci), ci]
    lib.fbp_plan_info.restype = ci
    lib.fbp_set_trace.argtypes = [vp, vp, ctypes.c_longlong]
    lib.fbp_set_trace.restype = ci
    lib.fbp_set_profiling.argtypes = [vp, ci]
    lib.fbp_set_profiling.restype = ci
    lib.fbp_get_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float)]
    lib.fbp_get_kernel_ms.restype = ci
    _lib = lib
    return lib


def _check(lib, plan, status: int):
    if status != FBP_OK:
        msg = lib.fbp_last_error(plan)
        raise FbpError(status, msg.decode() if msg else "")


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array or a raw integer address."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    return x.ctypes.data


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


# ---- the C entry points, same names, same order of arguments -------------------------

def _angle_array(n_angles, angles_rad):
    """K doubles for the C side, which reads exactly n_angles of them: a shorter list must not get through."""
    if angles_rad is None:
        return None
    vals = [float(a) for a in angles_rad]
    if len(vals) != int(n_angles):
        raise ValueError("angles_rad has %d values, n_angles is %d" % (len(vals), int(n_angles)))
    return (ctypes.c_double * max(len(vals), 1))(*vals)


def fbp_create(n_angles, n_det, angles_rad, det_spacing, image_n, pixel_size, dtype, max_batch=1, device=-1):
    """fbp_create of include/fbp.h; returns the opaque plan handle (an int address)."""
    lib = load_library()
    arr = _angle_array(n_angles, angles_rad)
    plan = ctypes.c_void_p()
    st = lib.fbp_create(ctypes.byref(plan), int(n_angles), int(n_det), arr, float(det_spacing), int(image_n),
                        float(pixel_size), int(dtype), int(max_batch), int(device))
    _check(lib, None, st)
    return plan.value


def fbp_create_tuned(n_angles, n_det, angles_rad, det_spacing, image_n, pixel_size, dtype, max_batch=1, device=-1,
                     options=None):
    """fbp_create_tuned of include/fbp.h; `options` maps option names (OPTIONS) or integer keys to ints."""
    lib = load_library()
    arr = _angle_array(n_angles, angles_rad)
    flat = []
    for k, v in (options or {}).items():
        flat += [int(OPTIONS.get(k, k)), int(v)]
    opts = (ctypes.c_int * max(len(flat), 1))(*flat)
    plan = ctypes.c_void_p()
    st = lib.fbp_create_tuned(ctypes.byref(plan), int(n_angles), int(n_det), arr, float(det_spacing), int(image_n),
                              float(pixel_size), int(dtype), int(max_batch), int(device), opts, len(flat) // 2)
    _check(lib, None, st)
    return plan.value


def fbp_filter(plan, d_sino, d_filtered, batch, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_filter(plan, _ptr(d_sino), _ptr(d_filtered), int(batch), _stream_handle(stream)))


def fbp_backproject(plan, d_filtered, d_image, batch, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_backproject(plan, _ptr(d_filtered), _ptr(d_image), int(batch), _stream_handle(stream)))


def fbp_reconstruct(plan, d_sino, d_image, batch, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_reconstruct(plan, _ptr(d_sino), _ptr(d_image), int(batch), _stream_handle(stream)))


def fbp_reconstruct_host(plan, h_sino, h_image, batch, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_reconstruct_host(plan, _ptr(h_sino), _ptr(h_image), int(batch), _stream_handle(stream)))


def fbp_destroy(plan):
    if plan:
        load_library().fbp_destroy(plan)


def fbp_last_error(plan=None) -> str:
    msg = load_library().fbp_last_error(plan)
    return msg.decode() if msg else ""


def fbp_plan_info(plan) -> dict:
    lib = load_library()
    n = len(PLAN_INFO_FIELDS)
    buf = (ctypes.c_int * n)()
    got = lib.fbp_plan_info(plan, buf, n)
    return {PLAN_INFO_FIELDS[i]: int(buf[i]) for i in range(min(n, got))}


def fbp_set_trace(plan, d_marks, capacity=0):
    lib = load_library()
    _check(lib, plan, lib.fbp_set_trace(plan, _ptr(d_marks), int(capacity)))


def fbp_set_profiling(plan, enable: bool):
    lib = load_library()
    _check(lib, plan, lib.fbp_set_profiling(plan, 1 if enable else 0))


def fbp_get_kernel_ms(plan):
    lib = load_library()
    f, b = ctypes.c_float(), ctypes.c_float()
    _check(lib, plan, lib.fbp_get_kernel_ms(plan, ctypes.byref(f), ctypes.byref(b)))
    return f.value, b.value


def fbp_metrics(plan, d_x, d_y, n, max_val, c1, c2, d_out8, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_metrics(plan, _ptr(d_x), _ptr(d_y), int(n), float(max_val), float(c1), float(c2),
                                      _ptr(d_out8), _stream_handle(stream)))


METRICS_STATIC_MAX_N = 1 << 31   # FBP_METRICS_STATIC_MAX_N of include/fbp.h


def fbp_metrics_static(dtype, d_x, d_y, n, max_val, c1, c2, d_out8, stream=None):
    """fbp_metrics_static of include/fbp.h: PSNR / SSIM of two device arrays with no plan and no device allocation.

    For programs that cannot let this library call cudaMalloc (all device memory already owned by their own pool,
    a latency-bound loop, a fixed memory budget): the kernel's work area is a fixed 73 984-byte array inside
    libfbp.so instead of plan-owned memory.  The caller passes every buffer, `d_out8` (8 doubles on the device)
    included, so this wrapper allocates nothing either.  `dtype` is FBP_F32 or FBP_F64; the current CUDA device
    must be the one the arrays live on.  n > METRICS_STATIC_MAX_N raises FbpError(FBP_EINVAL).  Calls share the
    work area: keep them on one stream (or order them with events), and make the first call on each device
    during start-up, before any stream capture."""
    lib = load_library()
    _check(lib, None, lib.fbp_metrics_static(int(dtype), _ptr(d_x), _ptr(d_y), int(n), float(max_val), float(c1),
                                             float(c2), _ptr(d_out8), _stream_handle(stream)))


def fbp_measure_issue_rate(dtype) -> float:
    """Measured FFMA / DFMA lane-instructions per second of the current device (include/fbp.h)."""
    lib = load_library()
    out = ctypes.c_double()
    _check(lib, None, lib.fbp_measure_issue_rate(int(dtype), ctypes.byref(out)))
    return out.value


WINDOWS = {"ramlak": 0, "shepp-logan": 1, "cosine": 2, "hamming": 3, "hann": 4}


def fbp_set_window(plan, window):
    lib = load_library()
    _check(lib, plan, lib.fbp_set_window(plan, int(WINDOWS.get(window, window))))


def fbp_set_angle_weights(plan, weights, n_angles=None):
    """`n_angles` = the plan's K: the C side reads exactly K doubles, so the length is checked here."""
    lib = load_library()
    if weights is None:
        arr = None
    else:
        vals = [float(w) for w in weights]
        if n_angles is None:
            raise ValueError("n_angles (the plan's K) is required with a weight list")
        if len(vals) != int(n_angles):
            raise ValueError("expected %d weights, got %d" % (int(n_angles), len(vals)))
        arr = (ctypes.c_double * max(len(vals), 1))(*vals)
    _check(lib, plan, lib.fbp_set_angle_weights(plan, arr))


def fbp_interpolate_stack(plan, d_stack, n_in, d_out, n_out, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_interpolate_stack(plan, _ptr(d_stack), int(n_in), _ptr(d_out), int(n_out),
                                                _stream_handle(stream)))


def fbp_project(plan, d_image, d_sino, batch, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_project(plan, _ptr(d_image), _ptr(d_sino), int(batch), _stream_handle(stream)))


def fbp_fdk_reconstruct(plan, d_proj, d_volume, n_rows, row_spacing, sad, n_z, voxel_z, stream=None):
    lib = load_library()
    _check(lib, plan, lib.fbp_fdk_reconstruct(plan, _ptr(d_proj), _ptr(d_volume), int(n_rows), float(row_spacing), float(sad),
                                              int(n_z), float(voxel_z), _stream_handle(stream)))
