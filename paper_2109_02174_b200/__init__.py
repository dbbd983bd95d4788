"""B200-native parallel-beam filtered back-projection (arxiv 2109.02174 hot path).

The product is ``libfbp.so`` (C ABI in ``include/fbp.h``, kernels in ``csrc/``); this
package is its ctypes binding plus the seeded input generators (``inputs``).  Nothing
here computes any step of the method on the CPU and nothing imports ``oracle/``.
"""
from __future__ import annotations

from .binding import (  # noqa: F401
    EXPORTS, FBP_F32, FBP_F64, FBP_OK, FBP_EINVAL, FBP_ENOMEM, FBP_ECUDA, FBP_EUNSUPPORTED,
    FbpError, load_library,
    fbp_create, fbp_create_tuned, OPTIONS, fbp_filter, fbp_backproject, fbp_reconstruct, fbp_reconstruct_host,
    fbp_destroy, fbp_last_error, fbp_plan_info, fbp_set_profiling, fbp_get_kernel_ms, fbp_set_trace, fbp_metrics, fbp_set_window, fbp_set_angle_weights, WINDOWS, fbp_interpolate_stack, fbp_project, fbp_fdk_reconstruct,
    fbp_metrics_static, METRICS_STATIC_MAX_N, fbp_measure_issue_rate,
)
from .build import build  # noqa: F401

_DTYPES = {"f32": FBP_F32, "f64": FBP_F64, "float32": FBP_F32, "float64": FBP_F64}


def shard_slices(n_slices: int, rank: int, world_size: int) -> range:
    """Slices [lo, hi) of a stack owned by ``rank``: contiguous, balanced, no overlap.

    Slices are independent problems (a volume is a stack of 2-D slices), so
    multi-GPU runs shard them with no data-path collective (option 1)."""
    if world_size < 1 or not 0 <= rank < world_size:
        raise ValueError("bad rank/world_size")
    base, rem = divmod(n_slices, world_size)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


class Plan:
    """RAII wrapper over an ``fbp_plan*`` taking torch CUDA tensors (marshalling only)."""

    def __init__(self, angles_rad, n_det, image_n, det_spacing=1.0, pixel_size=0.0, dtype="f32",
                 max_batch=1, device=-1, options=None):
        import torch
        self.torch_dtype = torch.float32 if _DTYPES[dtype] == FBP_F32 else torch.float64
        self.n_angles, self.n_det, self.image_n, self.max_batch = len(angles_rad), int(n_det), int(image_n), int(max_batch)
        self.device = torch.device("cuda", torch.cuda.current_device() if device < 0 else device)
        # pixel size as the C side resolves it (fbp_create: pixel_size <= 0 means "= det_spacing")
        self.pixel_size = float(pixel_size) if pixel_size > 0 else float(det_spacing)
        if options:
            self.handle = fbp_create_tuned(self.n_angles, n_det, angles_rad, det_spacing, image_n, pixel_size,
                                           _DTYPES[dtype], max_batch, device, options)
        else:
            self.handle = fbp_create(self.n_angles, n_det, angles_rad, det_spacing, image_n, pixel_size,
                                     _DTYPES[dtype], max_batch, device)

    def info(self) -> dict:
        return fbp_plan_info(self.handle)

    def _batch(self, t, inner):
        if t.dtype != self.torch_dtype or not t.is_cuda or not t.is_contiguous():
            raise ValueError("expected a contiguous CUDA tensor of the plan dtype")
        if tuple(t.shape[-2:]) != inner or t.dim() not in (2, 3):
            raise ValueError("expected shape [batch]%s, got %s" % (list(inner), list(t.shape)))
        return 1 if t.dim() == 2 else t.shape[0]

    def _empty(self, like, inner):
        import torch
        shape = inner if like.dim() == 2 else (like.shape[0],) + inner
        return torch.empty(shape, dtype=self.torch_dtype, device=like.device)

    def _out(self, out, like, inner):
        """A caller-supplied result tensor goes to the library as a bare pointer: check it first."""
        if out is None:
            return self._empty(like, inner)
        want = inner if like.dim() == 2 else (like.shape[0],) + inner
        if (out.dtype != self.torch_dtype or not out.is_cuda or not out.is_contiguous() or out.device != like.device
                or tuple(out.shape) != tuple(want)):
            raise ValueError("out must be a contiguous CUDA tensor of the plan dtype, shape %s, on %s" % (list(want), like.device))
        return out

    def filter(self, sino, out=None, stream=None):
        b = self._batch(sino, (self.n_angles, self.n_det))
        out = self._out(out, sino, (self.n_angles, self.n_det))
        fbp_filter(self.handle, sino, out, b, stream)
        return out

    def backproject(self, filtered, out=None, stream=None):
        b = self._batch(filtered, (self.n_angles, self.n_det))
        out = self._out(out, filtered, (self.image_n, self.image_n))
        fbp_backproject(self.handle, filtered, out, b, stream)
        return out

    def reconstruct(self, sino, out=None, stream=None):
        b = self._batch(sino, (self.n_angles, self.n_det))
        out = self._out(out, sino, (self.image_n, self.image_n))
        fbp_reconstruct(self.handle, sino, out, b, stream)
        return out

    def project(self, image, out=None, stream=None):
        """Matched forward projector R = B^T (unweighted): image [batch][N][N] -> sinogram [batch][K][D]."""
        b = self._batch(image, (self.image_n, self.image_n))
        out = self._out(out, image, (self.n_angles, self.n_det))
        fbp_project(self.handle, image, out, b, stream)
        return out

    def interpolate_stack(self, stack, n_out, out=None, stream=None):
        """Linear interpolation of a slice stack [n_in][N][N] to n_out slices along the stack axis."""
        import torch
        if stack.dtype != self.torch_dtype or not stack.is_cuda or not stack.is_contiguous() or stack.dim() != 3 \
                or tuple(stack.shape[1:]) != (self.image_n, self.image_n):
            raise ValueError("expected a contiguous CUDA stack [n_in][N][N] of the plan dtype")
        if out is None:
            out = torch.empty((int(n_out), self.image_n, self.image_n), dtype=self.torch_dtype, device=stack.device)
        elif (out.dtype != self.torch_dtype or not out.is_cuda or not out.is_contiguous() or out.device != stack.device
              or tuple(out.shape) != (int(n_out), self.image_n, self.image_n)):
            raise ValueError("out must be a contiguous CUDA tensor [n_out][N][N] of the plan dtype")
        fbp_interpolate_stack(self.handle, stack, stack.shape[0], out, n_out, stream)
        return out

    def fdk_reconstruct(self, proj, sad, n_z, row_spacing=1.0, voxel_z=None, out=None, stream=None):
        """Cone-beam FDK: projections [K][n_rows][n_det] -> volume [n_z][N][N] (include/fbp.h, fbp_fdk_reconstruct).
        voxel_z=None means isotropic voxels: the plan's pixel size (not the detector's row spacing)."""
        import torch
        if (proj.dtype != self.torch_dtype or not proj.is_cuda or not proj.is_contiguous() or proj.dim() != 3
                or proj.shape[0] != self.n_angles or proj.shape[2] != self.n_det):
            raise ValueError("expected a contiguous CUDA tensor [K][n_rows][n_det] of the plan dtype")
        shape = (int(n_z), self.image_n, self.image_n)
        if out is None:
            out = torch.empty(shape, dtype=self.torch_dtype, device=proj.device)
        elif (out.dtype != self.torch_dtype or not out.is_cuda or not out.is_contiguous() or tuple(out.shape) != shape
              or out.device != proj.device):
            raise ValueError("out must be a contiguous CUDA tensor [n_z][N][N] of the plan dtype")
        fbp_fdk_reconstruct(self.handle, proj, out, proj.shape[1], row_spacing, sad, n_z,
                            self.pixel_size if voxel_z is None else voxel_z, stream)
        return out

    def set_window(self, window):
        fbp_set_window(self.handle, window)

    def set_angle_weights(self, weights):
        if weights is not None and len(weights) != self.n_angles:
            raise ValueError("expected one weight per angle")
        fbp_set_angle_weights(self.handle, weights, self.n_angles)

    def metrics(self, x, y, max_val, c1=-1.0, c2=-1.0, stream=None) -> dict:
        """PSNR / SSIM (eq. 3, 4 of the paper) of two CUDA tensors of the plan dtype; one device-to-host read."""
        import torch
        if x.dtype != self.torch_dtype or y.dtype != self.torch_dtype or x.shape != y.shape:
            raise ValueError("expected two tensors of the plan dtype and the same shape")
        if not (x.is_cuda and y.is_cuda and x.is_contiguous() and y.is_contiguous()):
            raise ValueError("expected contiguous CUDA tensors")
        out = torch.empty(8, dtype=torch.float64, device=x.device)
        fbp_metrics(self.handle, x, y, x.numel(), max_val, c1, c2, out, stream)
        vals = out.cpu().tolist()
        return dict(zip(("mse", "psnr", "ssim", "mu_x", "mu_y", "var_x", "var_y", "cov_xy"), vals))

    def close(self):
        if getattr(self, "handle", None):
            fbp_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
