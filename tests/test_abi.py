"""CPU-side checks of the boundary: libfbp.so builds, loads and exports every symbol that
include/fbp.h declares; argument validation that happens before any CUDA call; host logic."""
import ctypes
import os
import re

import pytest

import paper_2109_02174_b200 as pkg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    pkg.build()
    return pkg.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "fbp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fbp_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = _declared_symbols()
    assert set(names) == set(pkg.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    ang = (ctypes.c_double * 4)(0.0, 0.5, 1.0, 1.5)
    nan = (ctypes.c_double * 4)(0.0, float("nan"), 1.0, 1.5)
    plan = ctypes.c_void_p(123)
    cases = [
        (4, 8, None, 1.0, 8, 1.0, 0, 1),      # NULL angles
        (0, 8, ang, 1.0, 8, 1.0, 0, 1),       # n_angles < 1
        (4, 1, ang, 1.0, 8, 1.0, 0, 1),       # n_det < 2
        (4, 8, ang, 0.0, 8, 1.0, 0, 1),       # d <= 0
        (4, 8, ang, float("inf"), 8, 1.0, 0, 1),
        (4, 8, ang, 1.0, 0, 1.0, 0, 1),       # image_n < 1
        (4, 8, ang, 1.0, 8, float("nan"), 0, 1),
        (4, 8, ang, 1.0, 8, 1.0, 7, 1),       # unknown dtype
        (4, 8, ang, 1.0, 8, 1.0, 0, 0),       # max_batch < 1
        (4, 8, nan, 1.0, 8, 1.0, 0, 1),       # non-finite angle
    ]
    for k, d, a, sp, n, px, dt, mb in cases:
        plan.value = 123
        st = lib.fbp_create(ctypes.byref(plan), k, d, a, sp, n, px, dt, mb, -1)
        assert st == pkg.FBP_EINVAL, (k, d, sp, n, px, dt, mb)
        assert plan.value is None
        assert pkg.fbp_last_error(None) != ""
    assert lib.fbp_create(None, 4, 8, ang, 1.0, 8, 1.0, 0, 1, -1) == pkg.FBP_EINVAL


def test_create_tuned_rejects_bad_option_lists(lib):
    ang = (ctypes.c_double * 4)(0.0, 0.5, 1.0, 1.5)
    plan = ctypes.c_void_p(123)
    bad_key = (ctypes.c_int * 2)(9999, 1)
    assert lib.fbp_create_tuned(ctypes.byref(plan), 4, 8, ang, 1.0, 8, 1.0, 0, 1, -1, bad_key, 1) == pkg.FBP_EINVAL
    assert plan.value is None
    assert lib.fbp_create_tuned(ctypes.byref(plan), 4, 8, ang, 1.0, 8, 1.0, 0, 1, -1, None, 2) == pkg.FBP_EINVAL
    assert lib.fbp_create_tuned(ctypes.byref(plan), 4, 8, ang, 1.0, 8, 1.0, 0, 1, -1, bad_key, -1) == pkg.FBP_EINVAL
    # FBP_OPT_FILTER_R: a group size no kernel has, or one the dtype does not have, is refused (checked before any CUDA call)
    for dtype, r in ((0, 8), (0, -6), (1, 10), (1, 14), (1, 7)):
        opt = (ctypes.c_int * 2)(pkg.OPTIONS["filter_r"], r)
        plan.value = 123
        assert lib.fbp_create_tuned(ctypes.byref(plan), 4, 8, ang, 1.0, 8, 1.0, dtype, 1, -1, opt, 1) == pkg.FBP_EINVAL, (dtype, r)
        assert plan.value is None and "FBP_OPT_FILTER_R" in pkg.fbp_last_error(None)
    with pytest.raises(ValueError):
        pkg.fbp_create(5, 8, [0.0, 0.5, 1.0, 1.5], 1.0, 8, 0.0, pkg.FBP_F32)     # the C side would read 5 doubles
    with pytest.raises(ValueError):
        pkg.fbp_create_tuned(3, 8, [0.0, 0.5, 1.0, 1.5], 1.0, 8, 0.0, pkg.FBP_F32)


def test_library_does_not_read_the_environment():
    """Behaviour depends on the arguments only (fbp_create_tuned): no getenv in the product sources."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2109_02174_b200", "csrc")):
        for f in files:
            src = open(os.path.join(dirpath, f)).read()
            assert "getenv" not in src and "environ[" not in src and "putenv" not in src, f
    binding = open(os.path.join(ROOT, "paper_2109_02174_b200", "binding.py")).read()
    assert "environ" not in binding and "getenv" not in binding          # which .so is loaded is an argument too


def test_null_plan_is_rejected_or_ignored(lib):
    assert lib.fbp_filter(None, 16, 32, 1, None) == pkg.FBP_EINVAL
    assert lib.fbp_backproject(None, 16, 32, 1, None) == pkg.FBP_EINVAL
    assert lib.fbp_reconstruct(None, 16, 32, 1, None) == pkg.FBP_EINVAL
    assert lib.fbp_reconstruct_host(None, 16, 32, 1, None) == pkg.FBP_EINVAL
    assert lib.fbp_set_profiling(None, 1) == pkg.FBP_EINVAL
    assert lib.fbp_plan_info(None, None, 0) == 0
    lib.fbp_destroy(None)


def test_no_gpu_means_error_not_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(pkg.FbpError) as ei:
        pkg.fbp_create(4, 8, [0.0, 0.5, 1.0, 1.5], 1.0, 8, 0.0, pkg.FBP_F32)
    assert ei.value.status in (pkg.FBP_ECUDA, pkg.FBP_EUNSUPPORTED)


def test_missing_library_fails_loudly(tmp_path):
    with pytest.raises(FileNotFoundError):
        pkg.load_library(str(tmp_path / "libfbp.so"))


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2109_02174_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "fbp_oracle" not in src, f


def test_shard_slices_partitions_exactly():
    for n in (0, 1, 7, 64, 65):
        for w in (1, 2, 3, 8):
            parts = [pkg.shard_slices(n, r, w) for r in range(w)]
            flat = [i for p in parts for i in p]
            assert flat == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        pkg.shard_slices(4, 2, 2)
