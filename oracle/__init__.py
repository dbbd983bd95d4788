"""ORACLE (test infrastructure, not the product): plain CPU fp64 filtered back-projection.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA
package ``paper_2109_02174_b200`` and the CUDA package imports nothing from here.
See ``fbp_oracle.c`` for the algorithm, its citations and its pins.
"""
from .oracle import (  # noqa: F401
    build,
    max_threads,
    taps,
    filter_sinogram,
    filter_rows,
    backproject,
    backproject_pixels,
    forward_scatter,
    reconstruct,
    WINDOWS,
    window_taps,
    filter_sinogram_window,
    backproject_weighted,
    metrics,
    interpolate_stack,
    fdk_weight,
    fdk_backproject,
    fdk_reconstruct,
)
