"""Writes tests/golden/oracle_cfg1.json: expected values computed by the ORACLE only.

    python tests/golden/make_golden.py

Calls `oracle/` and the seeded input generators, nothing else (never the CUDA path).  The
stored values let a test catch an unintended change of the oracle's arithmetic or of the
input recipe (the SHA-256 of the input bytes is stored beside them), and give the GPU
parity tests a fixed target that does not depend on the oracle being rebuilt.
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2109_02174_b200 import inputs as I  # noqa: E402

#: (row, column) samples of the config-1 image: corners, centre, feature interiors, edges
PIXELS = [(0, 0), (0, 63), (63, 0), (63, 63), (31, 31), (32, 32), (31, 32), (20, 40), (40, 22), (45, 31),
          (12, 32), (32, 6), (5, 50), (58, 20), (33, 47), (25, 25)]
#: (angle, bin) samples of the filtered sinogram
BINS = [(0, 0), (0, 45), (0, 90), (17, 30), (44, 45), (45, 46), (89, 12), (60, 77)]


def main():
    cfg = I.CONFIGS[1]
    ang = I.config_angles(1)
    sino32 = I.config_sinogram(1).astype(np.float32)          # the bytes the fp32 tests feed both sides
    sino = sino32.astype(np.float64)
    q = oracle.filter_sinogram(sino)
    f = oracle.reconstruct(sino, ang, cfg.image_n)
    out = {
        "_about": "written by tests/golden/make_golden.py from oracle/ only; cfg1 = 64x64, 90 angles, 91 bins, HEAD10 "
                  "(SURVEY.md 8(d)); input = analytic sinogram rounded to fp32; eq. 2 PAPER.md:59, filter PAPER.md:61",
        "input_sha256_f32": I.sha256(sino32),
        "image_min": float(f.min()), "image_max": float(f.max()),
        "image_samples": [[r, c, float(f[0, r, c])] for r, c in PIXELS],
        "filtered_samples": [[i, n, float(q[0, i, n])] for i, n in BINS],
    }
    with open(os.path.join(HERE, "oracle_cfg1.json"), "w") as fh:
        json.dump(out, fh, indent=1)
        fh.write("\n")


if __name__ == "__main__":
    main()
