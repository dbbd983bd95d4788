"""Micro-benchmark of the back-projector's inner loop: build and run csrc/ubench_bp_inner.cu.

    python -m paper_2109_02174_b200.ubench [--ctas-per-sm 4] [--sass]

A stand-alone CUDA program (not part of libfbp, no method arithmetic here): it times the operand schemes
DESIGN.md 6.2 compares -- the (mid, slope) entry, near/far end points, and the column walk -- on a B200 SM with
everything resident in shared memory.  --sass also prints the per-variant SASS instruction histogram (cuobjdump),
from which the issue slots per pixel pair quoted in DESIGN.md are counted.  Output: profiles/r2b_ubench_bp_inner.txt.
"""
from __future__ import annotations

import argparse
import collections
import os
import re
import subprocess
import sys

from .build import CSRC, NVCC_FLAGS, _nvcc

_HERE = os.path.dirname(os.path.abspath(__file__))


def build(ctas_per_sm: int) -> str:
    exe = os.path.join(_HERE, "ubench_bp_inner")
    flags = [f for f in NVCC_FLAGS if f not in ("-shared", "-Xcompiler", "-fPIC")]
    subprocess.run([_nvcc()] + flags + ["-DNB=%d" % ctas_per_sm, "-o", exe, os.path.join(CSRC, "ubench_bp_inner.cu")], check=True)
    return exe


def sass_histogram(exe: str) -> None:
    cuobjdump = os.path.join(os.path.dirname(_nvcc()), "cuobjdump") if os.path.sep in _nvcc() else "cuobjdump"
    text = subprocess.run([cuobjdump, "-sass", exe], check=True, capture_output=True, text=True).stdout
    fn, hist = None, collections.defaultdict(collections.Counter)
    for line in text.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+(?:\.(?:64|128|RM))?)", line)
        if m and fn:
            hist[fn][m.group(1)] += 1
    for fn in sorted(hist):
        print("%s: %d instructions (3 copies of the %s-pair loop body + prologue)" % (fn, sum(hist[fn].values()), "R"))
        print("   " + ", ".join("%s %d" % kv for kv in hist[fn].most_common(16)))


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--ctas-per-sm", type=int, default=4)
    ap.add_argument("--sass", action="store_true")
    args = ap.parse_args()
    exe = build(args.ctas_per_sm)
    if args.sass:
        sass_histogram(exe)
    return subprocess.run([exe]).returncode


if __name__ == "__main__":
    sys.exit(main())
