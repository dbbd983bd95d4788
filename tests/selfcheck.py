"""Small driver for `compute-sanitizer` (memcheck / racecheck / initcheck / synccheck):

    compute-sanitizer --tool racecheck python tests/selfcheck.py

Runs every kernel family once on tiny geometries (both dtypes, angle splits on and off, the batch
pipeline, the host path) and checks that repeated runs are bit-identical.  No oracle here: parity is
the business of tests/; this only gives the sanitizer something to watch."""
from __future__ import annotations

import math
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def main() -> int:
    import numpy as np
    import torch

    import paper_2109_02174_b200 as pkg

    pkg.load_library()
    torch.cuda.set_device(0)
    cases = [  # (N, K, D, batch, options of fbp_create_tuned)
        (40, 24, 61, 1, {}),
        (33, 10, 48, 2, {"bp_splits": 3}),
        (64, 16, 91, 9, {}),                       # batch >= 8: pipelined path
        (24, 8, 40, 1, {"pdl": 0}),
        (90, 12, 500, 1, {"filter_sb": 2}),        # two filter units per row
    ]
    for n, k, d, b, env in cases:
        if True:
            ang = [i * math.pi / k for i in range(k)]
            for dt, tdt in (("f32", torch.float32), ("f64", torch.float64)):
                sino = torch.from_numpy(np.random.default_rng(n + k).standard_normal((b, k, d))).to(tdt).cuda()
                with pkg.Plan(ang, d, n, dtype=dt, max_batch=b, options=env) as plan:
                    first = plan.reconstruct(sino).clone()
                    q = plan.filter(sino)
                    two = plan.backproject(q)
                    again = plan.reconstruct(sino)
                    torch.cuda.synchronize()
                    if not (torch.equal(first, again) and torch.equal(first, two)):
                        print("MISMATCH", n, k, d, b, dt, env)
                        return 1
                    host_in = sino.cpu().pin_memory()
                    host_out = torch.empty((b, n, n), dtype=tdt).pin_memory()
                    pkg.fbp_reconstruct_host(plan.handle, host_in, host_out, b)
                    if not torch.equal(host_out, first.cpu()):
                        print("HOST MISMATCH", n, k, d, b, dt, env)
                        return 1
                    # the forward projector (TMA-staged gather) and the cone-beam path on the same plan
                    y1 = plan.project(first).clone()
                    y2 = plan.project(first)
                    torch.cuda.synchronize()
                    if not torch.equal(y1, y2):
                        print("PROJECT MISMATCH", n, k, d, b, dt, env)
                        return 1
                    if b == 1:
                        proj = torch.from_numpy(np.random.default_rng(7).standard_normal((k, 5, d))).to(tdt).cuda()
                        v1 = plan.fdk_reconstruct(proj, 4.0 * n, 6).clone()
                        v2 = plan.fdk_reconstruct(proj, 4.0 * n, 6)
                        torch.cuda.synchronize()
                        if not torch.equal(v1, v2):
                            print("FDK MISMATCH", n, k, d, b, dt, env)
                            return 1
    print("selfcheck ok")
    return 0


def soak(runs: int) -> int:
    """``python tests/selfcheck.py --soak N``: N reconstructions per case with other work interleaved; every 25th result and the last are
    compared bit for bit with the first (the paper's parallel versions differed on every run)."""
    import numpy as np
    import torch

    import paper_2109_02174_b200 as pkg
    from paper_2109_02174_b200 import inputs as I

    pkg.load_library()
    torch.cuda.set_device(0)
    bad = 0
    for cid, dt, batch, env in ((3, "f32", 1, {}), (3, "f64", 1, {}), (3, "f32", 1, {"bp_splits": 3}),
                                (2, "f32", 12, {}), (1, "f32", 1, {})):
        if True:
            cfg = I.CONFIGS[cid]
            tdt = torch.float32 if dt == "f32" else torch.float64
            sino = torch.from_numpy(np.stack([I.config_slice(cid, s % 3) for s in range(batch)])).to(tdt).cuda()
            with pkg.Plan(list(I.config_angles(cid)), cfg.n_det, cfg.image_n, dtype=dt, max_batch=batch, options=env) as plan:
                first = plan.reconstruct(sino).clone()
                junk = torch.randn(2048, 2048, device="cuda")
                miss = 0
                for i in range(runs):
                    if i % 7 == 0:
                        junk = (junk @ junk) * 1e-4
                    out = plan.reconstruct(sino)
                    if i % 25 == 0 or i == runs - 1:
                        miss += int(not torch.equal(out, first))
                torch.cuda.synchronize()
                if cid == 3 and not env:
                    # the forward projector: mbarrier ring fed by a producer warp, consumers in four warps
                    y0 = plan.project(first).clone()
                    pmiss = 0
                    for i in range(runs):
                        if i % 7 == 0:
                            junk = (junk @ junk) * 1e-4
                        y = plan.project(first)
                        if i % 25 == 0 or i == runs - 1:
                            pmiss += int(not torch.equal(y, y0))
                    torch.cuda.synchronize()
                    print("cfg%d %s forward projector: %d runs, %d mismatches" % (cid, dt, runs, pmiss))
                    bad += pmiss
            print("cfg%d %s batch %d %s: %d runs, %d mismatches" % (cid, dt, batch, env, runs, miss))
            bad += miss
    return 1 if bad else 0


if __name__ == "__main__":
    if len(sys.argv) > 2 and sys.argv[1] == "--soak":
        sys.exit(soak(int(sys.argv[2])))
    sys.exit(main())
