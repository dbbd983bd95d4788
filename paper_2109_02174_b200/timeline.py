"""In-kernel timeline of one fbp_reconstruct: where the microseconds of a step go.

    python -m paper_2109_02174_b200.timeline [--config 3] [--dtype f32] [--reps 20] [--opt KEY=INT ...]

Uses the library's own trace hook (fbp_set_trace, include/fbp.h): thread 0 of every CTA of the filter and
of the back-projector stores %globaltimer at fixed points of the PRODUCT kernels (no instrumented build).
Each repetition flushes L2, reconstructs once and reads the marks back; the table is the median over
repetitions of per-CTA statistics, in microseconds after the first filter CTA started.  No arithmetic of
the method happens here.  The summaries under profiles/ (r2*_timeline_*.txt) are this tool's output.
"""
from __future__ import annotations

import argparse

import numpy as np

# slot names of include/fbp.h (fbp_set_trace), per filter kind (plan_info "filter_kind": 1 direct form, 2 FFT form)
FILTER_SLOTS = {
    1: ("start", "tables+row staged", "partial sums done", "row reduced", "last unit stored"),
    2: ("start", "rows read, 1st pass", "spectrum ready", "rows back in smem", "last row pair stored"),
}
BP_SLOTS = ("CTA resident", "past grid dependency", "first chunk landed", "main loop done", "pixels stored")


def main() -> int:
    import torch

    import paper_2109_02174_b200 as fbp
    from paper_2109_02174_b200 import inputs as I

    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=INT")
    ap.add_argument("--l2", default="flush", choices=["flush", "rotate", "warm"],
                    help="flush: 256 MiB memset before every repetition (everything cold, code and tables included); "
                         "rotate: every repetition reads another of 192 sinogram copies (> L2: inputs cold, code and tables warm); "
                         "warm: same buffers every time")
    ap.add_argument("--dump", default=None, metavar="FILE.npy", help="also save the raw marks [CTA][8] (ns) of the last repetition")
    args = ap.parse_args()
    cfg = I.CONFIGS[args.config]
    tdt = torch.float32 if args.dtype == "f32" else torch.float64
    B = min(cfg.batch, 7)                       # the batch pipeline's side streams are not traced
    sino = torch.from_numpy(np.stack([I.config_slice(args.config, s) for s in range(B)])).to(tdt).cuda()
    img = torch.empty((B, cfg.image_n, cfg.image_n), dtype=tdt, device="cuda")
    options = {kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.opt}
    plan = fbp.Plan(list(I.config_angles(args.config)), cfg.n_det, cfg.image_n, dtype=args.dtype, max_batch=B, options=options)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda") if args.l2 == "flush" else None
    n_pool = 192 if args.l2 == "rotate" else 1
    pool = [sino] + [sino.clone() for _ in range(n_pool - 1)]
    imgs = [img] + [torch.empty_like(img) for _ in range(n_pool - 1)]
    stream = torch.cuda.current_stream()
    for i in range(3):
        fbp.fbp_reconstruct(plan.handle, pool[i % n_pool], imgs[i % n_pool], B, stream)
    torch.cuda.synchronize()
    info = plan.info()
    n_f, n_b = info["filter_ctas"], info["bp_ctas_per_slice"] * B
    marks = torch.zeros(8 * (n_f + n_b), dtype=torch.int64, device="cuda")
    fbp.fbp_set_trace(plan.handle, marks, marks.numel())
    rows = []
    for rep in range(args.reps):
        if flush is not None:
            flush.zero_()
        marks.zero_()
        fbp.fbp_reconstruct(plan.handle, pool[(rep + 3) % n_pool], imgs[(rep + 3) % n_pool], B, stream)
        torch.cuda.synchronize()
        m = marks.cpu().numpy().reshape(-1, 8).astype(np.float64)
        t0 = m[:n_f, 0].min()
        f, b = (m[:n_f, :5] - t0) * 1e-3, (m[n_f:, :5] - t0) * 1e-3
        rows.append(np.concatenate([np.stack([f.min(0), np.median(f, 0), f.max(0)]).T.ravel(),
                                    np.stack([b.min(0), np.median(b, 0), b.max(0)]).T.ravel()]))
    fbp.fbp_set_trace(plan.handle, None, 0)
    plan.close()
    if args.dump:
        np.save(args.dump, m)
    med = np.median(np.array(rows), axis=0)
    print("config %d %s, batch %d, options %s: %d filter CTAs x %d threads (%d units/row), %d back-projection CTAs x %d threads"
          % (args.config, args.dtype, B, options, n_f, info["filter_threads"], info["filter_units_per_row"], n_b, info["bp_threads"]))
    print("microseconds after the first filter CTA started (median over %d repetitions, L2 mode '%s', of min / median / max over CTAs)" % (args.reps, args.l2))
    k = 0
    for kern, slots in (("filter", FILTER_SLOTS[info["filter_kind"]]), ("back-projection", BP_SLOTS)):
        for s in slots:
            print("%-16s %-22s %8.2f %8.2f %8.2f" % (kern, s, med[k], med[k + 1], med[k + 2]))
            k += 3
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
