"""bench.py -- one JSON line for the FBP hot path (filter + back-projection) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--dtype f32] [--impl ours|reference]

A "step" is one fbp_reconstruct (row filter, then back-projection: all rows of SURVEY.md
8(a)) of one batch of the chosen BASELINE.json configuration; the default is config 3
(512x512 image, 360 angles, 725 bins), the one BASELINE.json's metric is quoted on.  The
metric is quoted "fp32/fp64": the headline line is fp32 and carries an "f64" sub-record with
the same measurements in double precision (configs 3 and 5, the ones BASELINE.json lists
in both precisions; `--dtype f64` makes fp64 the headline instead).
`value` = back-projection updates (batch * N^2 * K) per second of WHOLE-STEP time, in
Gupdates/s, inputs resident in HBM, L2 flushed between steps (outside the timed events).
With --gpus N > 1 the script starts N ranks itself (torch.distributed.run, one per GPU,
127.0.0.1); under torchrun each rank reconstructs its own slices (weak scaling, no
collective: slices are independent problems).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2109_02174_b200 import inputs as I  # noqa: E402

METRIC = "backprojection_gupdates_per_s"
UNIT = "Gupdates/s"
FP_INSTR_PER_UPDATE = 7          # coordinate 2, floor 1, fraction 1, lerp 2, accumulate 1
FP32_LANES, FP64_LANES = 128, 64
BOTH_DTYPES = (3, 5)             # BASELINE.json configs listed "fp32 and fp64"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=3, choices=sorted(I.CONFIGS))
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-f64", action="store_true", help="skip the fp64 sub-record of a default (fp32) run")
    ap.add_argument("--window", default="ramlak", choices=["ramlak", "shepp-logan", "cosine", "hamming", "hann"],
                    help="reconstruction filter (SURVEY.md 8(f) row 1); the headline is ramlak")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=INT",
                    help="launch-configuration override passed to fbp_create_tuned (A/B runs), e.g. --opt filter_kind=1")
    ap.add_argument("--graph", action="store_true",
                    help="also time the step replayed as ONE CUDA graph (the two launches with their programmatic edge captured once)")
    ap.add_argument("--lib", default=None, metavar="PATH",
                    help="load this build of libfbp.so instead of the in-tree one (A/B of two builds; recorded in launch.lib)")
    ap.add_argument("--extras", action="store_true", help="also time fbp_metrics, fbp_interpolate_stack and fbp_project")
    return ap.parse_args()


def workload(cfg_id):
    """The `config` object: identical in both arms (it names the workload, nothing else)."""
    cfg = I.CONFIGS[cfg_id]
    return {"workload": "cfg%d: %dx%d image, %d angles in [0,pi), %d bins, batch %d" % (
        cfg_id, cfg.image_n, cfg.image_n, cfg.n_angles, cfg.n_det, cfg.batch),
        "image_n": cfg.image_n, "n_angles": cfg.n_angles, "n_det": cfg.n_det, "batch_per_gpu": cfg.batch,
        "input": cfg.description}


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def ncu_traffic(cfg_id, dtype, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the tracked table of
    `ncu --set full` captures (profiles/dram_traffic.csv; its .md names the commands); None if there is none."""
    try:
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if int(row["config"]) == cfg_id and row["dtype"] == dtype and row["kernel"] == kernel:
                    return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------
# clocks: sampled with NVML in a thread while the timed region runs
# ---------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False
        self.t = threading.Thread(target=self._run, daemon=True)

    def _once(self):
        nv = self.nv
        self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        for bit, name in self.REASONS.items():
            if mask & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            self._stop.wait(0.001)

    def __enter__(self):
        if self.ok:
            self.t.start()
        return self

    def __exit__(self, *exc):
        if self.ok:
            try:
                self._once()
            except Exception:
                pass
            self._stop.set()
            self.t.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": float(self.max_mhz),
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------
# the oracle leg: cpu_baseline of our line and the whole of `--impl reference`
# ---------------------------------------------------------------------------------------
_SLICE0 = {}


def _slice0(cfg_id):
    if cfg_id not in _SLICE0:
        _SLICE0[cfg_id] = I.config_slice(cfg_id, 0)
    return _SLICE0[cfg_id]


def time_oracle(cfg_id, frac=1.0, reps=1, threads=0):
    """The CPU fp64 oracle, as it stands, on `threads` host threads (0 = all cores), on a bounded sample of
    slice 0 of the workload: a fraction `frac` of the filter rows and of the pixels (all of them when
    frac >= 1), each timing scaled to the full slice.  Returns (best Gupdates/s, threads used, sample
    description, best seconds per full slice, list of Gupdates/s of every repetition)."""
    import oracle

    cfg = I.CONFIGS[cfg_id]
    ang = I.config_angles(cfg_id)
    sino = _slice0(cfg_id)
    cores = oracle.max_threads() if threads <= 0 else min(threads, oracle.max_threads())
    n, k = cfg.image_n, cfg.n_angles
    updates = n * n * k
    times = []
    if frac >= 1.0:
        for _ in range(reps):
            t0 = time.perf_counter()
            oracle.reconstruct(sino, ang, n, threads=cores)
            times.append(time.perf_counter() - t0)
        sample = "slice 0 of cfg%d in full (filter + back-projection)" % cfg_id
    else:
        rows = np.unique(np.linspace(0, k - 1, num=max(1, int(frac * k)), dtype=np.int32))
        npix = max(64, int(frac * n * n))
        rng = np.random.default_rng(0)
        rr = rng.integers(0, n, npix).astype(np.int32)
        cc = rng.integers(0, n, npix).astype(np.int32)
        for _ in range(reps):
            t0 = time.perf_counter()
            oracle.filter_rows(sino, rows, threads=cores)
            t_f = (time.perf_counter() - t0) * k / len(rows)
            t0 = time.perf_counter()
            oracle.backproject_pixels(sino, ang, n, rr, cc, threads=cores)
            t_b = (time.perf_counter() - t0) * (n * n) / npix
            times.append(t_f + t_b)
        sample = ("slice 0 of cfg%d: %d of %d filter rows and %d of %d pixels, each timing scaled to the full slice"
                  % (cfg_id, len(rows), k, npix, n * n))
    best = min(times)
    return updates / best / 1e9, cores, sample, best, [updates / t / 1e9 for t in times]


def oracle_fraction(cfg_id, budget_s, n_steps, threads=0):
    """Fraction of a slice per step so that n_steps oracle steps take about budget_s seconds."""
    cfg = I.CONFIGS[cfg_id]
    probe = min(1.0, 2e7 / (cfg.image_n * cfg.image_n * cfg.n_angles)) * (0.1 if threads == 1 else 1.0)
    _, _, _, t_full, _ = time_oracle(cfg_id, probe, threads=threads)
    return min(1.0, budget_s / (max(n_steps, 1) * t_full))


def cpu_baseline(cfg_id):
    """The oracle on the box's host cores, best of 5 with the spread, at 1 thread (the paper's "sequential CPU",
    PAPER.md:79, 109) and at all cores (its "CPU threads").  The thread count is passed to the oracle explicitly
    (OpenMP num_threads), not left to the environment."""
    legs = {}
    for name, thr in (("threads_1", 1), ("all_cores", 0)):
        frac = oracle_fraction(cfg_id, 10.0, 5, thr)
        g, cores, sample, _, all_g = time_oracle(cfg_id, frac, reps=5, threads=thr)
        legs[name] = {"value": g, "unit": UNIT, "cores": cores, "best_of": 5, "min": min(all_g), "max": max(all_g),
                      "sample": sample}
    top = legs["all_cores"]
    return {"value": top["value"], "unit": UNIT, "cores": top["cores"], "kind": "oracle",
            "sample": top["sample"] + "; best of 5 (spread in all_cores)", "threads_1": legs["threads_1"],
            "all_cores": legs["all_cores"]}


def run_reference(args):
    """--impl reference: the paper ships no code, so this arm times the CPU oracle, as it stands,
    on the same config and metric; every step is a bounded sample of the workload.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = I.CONFIGS[args.config]
    frac = oracle_fraction(args.config, 120.0, args.steps + args.warmup)
    for _ in range(args.warmup):
        time_oracle(args.config, frac)
    vals = [time_oracle(args.config, frac) for _ in range(args.steps)]
    g = float(np.mean([v[0] for v in vals]))
    sec = float(np.mean([v[3] for v in vals]))
    cores, sample = vals[0][1], vals[0][2]
    line = {"impl": "reference", "metric": METRIC, "value": g, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3 * cfg.batch,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload(args.config),
            "cpu_baseline": {"value": g, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": g, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------
def measure(args, dtype, world, rank, local, dist):
    """All measurements of one dtype on this rank: whole step (CUDA events, L2 flushed), per-kernel times,
    end to end through the host entry point.  Returns a dict of plain numbers (ms, bytes, info)."""
    import torch

    import paper_2109_02174_b200 as fbp

    cfg = I.CONFIGS[args.config]
    tdt = torch.float32 if dtype == "f32" else torch.float64
    npdt = np.float32 if dtype == "f32" else np.float64
    ang = I.config_angles(args.config)
    B, N, K, D = cfg.batch, cfg.image_n, cfg.n_angles, cfg.n_det
    # weak scaling: every rank owns a full batch of the config; slice s of rank r is seeded as
    # slice (r*B + s) of the recipe, so ranks do not share inputs.  Big stacks reuse 4 distinct slices.
    distinct = min(B, 4)
    base = np.stack([I.config_slice(args.config, rank * B + s) for s in range(distinct)]).astype(npdt)
    input_sha = I.sha256(base)                       # ties the result to the bytes that were reconstructed
    h_sino = torch.from_numpy(base[np.arange(B) % distinct].copy()).pin_memory()
    d_sino = h_sino.cuda()
    d_img = torch.empty((B, N, N), dtype=tdt, device="cuda")
    h_img = torch.empty((B, N, N), dtype=tdt).pin_memory()
    options = {kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.opt}
    plan = fbp.Plan(list(ang), D, N, dtype=dtype, max_batch=B, options=options)
    if args.window != "ramlak":
        plan.set_window(args.window)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_loop(fn, steps, per_step_hook=None):
        """K steps, each bracketed by its own CUDA events on the launching stream; the L2 flush
        sits between steps, outside the events.  Returns total milliseconds of the K steps."""
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        for a, b in evs:
            flush.zero_()
            a.record(stream)
            fn()
            b.record(stream)
            if per_step_hook:
                per_step_hook()
        barrier()
        return sum(a.elapsed_time(b) for a, b in evs)

    step = lambda: fbp.fbp_reconstruct(plan.handle, d_sino, d_img, B, stream)  # noqa: E731
    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    with ClockSampler(local) as clk:
        ms_total = timed_loop(step, args.steps)
    ms_step = ms_total / args.steps
    info = plan.info()

    # the same step replayed as a CUDA graph (captured once on a side stream after the warm-up above)
    graph_ms = None
    if args.graph:
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            fbp.fbp_reconstruct(plan.handle, d_sino, d_img, B, side)
            side.synchronize()
            with torch.cuda.graph(g, stream=side):
                fbp.fbp_reconstruct(plan.handle, d_sino, d_img, B, torch.cuda.current_stream())
        want = d_img.clone()
        step()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(d_img, want), "graph replay differs from the stream launch"
        graph_ms = timed_loop(g.replay, args.steps) / args.steps

    # per-kernel durations (library-side CUDA events on the same stream), separate loop
    fbp.fbp_set_profiling(plan.handle, True)
    kms = []
    timed_loop(step, min(args.steps, 50), lambda: kms.append(fbp.fbp_get_kernel_ms(plan.handle)))
    fbp.fbp_set_profiling(plan.handle, False)
    f_ms = float(np.mean([k[0] for k in kms]))
    b_ms = float(np.mean([k[1] for k in kms]))

    # end to end through the host-buffer entry point: H2D + kernels + D2H + wait, wall clock
    for _ in range(3):
        fbp.fbp_reconstruct_host(plan.handle, h_sino, h_img, B, stream)
    barrier()
    # every call is timed on its own (fbp_reconstruct_host returns after the stream has drained): the median is the
    # reported figure, min and max go beside it -- a mean hides a host that was busy for a few calls
    e2e_steps = max(3, min(args.steps, 100))
    e2e_each = []
    for _ in range(e2e_steps):
        t0 = time.perf_counter()
        fbp.fbp_reconstruct_host(plan.handle, h_sino, h_img, B, stream)
        e2e_each.append(time.perf_counter() - t0)
    barrier()
    e2e_s = float(np.median(e2e_each))
    e2e_spread = {"calls": e2e_steps, "ms_min": min(e2e_each) * 1e3, "ms_max": max(e2e_each) * 1e3, "ms_mean": float(np.mean(e2e_each)) * 1e3}

    extras = None
    if args.extras:
        # fbp_metrics on the whole output stack against a copy (HBM-bound)
        other = d_img.clone()
        out8 = torch.empty(8, dtype=torch.float64, device="cuda")
        mfn = lambda: fbp.fbp_metrics(plan.handle, d_img, other, d_img.numel(), 1.0, -1.0, -1.0, out8, stream)  # noqa: E731
        for _ in range(3):
            mfn()
        m_ms = timed_loop(mfn, 20) / 20
        m_bytes = 2.0 * d_img.numel() * d_img.element_size()        # algorithmic: each array read once
        # fbp_interpolate_stack: the output stack to 4x as many slices (reads <= 2, writes 1 array of the output size)
        n_out = 4 * B
        vol = torch.empty((n_out, N, N), dtype=tdt, device="cuda")
        ifn = lambda: fbp.fbp_interpolate_stack(plan.handle, d_img, B, vol, n_out, stream)  # noqa: E731
        for _ in range(3):
            ifn()
        i_ms = timed_loop(ifn, 20) / 20
        i_bytes = float(vol.numel() + d_img.numel()) * d_img.element_size()     # algorithmic: read the stack once, write the volume
        # fbp_project: forward projection of the output stack (the adjoint's pixel-angle pairs per second)
        pb = min(B, 8)
        d_proj = torch.empty((pb, K, D), dtype=tdt, device="cuda")
        pfn = lambda: fbp.fbp_project(plan.handle, d_img, d_proj, pb, stream)  # noqa: E731
        for _ in range(3):
            pfn()
        p_ms = timed_loop(pfn, 10) / 10
        # fbp_fdk_reconstruct: cone-beam FDK of a 64-slice volume on the config's x-y grid from n_det x 97 projections
        # (pre-weight + row filter + weighted bilinear back-projection); voxel-angle updates per second of the whole call
        # on the seeded three-ball projections that tests/test_extras_sizes_gpu.py checks against the oracle at this size
        # (the plan's angles span [0, pi): the timing does not depend on the angle values, the parity test uses 2 pi)
        _, sad, n_rows, n_z = I.fdk_bench_geometry(args.config)
        d_cone = torch.from_numpy(I.fdk_bench_projections(args.config).astype(npdt)).cuda()
        d_vol = torch.empty((n_z, N, N), dtype=tdt, device="cuda")
        kfn = lambda: fbp.fbp_fdk_reconstruct(plan.handle, d_cone, d_vol, n_rows, 1.0, sad, n_z, 1.0, stream)  # noqa: E731
        for _ in range(2):
            kfn()
        k_ms = timed_loop(kfn, 5) / 5
        extras = {"fdk_ms": k_ms, "fdk_volume": [n_z, N, N], "fdk_detector_rows": n_rows,
                  "fdk_gupdates_per_s": float(n_z) * N * N * K / (k_ms * 1e-3) / 1e9,
                  "project_ms": p_ms, "project_slices": pb,
                  "project_gupdates_per_s": float(pb) * N * N * K / (p_ms * 1e-3) / 1e9,
                  "stack_interp_ms": i_ms, "stack_interp_gbs": i_bytes / (i_ms * 1e-3) / 1e9, "stack_interp_bytes": i_bytes,
                  "stack_interp_slices_out": n_out,
                  "metrics_ms": m_ms, "metrics_gbs": m_bytes / (m_ms * 1e-3) / 1e9, "metrics_bytes": m_bytes,
                  "psnr": float(out8[1].item()), "ssim": float(out8[2].item())}

    issue_rate = fbp.fbp_measure_issue_rate(fbp.FBP_F32 if dtype == "f32" else fbp.FBP_F64)
    if world > 1:
        t = torch.tensor([ms_step, e2e_s, b_ms, f_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step, e2e_s, b_ms, f_ms = [float(v) for v in t.tolist()]
    plan.close()
    del flush
    torch.cuda.empty_cache()
    return dict(info=info, graph_ms=graph_ms, ms_step=ms_step, f_ms=f_ms, b_ms=b_ms, e2e_s=e2e_s, updates=float(B) * N * N * K,
                clocks=clk.summary(), esize=h_sino.element_size(),
                h2d=h_sino.numel() * h_sino.element_size(), d2h=h_img.numel() * h_img.element_size(),
                extras=extras, input_sha=input_sha, issue_rate=issue_rate, e2e_spread=e2e_spread)


def record(args, r, world, peaks, peaks_src, dtype):
    """The measurements of one dtype as JSON-able fields (shared by the headline and the f64 sub-record)."""
    cfg = I.CONFIGS[args.config]
    info = r["info"]
    n_sm = info.get("device_sms", 148)
    total_updates = r["updates"] * world
    lanes = FP32_LANES if dtype == "f32" else FP64_LANES
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    peak_tinstr = n_sm * lanes * sm_max_mhz * 1e6 / 1e12
    bp_gups = r["updates"] / (r["b_ms"] * 1e-3) / 1e9
    achieved = bp_gups * 1e9 * FP_INSTR_PER_UPDATE / 1e12
    # co-limiter: every update needs two operands of the dtype from shared memory (128 B/clk/SM), whatever the packing
    smem_peak_tbs = n_sm * 128 * sm_max_mhz * 1e6 / 1e12
    # bytes of shared-memory operands per update: fp32 one 16-byte (mid, slope) unit per pixel pair; fp64 one 16-byte
    # `far` unit per pixel pair (the column walk keeps `near` in registers)
    smem_bytes_per_update = 8.0
    smem_tbs = bp_gups * 1e9 * smem_bytes_per_update / 1e12
    filt_bytes = 2.0 * cfg.batch * cfg.n_angles * cfg.n_det * r["esize"]
    kern = {"filter_ms": r["f_ms"], "backproject_ms": r["b_ms"], "backproject_gupdates_per_s": bp_gups,
            "filter_kind": {1: "direct", 2: "fft"}.get(info.get("filter_kind"), "?"),
            "filter_hbm_gbs": filt_bytes / (r["f_ms"] * 1e-3) / 1e9,
            "filter_hbm_frac_of_%s" % peaks_src: filt_bytes / (r["f_ms"] * 1e-3) / 1e9 / float(peaks["hbm_gbs"]),
            "path": ("sequential launches: profiling switches the batch pipeline off, `value` is the pipelined path"
                     if info["kernels_per_reconstruct"] > 2 else "the two launches of the timed step")}
    if info.get("filter_kind") == 2:
        n_fft = info["fft_length"]
        pairs = cfg.batch * ((cfg.n_angles + 1) // 2)
        flops = pairs * (2 * 5.0 * n_fft * float(np.log2(n_fft)) + 6.0 * n_fft)      # two transforms + the point-wise product
        kern["filter_fft_length"] = n_fft
        kern["filter_fft_tflops"] = flops / (r["f_ms"] * 1e-3) / 1e12
        kern["filter_fft_flops_frac_of_derived_peak"] = flops / (r["f_ms"] * 1e-3) / 1e12 / (2 * peak_tinstr)
    else:
        de, dn = (cfg.n_det + 1) // 2, cfg.n_det // 2
        fma = cfg.batch * cfg.n_angles * ((2.0 * de * dn + cfg.n_det) if args.window == "ramlak" else float(cfg.n_det) ** 2)
        kern["filter_tfma_per_s"] = fma / (r["f_ms"] * 1e-3) / 1e12
        kern["filter_fma_frac_of_derived_peak"] = fma / (r["f_ms"] * 1e-3) / 1e12 / peak_tinstr
    measured_tinstr = r.get("issue_rate", 0.0) / 1e12          # fbp_measure_issue_rate: FMA chains at full occupancy, this run
    roof = {"bound": "alu", "kernel": "backproject_kernel<%s>" % dtype, "achieved": achieved,
            "peak": peak_tinstr, "unit": "T %s lane-instr/s" % ("fp32" if dtype == "f32" else "fp64"),
            "frac": achieved / peak_tinstr,
            "peak_measured": measured_tinstr, "frac_of_measured_peak": achieved / measured_tinstr if measured_tinstr > 0 else None,
            "traffic": ncu_traffic(args.config, dtype, "backproject"),
            "co_limit": {"bound": "smem", "achieved": smem_tbs, "peak": smem_peak_tbs, "unit": "TB/s of shared-memory operands",
                         "frac": smem_tbs / smem_peak_tbs,
                         "note": "8 bytes of shared-memory operands per update = 16 updates per clock and SM, %.3f of the "
                                 "issue roofline: the ceiling the fp32 kernel sits on; not binding in fp64 since the "
                                 "column walk (FP64 pipe / issue bound; DESIGN.md 6.2)"
                                 % (smem_peak_tbs / smem_bytes_per_update / (peak_tinstr / FP_INSTR_PER_UPDATE))},
            "how": "%d FP instr/update (SURVEY 8(d)) x updates per launch / mean CUDA-event duration of the "
                   "back-projection launch(es); peak = %d SMs x %d lanes x %.0f MHz (%s sm_max_mhz); peak_measured = "
                   "%.2f T lane-instr/s from the FMA issue-rate kernel of the library (fbp_measure_issue_rate) in this run"
                   % (FP_INSTR_PER_UPDATE, n_sm, lanes, sm_max_mhz, peaks_src, measured_tinstr)}
    return {"value": total_updates / (r["ms_step"] * 1e-3) / 1e9, "ms_per_step": r["ms_step"],
            "slices_per_s": cfg.batch * world / (r["ms_step"] * 1e-3), "kernels": kern, "roofline": roof,
            "e2e": {"value": total_updates / r["e2e_s"] / 1e9, "unit": UNIT, "h2d_bytes_per_step": r["h2d"],
                    "d2h_bytes_per_step": r["d2h"], "ms_per_step": r["e2e_s"] * 1e3,
                    "api": "fbp_reconstruct_host (pinned host buffers, wall clock; median of per-call times)",
                    "spread": r["e2e_spread"]},
            "clocks": r["clocks"], "plan": info, "input_sha256": r["input_sha"],
            "graph_ms_per_step": r["graph_ms"]}


def spawn_ranks(args):
    """--gpus N > 1 outside torchrun: start N ranks (one per GPU) of this same command on this node."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")             # keep the communicator log (stderr)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def main():
    args = parse_args()
    if args.gpus > 1 and "RANK" not in os.environ:
        sys.exit(spawn_ranks(args))
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import torch.distributed as dist

    import paper_2109_02174_b200 as fbp

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    fbp.load_library(args.lib)

    r = measure(args, args.dtype, world, rank, local, dist)
    r64 = None
    if args.dtype == "f32" and args.config in BOTH_DTYPES and not args.no_f64:
        r64 = measure(args, "f64", world, rank, local, dist)
    if rank == 0:
        peaks, peaks_src = load_peaks()
        rec = record(args, r, world, peaks, peaks_src, args.dtype)
        launches_per_step = rec["plan"]["kernels_per_reconstruct"]
        line = {
            "metric": METRIC, "value": rec["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": rec["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": workload(args.config),
            "launch": {"parallelism": "slices sharded over %d GPU(s), no collective" % world,
                       "l2": "flushed between steps (256 MiB memset outside the timed events)",
                       "window": args.window, "options": args.opt, "plan": rec["plan"], "input_sha256": rec["input_sha256"]},
            "slices_per_s": rec["slices_per_s"], "kernels": rec["kernels"], "roofline": rec["roofline"], "e2e": rec["e2e"],
            "gpu_launches": args.steps * launches_per_step,
            "clocks": rec["clocks"],
        }
        if rec["graph_ms_per_step"] is not None:
            line["graph_ms_per_step"] = rec["graph_ms_per_step"]
        if r64 is not None:
            rec64 = record(args, r64, world, peaks, peaks_src, "f64")
            line["f64"] = {k: rec64[k] for k in ("value", "ms_per_step", "slices_per_s", "kernels", "roofline", "e2e", "clocks")}
            line["f64"]["unit"] = UNIT
            line["f64"]["gpu_launches"] = args.steps * rec64["plan"]["kernels_per_reconstruct"]
        if r["extras"]:
            ex = r["extras"]
            line["extras"] = dict(ex, metrics_hbm_frac=ex["metrics_gbs"] / float(peaks["hbm_gbs"]),
                                  stack_interp_hbm_frac=ex["stack_interp_gbs"] / float(peaks["hbm_gbs"]))
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.config)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
