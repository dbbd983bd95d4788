"""bench.py -- one JSON line for the FBP hot path (filter + back-projection) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--dtype f32] [--impl ours|reference]

A "step" is one fbp_reconstruct (Ram-Lak filter, then back-projection: all rows of SURVEY.md
8(a)) of one batch of the chosen BASELINE.json configuration; the default is config 3
(512x512 image, 360 angles, 725 bins, fp32), the one BASELINE.json's metric is quoted on.
`value` = back-projection updates (batch * N^2 * K) per second of WHOLE-STEP time, in
Gupdates/s, inputs resident in HBM, L2 flushed between steps (outside the timed events).
Under torchrun each rank reconstructs its own slices (weak scaling, no collective:
slices are independent problems).
"""
from __future__ import annotations

import argparse
import json
import os
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
SM_COUNT, FP32_LANES, FP64_LANES = 148, 128, 64


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=3, choices=sorted(I.CONFIGS))
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--window", default="ramlak", choices=["ramlak", "shepp-logan", "cosine", "hamming", "hann"],
                    help="reconstruction filter (SURVEY.md 8(f) row 1); the headline is ramlak")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=INT",
                    help="launch-configuration override passed to fbp_create_tuned (A/B runs), e.g. --opt filter_sb=2")
    ap.add_argument("--extras", action="store_true", help="also time fbp_metrics (PSNR/SSIM) on the output stack")
    return ap.parse_args()


def workload(cfg_id):
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
            self._stop.wait(0.002)

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


def time_oracle(cfg_id, frac=1.0, reps=1):
    """The CPU fp64 oracle, as it stands, on the host cores, on a bounded sample of slice 0 of
    the workload: a fraction `frac` of the filter rows and of the pixels (all of them when
    frac >= 1), each timing scaled to the full slice.  Returns (Gupdates/s, cores, sample
    description, seconds per full slice)."""
    import oracle

    cfg = I.CONFIGS[cfg_id]
    ang = I.config_angles(cfg_id)
    sino = _slice0(cfg_id)
    cores = oracle.max_threads()
    n, k, d = cfg.image_n, cfg.n_angles, cfg.n_det
    updates = n * n * k
    best = float("inf")
    if frac >= 1.0:
        for _ in range(reps):
            t0 = time.perf_counter()
            oracle.reconstruct(sino, ang, n)
            best = min(best, time.perf_counter() - t0)
        sample = "slice 0 of cfg%d in full (filter + back-projection), best of %d" % (cfg_id, reps)
    else:
        rows = np.unique(np.linspace(0, k - 1, num=max(1, int(frac * k)), dtype=np.int32))
        npix = max(64, int(frac * n * n))
        rng = np.random.default_rng(0)
        rr = rng.integers(0, n, npix).astype(np.int32)
        cc = rng.integers(0, n, npix).astype(np.int32)
        for _ in range(reps):
            t0 = time.perf_counter()
            oracle.filter_rows(sino, rows)
            t_f = (time.perf_counter() - t0) * k / len(rows)
            t0 = time.perf_counter()
            oracle.backproject_pixels(sino, ang, n, rr, cc)
            t_b = (time.perf_counter() - t0) * (n * n) / npix
            best = min(best, t_f + t_b)
        sample = ("slice 0 of cfg%d: %d of %d filter rows and %d of %d pixels, each timing scaled to the full slice"
                  % (cfg_id, len(rows), k, npix, n * n))
    return updates / best / 1e9, cores, sample, best


def oracle_fraction(cfg_id, budget_s, n_steps):
    """Fraction of a slice per step so that n_steps oracle steps take about budget_s seconds."""
    cfg = I.CONFIGS[cfg_id]
    probe = min(1.0, 2e7 / (cfg.image_n * cfg.image_n * cfg.n_angles))
    _, _, _, t_full = time_oracle(cfg_id, probe)
    return min(1.0, budget_s / (max(n_steps, 1) * t_full))


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
def run_ours(args):
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
    fbp.load_library()

    cfg = I.CONFIGS[args.config]
    tdt = torch.float32 if args.dtype == "f32" else torch.float64
    npdt = np.float32 if args.dtype == "f32" else np.float64
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
    plan = fbp.Plan(list(ang), D, N, dtype=args.dtype, max_batch=B, options=options)
    if args.window != "ramlak":
        plan.set_window(args.window)
    info = plan.info()
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
    e2e_steps = max(3, min(args.steps, 100))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        fbp.fbp_reconstruct_host(plan.handle, h_sino, h_img, B, stream)
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps

    extras = None
    if args.extras:
        # fbp_metrics on the whole output stack against a copy: 2 passes x 2 arrays read (HBM-bound)
        other = d_img.clone()
        out8 = torch.empty(8, dtype=torch.float64, device="cuda")
        mfn = lambda: fbp.fbp_metrics(plan.handle, d_img, other, d_img.numel(), 1.0, -1.0, -1.0, out8, stream)  # noqa: E731
        for _ in range(3):
            mfn()
        m_ms = timed_loop(mfn, 20) / 20
        m_bytes = 4.0 * d_img.numel() * d_img.element_size()
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
        extras = {"project_ms": p_ms, "project_slices": pb,
                  "project_gupdates_per_s": float(pb) * N * N * K / (p_ms * 1e-3) / 1e9,
                  "stack_interp_ms": i_ms, "stack_interp_gbs": i_bytes / (i_ms * 1e-3) / 1e9, "stack_interp_bytes": i_bytes,
                  "stack_interp_slices_out": n_out,
                  "metrics_ms": m_ms, "metrics_gbs": m_bytes / (m_ms * 1e-3) / 1e9, "metrics_bytes": m_bytes,
                  "metrics_launches": 2, "psnr": float(out8[1].item()), "ssim": float(out8[2].item())}

    if world > 1:
        t = torch.tensor([ms_step, e2e_s, b_ms, f_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step, e2e_s, b_ms, f_ms = [float(v) for v in t.tolist()]
    updates = float(B) * N * N * K
    return dict(world=world, rank=rank, cfg=cfg, info=info, ms_step=ms_step, f_ms=f_ms, b_ms=b_ms, e2e_s=e2e_s,
                updates=updates, clocks=clk.summary(), esize=h_sino.element_size(),
                h2d=h_sino.numel() * h_sino.element_size(), d2h=h_img.numel() * h_img.element_size(), plan=plan,
                extras=extras, input_sha=input_sha)


# dram__bytes_read.sum + dram__bytes_write.sum of the back-projection kernel, per launch, from
# the committed `ncu --set full` capture (profiles/); None until a capture for that key exists.
NCU_TRAFFIC_BYTES = {(3, "f32"): 2968320, (3, "f64"): 5904640, (4, "f32"): 371400704 + 58770176}   # profiles/r1d_bp_cfg3_f32_ncu_full.txt, r1f_*.txt (ncu flushes caches per replay pass)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    r = run_ours(args)
    if r["rank"] != 0:
        return
    peaks, peaks_src = load_peaks()
    cfg, world = r["cfg"], r["world"]
    total_updates = r["updates"] * world
    value = total_updates / (r["ms_step"] * 1e-3) / 1e9
    e2e_value = total_updates / r["e2e_s"] / 1e9
    lanes = FP32_LANES if args.dtype == "f32" else FP64_LANES
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    peak_tinstr = SM_COUNT * lanes * sm_max_mhz * 1e6 / 1e12
    bp_gups = r["updates"] / (r["b_ms"] * 1e-3) / 1e9
    achieved = bp_gups * 1e9 * FP_INSTR_PER_UPDATE / 1e12
    filt_bytes = 2.0 * cfg.batch * cfg.n_angles * cfg.n_det * r["esize"]
    de, dn = (cfg.n_det + 1) // 2, cfg.n_det // 2
    filt_fma = cfg.batch * cfg.n_angles * (2.0 * de * dn + cfg.n_det)
    if args.window != "ramlak":
        filt_fma = cfg.batch * cfg.n_angles * float(cfg.n_det) * cfg.n_det      # every tap is non-zero
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": r["ms_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": dict(workload(args.config), parallelism="slices sharded over %d GPU(s), no collective" % world,
                       l2="flushed between steps (256 MiB memset outside the timed events)",
                       plan=r["info"]),
        "slices_per_s": cfg.batch * world / (r["ms_step"] * 1e-3),
        "kernels": {"filter_ms": r["f_ms"], "backproject_ms": r["b_ms"], "backproject_gupdates_per_s": bp_gups,
                    "backproject_smem_operand_tbs": bp_gups * 1e9 * 2 * r["esize"] / 1e12,
                    "backproject_frac_of_smem_ceiling": bp_gups * 1e9 * 2 * r["esize"] / (SM_COUNT * 128 * sm_max_mhz * 1e6),
                    "filter_hbm_gbs": filt_bytes / (r["f_ms"] * 1e-3) / 1e9,
                    "filter_hbm_frac_of_%s" % peaks_src: filt_bytes / (r["f_ms"] * 1e-3) / 1e9 / float(peaks["hbm_gbs"]),
                    "filter_tfma_per_s": filt_fma / (r["f_ms"] * 1e-3) / 1e12,
                    "filter_fma_frac_of_derived_peak": filt_fma / (r["f_ms"] * 1e-3) / 1e12 / peak_tinstr},
        "roofline": {"bound": "alu", "kernel": "backproject_kernel<%s>" % args.dtype, "achieved": achieved,
                     "peak": peak_tinstr, "unit": "T %s lane-instr/s" % ("fp32" if args.dtype == "f32" else "fp64"),
                     "frac": achieved / peak_tinstr,
                     "traffic": NCU_TRAFFIC_BYTES.get((args.config, args.dtype)),
                     "how": "%d FP instr/update (SURVEY 8(d)) x updates per launch / mean CUDA-event duration of the "
                            "back-projection launch(es); peak = %d SMs x %d lanes x %.0f MHz (%s sm_max_mhz)"
                            % (FP_INSTR_PER_UPDATE, SM_COUNT, lanes, sm_max_mhz, peaks_src)},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"],
                "ms_per_step": r["e2e_s"] * 1e3, "api": "fbp_reconstruct_host (pinned host buffers, wall clock)"},
        "gpu_launches": args.steps * r["info"]["kernels_per_reconstruct"],
        "clocks": r["clocks"],
    }
    line["config"]["window"] = args.window
    line["config"]["input_sha256"] = r["input_sha"]
    if r["extras"]:
        line["extras"] = dict(r["extras"], metrics_hbm_frac=r["extras"]["metrics_gbs"] / float(peaks["hbm_gbs"]),
                              stack_interp_hbm_frac=r["extras"]["stack_interp_gbs"] / float(peaks["hbm_gbs"]))
    if world == 1 and not args.no_cpu_baseline:
        frac = oracle_fraction(args.config, 15.0, 3)
        g, cores, sample, _ = time_oracle(args.config, frac, reps=3)
        line["cpu_baseline"] = {"value": g, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    r["plan"].close()
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
