#!/usr/bin/env python
"""bench.py — headline benchmark of the galario-b200 hot path.

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands, on the host cores

A "step" is one pass of the whole hot path — chi2Image: row FFT pass, column FFT pass, fused
rotate + bilinear gather + phase + chi-square — over one batch of
synthetic input.  The workload is BASELINE.json configs[3], the one its metric is quoted on
(nxy = 4096, M = 5e6, fp64, 500 Gaussians, 50-antenna tracks); the other configs are parity-test
cases.  Prints ONE JSON line (contract in the round prompt; extra keys are additive).

Multi-GPU: the path does not shard: under torchrun every rank runs an
independent replica of the same workload on its own GPU, no data-path collective; the time is the
max over ranks and `value` counts the evaluations of all ranks ("replicas only", scaling weak).
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

METRIC = "chi2Image evals/s at nxy=4096,M=5e6 fp64"
UNIT = "evals/s"


def algorithmic_bytes(nxy: int, M: int, esz: int, entry: str = "chi2Image", extent=None, C: int = 1):
    """what the METHOD must move, per kernel and per step (bytes).

    extent = None: the two-pass transform of the whole half plane (the table of §8(d)).
    extent = (kumax, kvs_min, kvs_max): the method's bytes of a transform pruned to that part of the half plane —
    the image is read once, only columns 0..kumax of the row-transformed image are written and read back, only
    rows kvs_min..kvs_max of those columns are written as the spectrum (once).  What this implementation moves on
    top of that (the uv-extent kernel re-reads u and v; the column-pair layout stores every value twice) is NOT
    counted: it lowers the achieved fraction instead.  *Profile entries read no image (the sweep is evaluated in
    the row-pass loader); sample* entries stream u, v in and V out (4 reals per point), chi2* five reals in."""
    img = 0 if "Profile" in entry else nxy * nxy * esz
    per_point = 5 * esz if entry.startswith("chi2") else 4 * esz
    samp = per_point * M
    if extent is None:
        spec = nxy * (nxy // 2 + 1) * 2 * esz
        row = img + spec               # read image, write half-spectrum
        col = 2 * spec                 # read + write half-spectrum
    else:
        kumax, rmin, rmax = extent
        cols = kumax + 1
        row = img + cols * nxy * 2 * esz
        col = cols * nxy * 2 * esz + cols * (rmax - rmin + 1) * 2 * esz
    out = {"uv_extent": 0, "row_pass": row, "col_pass": col, "sample": samp}
    out = {k: C * v for k, v in out.items()}
    out["step"] = sum(out.values())
    return out


# FP64 FMA rate measured on this box by gal_measure_fp64_fma_peak at the start of the run (TFLOP/s, 2 flop per DFMA);
# the ALU fractions below divide by it.  None until main() has measured it.
FP64_PEAK_TFLOPS = None

# Warp-level FP64 instructions (DADD + DMUL + DFMA: one issue slot of the FP64 pipe each) per launch of the three
# kernels of the headline call on its pruned extent, from the instruction mix of profiles/r2_stalls.md (c3:
# executed warp instructions x the FP64 share of the mix; the shares are rounded to 1 %, so these are +-3 %).
FP64_WARP_INSTR_CFG3 = {"row_pass": 19362880 * 0.64, "col_pass": 5298719 * 0.59, "sample": 31638068 * 0.34}


def alu_frac(warp_instr: float, ms: float):
    """Fraction of the measured FP64 pipe rate: lane-instructions per second over DFMA lanes per second."""
    if not FP64_PEAK_TFLOPS or ms <= 0:
        return None
    return warp_instr * 32.0 / (ms * 1e-3) / (FP64_PEAK_TFLOPS * 1e12 / 2.0)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(kernel: str):
    """DRAM bytes per launch (read + write) of `kernel` from the newest committed `ncu --set full` summary
    (profiles/*_ncu_traffic.csv: kernel,dram_bytes_read,dram_bytes_write,gpu_time_us), or None."""
    import csv
    import glob
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_ncu_traffic.csv"))):
        try:
            with open(path) as f:
                for row in csv.DictReader(f):
                    if row["kernel"] == kernel or row["kernel"].startswith(kernel + "_kernel"):
                        best = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
        except (OSError, ValueError, KeyError):
            continue
    return best


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def max_over_ranks(ms_local: float, world: int, device=None) -> float:
    """Timing rule: the job's time is the slowest rank's.  (Also used by the gloo CPU test.)"""
    if world <= 1:
        return ms_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def time_oracle(w, nthreads: int, repeats: int):
    import oracle
    best = float("inf")
    chi2 = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        chi2 = oracle.chi2Image(w.image, w.dxy, w.u, w.v, w.re_obs, w.im_obs, w.w, w.dRA, w.dDec, w.PA,
                                nthreads=nthreads)
        best = min(best, time.perf_counter() - t0)
    return best, chi2


def base_config(w, precision):
    return {"workload": "BASELINE.json configs[3]: chi2Image, 500 elliptical Gaussians (total 1 Jy), nxy=4096, "
                        "dxy=0.0015 arcsec, M=5e6 ALMA-like tracks (50 antennas, 16 km, 0.87 mm), log-normal weights",
            "entry": "chi2Image", "nxy": w.nxy, "M": w.M, "precision": precision, "seed": w.meta.get("seed"),
            "pruning": "library default (automatic): transform pruned to the part of the half plane the uv points can reach; "
                       "from the second call on the extent is the one the previous call derived, verified per point "
                       "(speculative extent, DESIGN.md section 5); unbound observations",
            "l2": "inputs+workspace per step (image 134 MB + spectrum 134 MB + 200 MB of per-point arrays) exceed "
                  "the 126 MB L2; no explicit flush"}


def run_reference(args, rank: int):
    """--impl reference: the oracle (never tuned) on the host cores; each step = the full workload."""
    if rank != 0:
        return
    import oracle
    import workloads
    oracle.build()
    w = workloads.config(3)
    T = oracle.host_threads()
    for _ in range(max(args.warmup, 0) and 1):
        time_oracle(w, T, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time_oracle(w, T, 1)
    dt = time.perf_counter() - t0
    val = args.steps / dt
    sample = f"full configs[3] workload per step (nxy=4096, M=5e6), {T} host threads, {args.steps} steps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": base_config(w, "f64"),
        "visibilities_per_s": val * w.M,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": T, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def event_time_ms(fn, steps: int, torch) -> float:
    """`steps` back-to-back calls between two CUDA events on the current stream (synchronised on both sides)."""
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def kernel_times_ms(plan, fn, steps: int, torch):
    """Per-kernel durations of `fn`'s calls, live: CUDA events recorded by the plan between its kernels."""
    plan.timing_enable(steps)
    for _ in range(steps):
        fn()
    torch.cuda.synchronize()
    ms, n = plan.timing_read()
    plan.timing_enable(0)
    return dict(zip(("uv_extent", "row_pass", "col_pass", "sample"), ms)), n


def measure_case(g, torch, dev, peak, name, w, dtype, entry, prune, steps, warmup, bind=False):
    """One row of the `other` block: us per call, fraction of the HBM roofline on the method's bytes (whole plane,
    and of the extent the call pruned to), per-kernel us.  Same event timing as the headline."""
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a), device=dev)
    esz = 8 if dtype == torch.float64 else 4
    C = w.image.shape[0] if entry == "chi2ImageBatch" else 1
    K = int(entry[len("chi2ImageSets"):]) if entry.startswith("chi2ImageSets") else 0     # observation sets of one image
    plan = g.Plan(w.nxy, max(C, K), dtype, dev.index)
    plan.set_pruning(prune)
    u, v = up(w.u), up(w.v)
    if entry == "sampleImage":
        image = up(w.image)
        out = torch.empty(w.M, dtype=torch.complex128 if esz == 8 else torch.complex64, device=dev)
        fn = lambda: plan.sampleImage(image, w.dxy, u, v, w.PA, w.dRA, w.dDec, out=out)
    else:
        re, im, wt = up(w.re_obs), up(w.im_obs), up(w.w)
        if entry == "chi2Profile":
            prof = up(w.profile)
            out = torch.empty(1, dtype=torch.float64, device=dev)
            fn = lambda: plan.chi2Profile(prof, w.Rmin, w.dR, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA, w.inc, out=out)
        elif entry == "chi2ProfileHankel":              # Eq. 25 directly: no image, no transform
            prof = up(w.profile)
            out = torch.empty(1, dtype=torch.float64, device=dev)
            fn = lambda: plan.chi2ProfileHankel(prof, w.Rmin, w.dR, u, v, re, im, wt, w.dRA, w.dDec, w.PA, w.inc, out=out)
        elif entry.startswith("chi2ImageMulti"):        # S placements of one model in one sampling launch
            S = int(entry[len("chi2ImageMulti"):])
            image = up(w.image)
            out = torch.empty(1, dtype=torch.float64, device=dev)
            pl = [(w.dRA * (1 + 0.1 * s), w.dDec * (1 - 0.1 * s), w.PA + 0.05 * s, 1.0 / S) for s in range(S)]
            fn = lambda: plan.chi2ImageMulti(image, w.dxy, u, v, re, im, wt, pl, out=out)
        elif K:                                         # K observation sets against one image: one transform, K samplings
            image = up(w.image)
            stack = lambda a, sc=None: torch.stack([torch.roll(a, 1009 * k) * ((1.0 - 0.1 * k) if sc else 1.0) for k in range(K)]).contiguous()
            us, vs, res, ims, wts = stack(u, True), stack(v, True), stack(re), stack(im), stack(wt)
            out = torch.empty(K + 1, dtype=torch.float64, device=dev)
            fn = lambda: plan.chi2ImageSets(image, w.dxy, us, vs, res, ims, wts, w.dRA, w.dDec, w.PA, out=out)
        elif entry == "chi2ImageBatch":
            image = up(w.image)
            out = torch.empty(C + 1, dtype=torch.float64, device=dev)
            fn = lambda: plan.chi2ImageBatch(image, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA, out=out)
        else:
            image = up(w.image)
            out = torch.empty(1, dtype=torch.float64, device=dev)
            fn = lambda: plan.chi2Image(image, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA, out=out)
        if bind:
            plan.bind_obs(u, v, re, im, wt)
    for _ in range(warmup):
        fn()
    ms = event_time_ms(fn, steps, torch)
    kms, _ = kernel_times_ms(plan, fn, min(steps, 100), torch)
    extent = tuple(plan.last_uv_extent())
    whole = (w.nxy // 2, 0, w.nxy - 1)
    B = algorithmic_bytes(w.nxy, w.M, esz, entry, None, C)
    Bp = algorithmic_bytes(w.nxy, w.M, esz, entry, extent, C) if extent != whole else B
    if K:                                               # the per-point arrays of the K - 1 further sets
        B, Bp = dict(B), dict(Bp)
        for d in (B, Bp):
            d["step"] += (K - 1) * d["sample"]
            d["sample"] *= K
    if kms.get("row_pass", 0) <= 0 < kms.get("col_pass", 0):       # nxy = 256 / 1024: both passes in one fused launch
        kms = {"uv_extent": kms["uv_extent"], "fft_fused": kms["col_pass"], "sample": kms["sample"]}
        B, Bp = dict(B), dict(Bp)
        B["fft_fused"], Bp["fft_fused"] = B["row_pass"] + B["col_pass"], Bp["row_pass"] + Bp["col_pass"]
    row = {"case": name, "entry": entry, "dtype": "f64" if esz == 8 else "f32", "nxy": w.nxy, "M": w.M, "C": C,
           "prune_mode": prune, "bound_obs": bool(bind), "us_per_call": 1e3 * ms, "uv_extent": list(extent),
           "pruned": extent != whole,
           "method_bytes_whole_plane": B["step"], "frac_whole_plane_bytes": B["step"] / (ms * 1e-3) / 1e9 / peak,
           "method_bytes_this_extent": Bp["step"], "frac": Bp["step"] / (ms * 1e-3) / 1e9 / peak,
           "kernels_us": {k: round(1e3 * t, 2) for k, t in kms.items() if t > 0},
           "kernels_frac": {k: round(Bp[k] / (t * 1e-3) / 1e9 / peak, 3) for k, t in kms.items() if t > 0 and Bp[k] > 0}}
    if entry == "chi2ProfileHankel":
        # no image, no transform: M * nr Bessel evaluations, FP64-ALU bound.  One evaluation is
        # about 45 FP64 instructions (hand count of hankel.cuh's inner loop); the pipe rate is the one measured on this box.
        nr = len(w.profile)
        for k in ("method_bytes_whole_plane", "frac_whole_plane_bytes", "method_bytes_this_extent", "frac", "uv_extent", "pruned"):
            row.pop(k)
        lanes_per_s = FP64_PEAK_TFLOPS * 1e12 / 2.0 if FP64_PEAK_TFLOPS else None      # measured DFMA lanes per second
        row.update({"bound": "alu", "j0_evaluations": w.M * nr, "j0_evaluations_per_s": w.M * nr / (ms * 1e-3),
                    "fp64_tflops_measured": FP64_PEAK_TFLOPS,
                    "fp64_pipe_frac_at_45_instr": 45.0 * w.M * nr / (ms * 1e-3) / lanes_per_s if lanes_per_s else None})
    del plan
    torch.cuda.empty_cache()
    return row


def measure_other(g, torch, dev, peak, w3, args, only=None):
    """Every other BASELINE.json config, the whole-plane path, fp32, sampleImage, nxy = 8192 and 16384, measured in
    this run with the headline's method.  Workloads are the seeded generators' full sizes, built
    when their case runs.  `only`: run the cases whose name contains this string (`--case`, used for ncu captures)."""
    import workloads
    rows = []
    S, Wm = args.other_steps, 5
    cache = {}

    def wl(key):
        if key not in cache:
            cache.clear()                              # one big workload in host memory at a time
            if key == "3":
                cache[key] = w3 if w3 is not None else workloads.config(3)
            elif key == "3f":
                cache[key] = (w3 if w3 is not None else workloads.config(3)).as_f32()
            elif key in ("8192", "16384"):
                # a seeded random image, the cfg-2 uv set scaled to the same pixel indices
                # (16384 is the paper's largest size: 810 ms per chi2Image on a GTX 1060 with
                # M = 1e6, copies included; context only)
                n = int(key)
                w2 = workloads.config(2)
                rng = np.random.default_rng(n)
                cache[key] = workloads.Workload(f"n{n}", "chi2Image", n, w2.dxy * 2048 / n, w2.u, w2.v, w2.re_obs, w2.im_obs,
                                                w2.w, w2.dRA, w2.dDec, w2.PA, image=rng.random((n, n)))
            else:
                cache[key] = workloads.config(int(key))
        return cache[key]

    def add(name, key, *a, **k):
        if only is not None and only not in name:
            return
        try:
            rows.append(measure_case(g, torch, dev, peak, name, wl(key), *a, steps=S, warmup=Wm, **k))
        except Exception as exc:                       # a failing case is reported, not hidden
            rows.append({"case": name, "error": repr(exc)})

    f64, f32 = torch.float64, torch.float32
    add("cfg3 f64 chi2Image (automatic pruning)", "3", f64, "chi2Image", 1)
    add("cfg3 f64 chi2Image, whole plane (prune 0)", "3", f64, "chi2Image", 0)
    add("cfg3 f64 chi2Image, bound observations", "3", f64, "chi2Image", 1, bind=True)
    add("cfg3 f64 sampleImage", "3", f64, "sampleImage", 1)
    add("cfg3 f32 chi2Image (automatic pruning)", "3f", f32, "chi2Image", 1)
    add("cfg3 f32 sampleImage", "3f", f32, "sampleImage", 1)
    add("cfg3 f32 chi2Image, whole plane (prune 0)", "3f", f32, "chi2Image", 0)
    add("cfg3 f32 chi2Image, bound observations", "3f", f32, "chi2Image", 1, bind=True)
    add("cfg2 f64 chi2Image", "2", f64, "chi2Image", 1)
    add("nxy=8192 f64 chi2Image (cfg-2 uv set, random image)", "8192", f64, "chi2Image", 1)
    add("nxy=16384 f64 chi2Image (cfg-2 uv set, random image)", "16384", f64, "chi2Image", 1)
    add("cfg1 f64 chi2Profile", "1", f64, "chi2Profile", 1)
    add("cfg1 f64 chi2Profile by the direct Hankel transform (Eq. 25)", "1", f64, "chi2ProfileHankel", 1)
    add("cfg2 f64 chi2ImageMulti, 4 placements in one sampling launch", "2", f64, "chi2ImageMulti4", 1)
    add("cfg2 f64 chi2ImageSets, 4 observation sets against one image in one call", "2", f64, "chi2ImageSets4", 1)
    add("cfg0 f64 chi2Image", "0", f64, "chi2Image", 1)
    add("cfg4 f64 chi2ImageBatch (128 channels)", "4", f64, "chi2ImageBatch", 1)
    add("cfg4 f64 chi2ImageBatch (128 channels), bound observations", "4", f64, "chi2ImageBatch", 1, bind=True)
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the `other` block (every other config and path)")
    ap.add_argument("--other-steps", type=int, default=50)
    ap.add_argument("--case", default=None,
                    help="run only the `other` cases whose name contains this string and print them (no headline, no "
                         "e2e, no oracle): the command the ncu captures under profiles/ were taken with")
    ap.add_argument("--prune", type=int, default=1, choices=[0, 1, 2],
                    help="gal_plan_set_pruning mode: 0 never, 1 automatic (library default), 2 always")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import paper_1709_06999_b200 as g
    import workloads
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the galario-b200 path has no CPU fallback")
    g.load_library()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    if args.case is not None:              # a selection of the `other` cases alone (profiling runs)
        if rank == 0:
            peak, _ = measured_peaks()
            print(json.dumps({"cases": measure_other(g, torch, dev, peak, None, args, only=args.case)}))
        if world > 1:
            torch.distributed.destroy_process_group()
        return

    w = workloads.config(3)               # every rank: the same seeded replica
    esz = 8
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a), device=dev)
    image, u, v, re, im, wt = map(up, (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    plan = g.Plan(w.nxy, 1, torch.float64, local_rank)
    plan.set_pruning(args.prune)
    out = torch.empty(1, dtype=torch.float64, device=dev)
    step = lambda: plan.chi2Image(image, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA, out=out)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    global FP64_PEAK_TFLOPS
    # the clock is sampled over the whole GPU-busy part of the headline (FP64 peak, warm-up, timed loop, per-kernel
    # timing, bound-observation loop): the timed loop alone lasts 2-3 ms, one or two samples
    clk = ClockSampler(local_rank)
    clk.__enter__()
    FP64_PEAK_TFLOPS, fp64_peak_ms = g.measure_fp64_peak(local_rank)
    for _ in range(args.warmup):
        step()
    barrier()
    l0 = plan.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    launches = plan.launch_count() - l0
    chi2_val = float(out.cpu()[0])
    ms_step = ms_total / args.steps
    value = world * args.steps / (ms_total * 1e-3)

    # per-kernel durations, live, CUDA events on the launching stream between the kernels
    kms, ncalls = kernel_times_ms(plan, step, min(args.steps, 200), torch)
    extent = plan.last_uv_extent()
    pruned = tuple(extent) != (w.nxy // 2, 0, w.nxy - 1)

    peak, peak_src = measured_peaks()
    B = algorithmic_bytes(w.nxy, w.M, esz)                                   # whole half plane
    Bk = algorithmic_bytes(w.nxy, w.M, esz, extent=extent) if pruned else B  # the method's bytes of this extent
    kernels = []
    ms_sum = max(sum(kms.values()), 1e-12)
    for name, ms in kms.items():
        if ms <= 0:
            continue
        gbs = Bk[name] / (ms * 1e-3) / 1e9
        kernels.append({"kernel": name, "ms": ms, "algorithmic_bytes": Bk[name], "achieved_gbs": gbs,
                        "frac": gbs / peak, "share_of_step": ms / ms_sum,
                        "alu_frac": alu_frac(FP64_WARP_INSTR_CFG3[name], ms) if (pruned and name in FP64_WARP_INSTR_CFG3) else None})
    dom = max(kernels, key=lambda k: k["ms"])
    roofline = {"bound": "hbm", "kernel": dom["kernel"], "achieved": dom["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": dom["frac"], "traffic": ncu_traffic(dom["kernel"]),
                "traffic_source": "committed ncu --set full summary (profiles/*_ncu_traffic.csv), not measured in this run",
                "peak_source": peak_src, "ms_per_launch": dom["ms"], "launches_timed": ncalls}
    whole_gbs = B["step"] / (ms_step * 1e-3) / 1e9
    moved_gbs = Bk["step"] / (ms_step * 1e-3) / 1e9
    step_roofline = {"bound": "hbm", "algorithmic_bytes": Bk["step"], "achieved": moved_gbs, "peak": peak,
                     "unit": "GB/s", "frac": moved_gbs / peak, "target_frac": 0.60,
                     "pruned_transform": pruned, "uv_extent": list(extent),
                     "whole_plane_bytes": B["step"], "frac_whole_plane_credit": whole_gbs / peak,
                     "note": "frac: the method's bytes of the extent this call pruned to (image once, reachable columns "
                             "of the row-transformed image out and in, reachable rows of the spectrum out once, "
                             "per-point arrays once) over the step time; frac_whole_plane_credit: SURVEY.md 8(d)'s "
                             "two-pass whole-half-plane byte count over the same time (credits traffic a pruned call "
                             "never moves; the whole-plane path itself is measured in `other`)"}

    # the same step on a BOUND observation set (gal_plan_bind_obs: the caller promises the five observation arrays
    # stay unchanged, as in a fit of one data set; the plan samples its private uv-sorted copy and skips the
    # per-call uv-extent kernel).  Reported beside the headline, not instead of it.
    plan.bind_obs(u, v, re, im, wt)
    for _ in range(args.warmup):
        step()
    barrier()
    b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    b0.record()
    for _ in range(args.steps):
        step()
    b1.record()
    barrier()
    ms_bound = max_over_ranks(b0.elapsed_time(b1), world, dev) / args.steps
    chi2_bound = float(out.cpu()[0])
    bkms, _ = kernel_times_ms(plan, step, min(args.steps, 200), torch)
    bext = plan.last_uv_extent()
    Bb = algorithmic_bytes(w.nxy, w.M, esz, extent=bext)
    bound_obs = {"ms_per_step": ms_bound, "value": world / (ms_bound * 1e-3), "unit": UNIT,
                 "chi2_rel_diff_vs_unbound": abs(chi2_bound - chi2_val) / abs(chi2_val), "uv_extent": list(bext),
                 "algorithmic_bytes": Bb["step"], "frac": Bb["step"] / (ms_bound * 1e-3) / 1e9 / peak,
                 "frac_whole_plane_credit": B["step"] / (ms_bound * 1e-3) / 1e9 / peak,
                 "kernels_us": {k: round(1e3 * t, 2) for k, t in bkms.items() if t > 0},
                 "kernels_frac": {k: round(Bb[k] / (t * 1e-3) / 1e9 / peak, 3) for k, t in bkms.items() if t > 0 and Bb[k] > 0}}
    plan.unbind_obs()
    clk.__exit__(None, None, None)

    # end to end through the host-pointer C-ABI call: pinned host inputs, H2D + kernels + D2H each step
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    himg, hu, hv, hre, him, hw = map(pin, (w.image, w.u, w.v, w.re_obs, w.im_obs, w.w))
    h2d = sum(t.numel() * t.element_size() for t in (himg, hu, hv, hre, him, hw))
    estep = lambda: plan.chi2Image_host(himg, w.dxy, hu, hv, hre, him, hw, w.dRA, w.dDec, w.PA)
    for _ in range(2):
        e2e_chi2 = estep()
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(args.e2e_steps):
        e2e_chi2 = estep()
    f1.record()
    barrier()
    e2e_ms = max_over_ranks(f0.elapsed_time(f1), world, dev)
    e2e = {"value": world * args.e2e_steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": 8, "steps": args.e2e_steps, "ms_per_step": e2e_ms / args.e2e_steps,
           "api": "gal_chi2_image_host_f64 (pinned host buffers in, chi2 to a host double out)",
           "matches_device_path": bool(e2e_chi2 == chi2_val)}
    # the fit loop the library is made for: the observations stay on the device, every step brings a
    # new MODEL IMAGE from the host (pinned) and takes chi2 back.  Reported beside `e2e`, not instead of it.
    img_dev = torch.empty_like(image)
    hout = torch.empty(1, dtype=torch.float64).pin_memory()

    def istep():
        img_dev.copy_(himg, non_blocking=True)
        plan.chi2Image(img_dev, w.dxy, u, v, re, im, wt, w.dRA, w.dDec, w.PA, out=out)
        hout.copy_(out, non_blocking=True)

    for _ in range(3):
        istep()
    barrier()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record()
    for _ in range(args.e2e_steps):
        istep()
    g1.record()
    barrier()
    img_ms = max_over_ranks(g0.elapsed_time(g1), world, dev)
    e2e_image_only = {"value": world * args.e2e_steps / (img_ms * 1e-3), "unit": UNIT,
                      "h2d_bytes_per_step": himg.numel() * himg.element_size(), "d2h_bytes_per_step": 8,
                      "steps": args.e2e_steps, "ms_per_step": img_ms / args.e2e_steps,
                      "what": "observations resident on the device, the model image copied from pinned host memory and chi2 "
                              "copied back every step (torch copies + gal_chi2_image_f64)",
                      "matches_device_path": bool(float(hout[0]) == chi2_val)}
    del himg, hu, hv, hre, him, hw, img_dev

    result = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": dict(base_config(w, "f64"), uv_extent=list(extent), pruned_transform=pruned,
                                            method_bytes_this_extent=Bk["step"]),
        "clocks": clk.summary(), "fp64_tflops_measured": FP64_PEAK_TFLOPS, "fp64_peak_launch_ms": fp64_peak_ms,
        "fp64_peak_note": "gal_measure_fp64_fma_peak: 8 independent DFMA chains per thread, 8 x 256 threads per SM, best of 5; "
                          "kernels[].alu_frac = FP64 lane-instructions/s (profiles/r2_stalls.md mix) over this rate", "e2e": e2e, "e2e_image_only": e2e_image_only,
        "gpu_launches": int(launches), "roofline": roofline, "step_roofline": step_roofline, "kernels": kernels,
        "visibilities_per_s": value * w.M, "chi2": chi2_val, "multi_gpu": "replicas only", "bound_obs": bound_obs,
        "paper_context": "GTX 1060, M=1e6, PCIe copies included: chi2Image 4096^2 = 59 ms (PAPER.md:619); not like for like",
    }

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle                      # the cpu_baseline leg: the one place bench.py may run the oracle
        oracle.build()
        T = oracle.host_threads()
        tT, chi2_o = time_oracle(w, T, 3)
        t1, _ = time_oracle(w, 1, 1)
        result["cpu_baseline"] = {"value": 1.0 / tT, "unit": UNIT, "cores": T, "kind": "oracle",
                                  "sample": f"the full configs[3] workload (one evaluation), best of 3 with {T} threads",
                                  "value_1thread": 1.0 / t1, "seconds_T_threads": tT, "seconds_1_thread": t1,
                                  "chi2_rel_diff_vs_gpu": abs(chi2_o - chi2_val) / abs(chi2_o)}
    if rank == 0 and world == 1 and not args.no_other:
        del plan, image, u, v, re, im, wt
        torch.cuda.empty_cache()
        result["other"] = measure_other(g, torch, dev, peak, w, args)
    if rank == 0:
        print(json.dumps(result))
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
