#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (multi-scale filter + local threshold, every row of
SURVEY.md 8(a)) on synthetic cubes shaped like BASELINE.json's configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config {1..5}] [--impl b200|reference]

One "step" = one pgsf_find_multiscale call over one batch of synthetic input (all scales, filtered
cubes kept as outputs, mask, count).  Prints ONE JSON line (rank 0).
for the definition of every field.  N > 1 = N independent replicas (the path does not shard:
DESIGN.md "Multi-GPU"), no data-path collective; the timing is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gvoxel/s per Gaussian scale (filter+threshold)"
UNIT = "Gvoxel-scales/s"
STATS_FLOPS = 21            # statistics + threshold per voxel per scale
STATS_Z_FLOPS = 5           # of which the z-direction window: 2 x (add + subtract) + 1 square
FP32_LANES_PER_SM = 128     # B200_PROFILING.md unit counts: 148 SMs, 1965 MHz max SM clock


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            j = json.load(fh)
        return {"hbm_gbs": float(j["hbm_gbs"]), "sm_max_mhz": float(j.get("sm_max_mhz", 1965.0)),
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


def _dram_traffic(workload: str, kernel: str):
    """DRAM bytes per launch of `kernel` from the committed ncu capture of the current kernels
    (profiles/r02_dram_traffic.csv), or None when no capture exists for this workload / kernel."""
    path = os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")
    if not os.path.exists(path):
        return None
    import csv
    with open(path) as fh:
        for row in csv.DictReader(fh):
            if row["workload"] == workload and row["kernel"] == kernel:
                return float(row["dram_bytes_per_launch"])
    return None


def _alu_peak_tflops(sm_count: int, sm_mhz: float) -> float:
    """FP32 CUDA-core peak: SMs x 128 lanes x 2 flop x clock."""
    return sm_count * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def _radius(sigma: float, truncate: float) -> int:
    import math
    return int(math.ceil(truncate * sigma)) if sigma > 0 else 0


def _taps(w):
    """[(Tx, Ty, Tz)] per scale: the true tap counts 2 ceil(3 sigma) + 1."""
    return [tuple(2 * _radius(s[a], w.truncate) + 1 for a in range(3)) for s in w.sigmas]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------ CPU oracle leg

CPU_SAMPLE = (256, 256, 512)   # cpu_baseline leg: ~10-30 s of host work
REF_SAMPLE = (128, 128, 256)   # --impl reference: a few seconds per step, K steps within minutes


def _oracle_sample_region(w, size=CPU_SAMPLE):
    """The bounded sample the oracle is timed on: a centred brick of at most `size` voxels of the
    workload's cube, all scales."""
    lo = tuple(max(0, (n - s) // 2) for n, s in zip(w.dims, size))
    hi = tuple(min(n, l + s) for n, l, s in zip(w.dims, lo, size))
    return lo, hi


def time_oracle(w, sub, a, lo, hi, repeats: int = 1):
    """Seconds per pass of the fp64 oracle (as it stands, all host cores via its OpenMP loops) over
    the sample region; returns (seconds, voxel_scales, threads)."""
    from oracle import pgsf_oracle
    pgsf_oracle.build()
    threads = pgsf_oracle.set_threads(0)
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        pgsf_oracle.find_region(sub, a, w.dims, w.sigmas, w.box_half, w.k, lo, hi, w.halo, w.truncate)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    vs = (hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2]) * len(w.sigmas)
    return best, vs, threads


def _sample_text(w, lo, hi):
    return (f"centred brick {hi[0]-lo[0]}x{hi[1]-lo[1]}x{hi[2]-lo[2]} of {w.name}, all {len(w.sigmas)} scales, "
            f"oracle region mode (input brick +-(r+h)); rate = brick voxel-scales / wall time")


def run_reference(args, w):
    """--impl reference: the oracle (oracle/, fp64, gcc -O2 + OpenMP) on the host cores; every step is
    one pass over the bounded sample of the same workload.  Rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    from paper_1507_04941_b200 import synth
    lo, hi = _oracle_sample_region(w, REF_SAMPLE)
    # the sample brick is cut from the same seeded cube when a GPU is there to generate it quickly;
    # otherwise (no GPU) an equally shaped seeded brick is generated on the host
    from oracle import pgsf_oracle
    a, e = pgsf_oracle.required_input_box(w.dims, w.sigmas, w.box_half, lo, hi, w.truncate)
    shape = (e[2] - a[2], e[1] - a[1], e[0] - a[0])
    if torch.cuda.is_available():
        torch.cuda.set_device(0)
        d = synth.make_workload(w, "cuda:0")
        sub = d[0, a[2]:e[2], a[1]:e[1], a[0]:e[0]].cpu().numpy()
        del d
        torch.cuda.empty_cache()
    else:
        sub = synth.make_cube(shape, w.seed, max(1, w.n_sources // 64), device="cpu", sxy_range=w.sxy_range,
                              sz_range=w.sz_range, amp_range=w.amp_range).numpy()
    for _ in range(min(args.warmup, 1)):
        time_oracle(w, sub, a, lo, hi)
    t = []
    threads = 1
    for _ in range(args.steps):
        dt, vs, threads = time_oracle(w, sub, a, lo, hi)
        t.append(dt)
    sec = sum(t) / len(t)
    value = vs / sec / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "sample": _sample_text(w, lo, hi)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": _sample_text(w, lo, hi)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ B200 arm

def replica_workload(w, rank: int):
    """Replicas only: rank r runs its own copy of the workload, seed offset by 100 r."""
    from dataclasses import replace
    return replace(w, seed=w.seed + 100 * rank) if rank else w


def max_over_ranks(ms: float, world: int, device) -> float:
    """Step time of the job = the slowest rank's (all-reduce MAX over the process group)."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(n_vox: int, n_scales: int, world: int, ms_step: float) -> float:
    """Whole-job G voxel-scales/s: every rank processed n_vox x n_scales in ms_step."""
    return n_vox * n_scales * world / (ms_step * 1e-3) / 1e9


def _kernel_work(name: str, w, taps, n_vox: int):
    """Algorithmic (flops, bytes) of ONE launch of the kernel `name`: the work
    the separable method must do, not what the implementation happens to move.  Bytes follow SURVEY.md 8(d)
    strictly: the input is read once (charged to the x/y kernel), every filtered cube is written once (charged
    to its z kernel), the mask is written once (charged to the statistics kernel); every intermediate (t2, the
    window sums, the re-read of f) is implementation traffic and counts for nothing here."""
    S = len(taps)
    kind, _, tail = name.partition("_")
    if kind in ("bxy", "bz"):                     # the filter kernels with all-ones taps (Eq. 1 denominator)
        kind = kind[1:]
    if kind == "xy" and tail.startswith("m"):  # x and y passes of the scales in the bit mask, one read of the input
        grp = [t for i, t in enumerate(taps) if (int(tail[1:]) >> i) & 1]
        return 2 * sum(t[0] + t[1] for t in grp) * n_vox, 4 * n_vox
    if kind == "xy" and tail.startswith("s"):
        t = taps[int(tail[1:])]
        return 2 * (t[0] + t[1]) * n_vox, 4 * n_vox
    if kind == "z" and tail.startswith("s"):
        t = taps[int(tail[1:])]
        return 2 * t[2] * n_vox, 4 * n_vox
    if kind == "zm" and tail.startswith("s"):   # z pass + z-direction window sums (5 of the 21 statistics flops)
        t = taps[int(tail[1:])]
        return (2 * t[2] + STATS_Z_FLOPS) * n_vox, 4 * n_vox
    if kind == "stats" and tail == "xybox":     # x/y window sums + selection after a fused zm launch
        return (STATS_FLOPS - STATS_Z_FLOPS) * n_vox, 1 * n_vox
    if kind == "w":                              # Eq. 1 helpers: product, box sum of the weights, division
        return {"mul": (1, 12), "box": (6, 8), "div": (1, 12)}.get(tail, (0, 0))[0] * n_vox, \
               {"mul": (1, 12), "box": (6, 8), "div": (1, 12)}.get(tail, (0, 0))[1] * n_vox
    if kind == "stats" and tail == "all":    # statistics of every scale, one mask write
        return STATS_FLOPS * S * n_vox, (4 * S + 1) * n_vox
    if kind == "stats":
        return STATS_FLOPS * n_vox, 1 * n_vox
    return 0, 0


def _path_roofline(w, taps, n_vox, ms_step, alu_peak, hbm_peak):
    S = len(taps)
    path_flops = sum(2 * sum(t) + STATS_FLOPS for t in taps) * n_vox
    path_bytes = (4 + 4 * S + 1) * n_vox
    t_alu, t_hbm = path_flops / (alu_peak * 1e12), path_bytes / (hbm_peak * 1e9)
    t_path = max(t_alu, t_hbm)
    return {"flops_per_voxel": path_flops / n_vox, "bytes_per_voxel": path_bytes / n_vox,
            "roofline_ms": t_path * 1e3, "frac": t_path * 1e3 / ms_step, "bound": "alu" if t_alu >= t_hbm else "hbm"}


FLAGS = 0     # --flags: PGSF_FLAG_* plan flags (8 = the optional tensor-core z pass)
TUNE = 0      # --tune: PGSF_OPT_TUNE bits (kernel variants for A/B measurements; results are identical)


def measure_workload(w, dev, device_index, rank, world, steps, warmup, peaks, sm_count, detail=True):
    """One workload on this rank's GPU: W warm-up steps, K timed steps (CUDA events on the launching stream,
    per-launch profiling events OFF), then -- with detail -- a second, profiled pass for the per-kernel table and
    the per-scale calls of SURVEY.md 8(d) metric (i).  Returns (dict of results, ctx with the live buffers)."""
    import torch
    import torch.distributed as dist
    from paper_1507_04941_b200 import binding, synth

    d = synth.make_workload(replica_workload(w, rank), dev)
    n_vox = w.voxels
    S = len(w.sigmas)
    taps = _taps(w)
    plan = binding.Plan(w.dims, w.sigmas, w.box_half, w.k, batch=w.batch, halo=w.halo, truncate=w.truncate,
                        device=device_index, flags=FLAGS)
    if TUNE:
        plan.pgsf_plan_set_option(binding.PGSF_OPT_TUNE, TUNE)
    filt = [torch.empty_like(d) for _ in range(S)]
    mask = torch.empty(d.shape, dtype=torch.uint8, device=dev)
    cnt = torch.zeros(1, dtype=torch.int64, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        plan.pgsf_find_multiscale(d, d_filtered=filt, d_mask=mask, d_count=cnt, stream=stream)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(device_index)
    sampler.start()
    l0 = plan.pgsf_plan_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(stream)
    for _ in range(steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = plan.pgsf_plan_launch_count() - l0
    clocks = sampler.stop()
    count = int(cnt.item())
    ms_step = max_over_ranks(ms_total, world, dev) / steps
    alu_peak = _alu_peak_tflops(sm_count, peaks["sm_max_mhz"])
    hbm_peak = peaks["hbm_gbs"]
    out = {"ms_per_step": ms_step, "value": aggregate_value(n_vox, S, world, ms_step), "count": count,
           "launches": int(launches), "clocks": clocks,
           "path_roofline": _path_roofline(w, taps, n_vox, ms_step, alu_peak, hbm_peak)}
    ctx = dict(plan=plan, d=d, filt=filt, mask=mask, cnt=cnt, rank=rank, world=world, dev=dev)
    if not detail:
        return out, ctx

    # ---- second pass, per-launch CUDA events on: which kernel dominates, and its roofline
    psteps = max(1, min(steps, 5))
    plan.pgsf_plan_set_profiling(True)
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record(stream)
    for _ in range(psteps):
        step()
    pe1.record(stream)
    torch.cuda.synchronize()
    prof = plan.pgsf_plan_profile()
    plan.pgsf_plan_set_profiling(False)
    ms_prof_total = pe0.elapsed_time(pe1)
    kern = []
    cube = w.dims[0] * w.dims[1] * w.dims[2]
    for name, (n, ms) in prof.items():
        # voxels per launch: a batch goes through in groups of cubes; a name shared by all scales
        # (stats_*) is launched once per scale and group
        per_step = S if name.startswith("stats_") else 1
        vox_launch = cube * w.batch * per_step * psteps / max(n, 1)
        if name == "pivot":
            vox_launch = 0
        fl, by = _kernel_work(name, w, taps, vox_launch)
        kern.append({"name": name, "launches": n, "ms_per_launch": ms / max(n, 1), "share": ms / max(ms_prof_total, 1e-9),
                     "flops": fl, "bytes": by})
    kern.sort(key=lambda k: -k["share"])
    roofline = None
    if kern:
        k0 = kern[0]
        t_alu = k0["flops"] / (alu_peak * 1e12)
        t_hbm = k0["bytes"] / (hbm_peak * 1e9)
        sec = k0["ms_per_launch"] * 1e-3
        if t_alu >= t_hbm:
            ach = k0["flops"] / sec / 1e12
            roofline = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak}
        else:
            ach = k0["bytes"] / sec / 1e9
            roofline = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak}
        roofline.update({"kernel": k0["name"], "ms_per_launch": k0["ms_per_launch"], "share_of_step": k0["share"],
                         "algorithmic_flops": k0["flops"], "algorithmic_bytes": k0["bytes"],
                         "traffic": _dram_traffic(w.name, k0["name"]),
                         "peak_source": ("148 SM x 128 lanes x 2 x sm_max_mhz" if t_alu >= t_hbm else peaks["source"]),
                         "timed": "per-launch CUDA events in a separate pass of %d steps (%.3f ms per step with the "
                                  "events on; the headline loop runs with them off)" % (psteps, ms_prof_total / psteps)})
    out["roofline"] = roofline
    def _entry(k):
        # every kernel against its own roofline (algorithmic work as _kernel_work counts it) and, where the committed
        # ncu launch list has it, the DRAM bytes it really moved as a fraction of the HBM peak
        sec = max(k["ms_per_launch"] * 1e-3, 1e-12)
        f_alu = k["flops"] / sec / 1e12 / alu_peak
        f_hbm = k["bytes"] / sec / 1e9 / hbm_peak
        tr = _dram_traffic(w.name, k["name"])
        e = {"name": k["name"], "launches": k["launches"], "ms_per_launch": round(k["ms_per_launch"], 4),
             "share": round(k["share"], 4), "bound": "alu" if f_alu >= f_hbm else "hbm",
             "frac": round(max(f_alu, f_hbm), 4)}
        if tr is not None:
            e["traffic_frac_of_hbm_peak"] = round(tr / sec / 1e9 / hbm_peak, 4)
        return e
    out["kernels"] = [_entry(k) for k in kern]
    if roofline is not None and roofline.get("traffic"):
        roofline["traffic_frac_of_hbm_peak"] = roofline["traffic"] / (roofline["ms_per_launch"] * 1e-3) / 1e9 / hbm_peak

    # ---- SURVEY.md 8(d) metric (i): per scale, N / (t_filter3d + t_local_threshold) through the per-scale calls
    per_scale = []
    for s_i in range(S):
        times = []
        for which in ("filter3d", "local_threshold"):
            best = None
            for rep in range(3):                     # first repetition = warm-up
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                if which == "filter3d":
                    plan.pgsf_filter3d(s_i, d, d_out=filt[s_i], stream=stream)
                else:
                    plan.pgsf_local_threshold(filt[s_i], d_mask=mask, want_count=False, stream=stream)
                b.record(stream)
                torch.cuda.synchronize()
                if rep:
                    t = a.elapsed_time(b)
                    best = t if best is None else min(best, t)
            times.append(best)
        t_sum = max_over_ranks(times[0] + times[1], world, dev)
        per_scale.append({"sigma": list(w.sigmas[s_i]), "ms_filter3d": round(times[0], 4),
                          "ms_local_threshold": round(times[1], 4),
                          "gvoxel_per_s": n_vox * world / (t_sum * 1e-3) / 1e9})
    out["per_scale"] = per_scale

    # ---- NEXT-4: the mask of the last step merged into objects (26-connected components), timed on its own
    try:
        labels = torch.empty(d.shape, dtype=torch.int32, device=dev)
        best = None
        for rep in range(3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            _, nobj = plan.pgsf_label_objects(mask, d_labels=labels, stream=stream)
            b.record(stream)
            torch.cuda.synchronize()
            if rep:
                t = a.elapsed_time(b)
                best = t if best is None else min(best, t)
        out["label_objects"] = {"ms": round(best, 4), "objects": int(nobj.item()), "set_voxels": count,
                                "what": "pgsf_label_objects on the step's OR mask (not part of the timed step)"}
        del labels
    except Exception as exc:                      # (an extra leg must never cost the headline line)
        out["label_objects"] = {"error": str(exc)}
    return out, ctx


def run_b200(args, w):
    import torch
    import torch.distributed as dist
    from paper_1507_04941_b200 import binding, build

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a B200: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    binding.load_library()
    props = torch.cuda.get_device_properties(local_rank)
    peaks = _peaks()
    res, ctx = measure_workload(w, dev, local_rank, rank, world, args.steps, args.warmup, peaks,
                                props.multi_processor_count)
    n_vox, S = w.voxels, len(w.sigmas)
    line = {
        "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": w.name, "dims_xyz": list(w.dims), "batch": w.batch, "halo": list(w.halo),
                   "sigmas": [list(s) for s in w.sigmas], "box_half": list(w.box_half), "k": w.k,
                   "voxels": n_vox, "scales": S, "filtered_cubes_kept": True, "count": res["count"],
                   "l2": "inputs larger than L2 (input %.1f GiB, outputs %.1f GiB per step)" % (
                       n_vox * 4 / 2**30, n_vox * (4 * S + 1) / 2**30),
                   "timing": "CUDA events on the launching stream around the K steps; per-launch profiling events off",
                   "kernel_path": ctx["plan"].pgsf_plan_path()[1],
                   "parallelism": "replicas only (no collective)"},
        "clocks": res["clocks"], "gpu_launches": res["launches"], "roofline": res["roofline"],
        "path_roofline": res["path_roofline"], "kernels": res["kernels"], "per_scale": res["per_scale"], "label_objects": res.get("label_objects"),
    }
    ctx["peaks"], ctx["sm_count"], ctx["local_rank"] = peaks, props.multi_processor_count, local_rank
    return line, ctx


def run_other_configs(args, main_w, ctx):
    """ms per step and path-roofline fraction of the other BASELINE.json configs, measured in this same invocation
    after the headline (buffers allocated and freed per config; K <= 5 steps, no kernel table)."""
    import gc
    import torch
    from paper_1507_04941_b200 import synth
    out = []
    for c in sorted(synth.WORKLOADS):
        w = synth.WORKLOADS[c]
        if w.name == main_w.name:
            continue
        gc.collect()
        torch.cuda.empty_cache()
        res, c2 = measure_workload(w, ctx["dev"], ctx["local_rank"], 0, 1, max(1, min(args.steps, 5)), 3, ctx["peaks"],
                                   ctx["sm_count"], detail=False)
        c2["plan"].close()
        pr = res["path_roofline"]
        out.append({"workload": w.name, "ms_per_step": res["ms_per_step"], "value": res["value"], "unit": UNIT,
                    "count": res["count"], "gpu_launches": res["launches"], "roofline_ms": pr["roofline_ms"],
                    "path_frac": pr["frac"], "bound": pr["bound"], "sm_mhz": res["clocks"].get("sm_mhz"),
                    "reasons": res["clocks"].get("reasons")})
        del c2, res
    gc.collect()
    torch.cuda.empty_cache()
    return out


def run_e2e(args, w, ctx):
    """Same metric through pgsf_find_multiscale_host: HOST (pinned) buffers in and out, the
    host->device copy of the cube and the device->host copy of mask + count inside the timed region."""
    import torch
    import torch.distributed as dist
    plan, d, world, dev = ctx["plan"], ctx["d"], ctx["world"], ctx["dev"]
    S = len(w.sigmas)
    h_in = torch.empty(d.shape, dtype=torch.float32, pin_memory=True)
    h_in.copy_(d)
    expect = int(ctx["cnt"].item())
    # free the device-resident buffers of the first leg: the host entry point owns its own staging
    ctx["filt"].clear()
    ctx["d"] = None
    del d
    plan._ws = None
    torch.cuda.empty_cache()
    h_mask = torch.empty(h_in.shape, dtype=torch.uint8, pin_memory=True)
    steps = max(1, min(args.steps, 5))
    count = 0
    for _ in range(min(args.warmup, 2)):
        _, count = plan.pgsf_find_multiscale_host(h_in, h_mask)
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        _, count = plan.pgsf_find_multiscale_host(h_in, h_mask)   # synchronises before returning
    torch.cuda.synchronize()
    sec = (time.perf_counter() - t0) / steps
    sec = max_over_ranks(sec, world, dev)
    assert count == expect, f"host entry point count {count} != device path count {expect}"
    return {"value": w.voxels * S * world / sec / 1e9, "unit": UNIT, "ms_per_step": sec * 1e3, "steps": steps,
            "h2d_bytes_per_step": w.voxels * 4, "d2h_bytes_per_step": w.voxels + 8,
            "api": "pgsf_find_multiscale_host (pinned host cube in; mask + count out; streamed in z sections, copies overlapped with compute)"}


CPU_SAMPLE_1T = (128, 128, 128)    # the 1-thread leg: a smaller brick of the same cube (~10 s)


def run_cpu_baseline(w, sub, a, lo, hi, d_full=None):
    """The oracle as it stands on the box's host cores: all cores (OpenMP) on the sample brick and, per
    SURVEY.md 8(d), one thread on a smaller brick of the same cube."""
    from oracle import pgsf_oracle
    sec, vs, threads = time_oracle(w, sub, a, lo, hi)
    out = {"value": vs / sec / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": sec,
           "sample": _sample_text(w, lo, hi)}
    if d_full is not None:
        lo1, hi1 = _oracle_sample_region(w, CPU_SAMPLE_1T)
        a1, e1 = pgsf_oracle.required_input_box(w.dims, w.sigmas, w.box_half, lo1, hi1, w.truncate)
        sub1 = d_full[a1[2] - a[2]:e1[2] - a[2], a1[1] - a[1]:e1[1] - a[1], a1[0] - a[0]:e1[0] - a[0]]
        pgsf_oracle.set_threads(1)
        t0 = time.perf_counter()
        pgsf_oracle.find_region(sub1, a1, w.dims, w.sigmas, w.box_half, w.k, lo1, hi1, w.halo, w.truncate)
        dt = time.perf_counter() - t0
        pgsf_oracle.set_threads(0)
        vs1 = (hi1[0] - lo1[0]) * (hi1[1] - lo1[1]) * (hi1[2] - lo1[2]) * len(w.sigmas)
        out["single_thread"] = {"value": vs1 / dt / 1e9, "unit": UNIT, "cores": 1, "seconds": dt,
                                "sample": _sample_text(w, lo1, hi1)}
    return out


# ------------------------------------------------------------------------------------ Eq. 1 (weighted), NEXT-1

W_METRIC = "Gvoxel/s per Gaussian scale (weighted filter, Eq. 1)"
W_SAMPLE = (128, 128, 256)


def run_weighted(args, w):
    """--path weighted: one step = pgsf_filter3d_weighted (denominator as printed) for every scale of the
    config over its cube; single GPU.  Same JSON contract as the main path."""
    import torch
    from paper_1507_04941_b200 import binding, build, synth
    from oracle import pgsf_oracle
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a B200: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    build.build()
    binding.load_library()
    props = torch.cuda.get_device_properties(0)
    peaks = _peaks()
    d = synth.make_workload(w, "cuda:0")
    g = torch.Generator(device="cuda:0").manual_seed(w.seed + 5000)
    wt = torch.empty_like(d).uniform_(0.25, 2.0, generator=g)
    S = len(w.sigmas)
    taps = _taps(w)
    cube = w.dims[0] * w.dims[1] * w.dims[2]
    plan = binding.Plan(w.dims, w.sigmas, w.box_half, w.k, batch=w.batch, halo=w.halo, truncate=w.truncate)
    out = torch.empty_like(d)
    stream = torch.cuda.current_stream()

    def step():
        for s in range(S):
            plan.pgsf_filter3d_weighted(s, d, wt, binding.PGSF_WEIGHTED_AS_PRINTED, d_out=out, stream=stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    plan.pgsf_plan_set_profiling(True)
    l0 = plan.pgsf_plan_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    ms_step = ev0.elapsed_time(ev1) / args.steps
    launches = plan.pgsf_plan_launch_count() - l0
    prof = plan.pgsf_plan_profile()
    plan.pgsf_plan_set_profiling(False)
    clocks = sampler.stop()
    alu_peak = _alu_peak_tflops(props.multi_processor_count, peaks["sm_max_mhz"])
    hbm_peak = peaks["hbm_gbs"]
    kern = []
    for name, (n, ms) in prof.items():
        fl, by = _kernel_work(name, w, taps, cube)
        kern.append({"name": name, "launches": n, "ms_per_launch": ms / max(n, 1),
                     "share": ms / max(ms_step * args.steps, 1e-9), "flops": fl, "bytes": by})
    kern.sort(key=lambda k: -k["share"])
    k0 = kern[0]
    t_alu, t_hbm = k0["flops"] / (alu_peak * 1e12), k0["bytes"] / (hbm_peak * 1e9)
    sec = k0["ms_per_launch"] * 1e-3
    if t_alu >= t_hbm:
        ach = k0["flops"] / sec / 1e12
        roofline = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak}
    else:
        ach = k0["bytes"] / sec / 1e9
        roofline = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak}
    roofline.update({"kernel": k0["name"], "ms_per_launch": k0["ms_per_launch"], "share_of_step": k0["share"],
                     "traffic": None})
    n_vox = w.voxels
    path_flops = sum(2 * sum(t) + 8 for t in taps) * n_vox
    path_bytes = 12 * S * n_vox
    t_path = max(path_flops / (alu_peak * 1e12), path_bytes / (hbm_peak * 1e9))
    # end to end: pinned host cubes in, every scale's result out
    e2e = None
    if not args.no_e2e:
        h_d = torch.empty(d.shape, dtype=torch.float32, pin_memory=True).copy_(d)
        h_w = torch.empty(d.shape, dtype=torch.float32, pin_memory=True).copy_(wt)
        h_o = torch.empty(d.shape, dtype=torch.float32, pin_memory=True)
        steps = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(steps):
            d.copy_(h_d, non_blocking=True)
            wt.copy_(h_w, non_blocking=True)
            for s in range(S):
                plan.pgsf_filter3d_weighted(s, d, wt, binding.PGSF_WEIGHTED_AS_PRINTED, d_out=out, stream=stream)
                h_o.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        sec_e = (time.perf_counter() - t0) / steps
        e2e = {"value": n_vox * S / sec_e / 1e9, "unit": UNIT, "ms_per_step": sec_e * 1e3, "steps": steps,
               "h2d_bytes_per_step": 8 * n_vox, "d2h_bytes_per_step": 4 * n_vox * S,
               "api": "binding.Plan.pgsf_filter3d_weighted on pinned host cubes (torch copies)"}
    cpu = None
    if not args.no_cpu_baseline:
        lo = [max(0, (n - sz) // 2) for n, sz in zip(w.dims, W_SAMPLE)]
        hi = [min(n, l + sz) for n, l, sz in zip(w.dims, lo, W_SAMPLE)]
        sd = d[0, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]].cpu().numpy()
        sw = wt[0, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]].cpu().numpy()
        plan.close()
        threads = pgsf_oracle.set_threads(0)
        t0 = time.perf_counter()
        for sg in w.sigmas:
            pgsf_oracle.wfilter_full(sd, sw, sg, 0, w.truncate)
        dt = time.perf_counter() - t0
        cpu = {"value": sd.size * S / dt / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": dt,
               "sample": f"centred brick {sd.shape[2]}x{sd.shape[1]}x{sd.shape[0]} of {w.name} taken as a "
                         f"standalone cube, all {S} scales, oracle Eq. 1 (L1 separable, fp64)"}
    line = {"metric": W_METRIC, "value": n_vox * S / (ms_step * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "path": "weighted (Eq. 1, denominator as printed)",
                       "weights": "U(0.25, 2) fp32, seeded", "scales": S,
                       "l2": "inputs larger than L2" if n_vox * 4 > 2**28 else "inputs fit L2 (small config)"},
            "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline,
            "path_roofline": {"flops_per_voxel": path_flops / n_vox, "bytes_per_voxel": path_bytes / n_vox,
                              "roofline_ms": t_path * 1e3, "frac": t_path * 1e3 / ms_step},
            "kernels": [{"name": k["name"], "launches": k["launches"], "ms_per_launch": round(k["ms_per_launch"], 4),
                         "share": round(k["share"], 4)} for k in kern],
            "e2e": e2e, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ Eq. 2 direct (NEXT-2)

D_METRIC = "Gvoxel/s (direct 3-D filter, Eq. 2, arbitrary taps)"
D_SAMPLE = (96, 96, 96)


def run_direct(args, w):
    """--path direct: one step = pgsf_filter3d_direct over the config's cube with the (2rz+1)(2ry+1)(2rx+1)
    taps of its FIRST scale as a general filter array (fp32 accumulation; --fp64 for the paper's fp64).
    Single GPU.  Same JSON contract as the main path."""
    import numpy as np
    import torch
    from paper_1507_04941_b200 import binding, build, synth
    from oracle import pgsf_oracle
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a B200: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    build.build()
    binding.load_library()
    props = torch.cuda.get_device_properties(0)
    peaks = _peaks()
    d = synth.make_workload(w, "cuda:0")
    g = [pgsf_oracle.taps(sg, w.truncate) for sg in w.sigmas[0]]
    f = (g[2][:, None, None] * g[1][None, :, None] * g[0][None, None, :]).astype(np.float32)
    d_f = torch.from_numpy(f).cuda()
    ntaps = f.size
    plan = binding.Plan(w.dims, w.sigmas, w.box_half, w.k, batch=w.batch, halo=w.halo, truncate=w.truncate)
    out = torch.empty_like(d)
    stream = torch.cuda.current_stream()
    step = lambda: plan.pgsf_filter3d_direct(d_f, d, fp64_accum=args.fp64, d_out=out, stream=stream)
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    l0 = plan.pgsf_plan_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    ms_step = ev0.elapsed_time(ev1) / args.steps
    launches = plan.pgsf_plan_launch_count() - l0
    clocks = sampler.stop()
    n_vox = w.voxels
    alu_peak = _alu_peak_tflops(props.multi_processor_count, peaks["sm_max_mhz"]) * (0.5 if args.fp64 else 1.0)
    flops = 2.0 * ntaps * n_vox
    ach = flops / (ms_step * 1e-3) / 1e12
    roofline = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
                "kernel": "direct_f64" if args.fp64 else "direct_f32", "ms_per_launch": ms_step / max(w.batch, 1),
                "share_of_step": 1.0, "traffic": None,
                "peak_source": "148 SM x 128 lanes x 2 x sm_max_mhz" + (" / 2 (fp64)" if args.fp64 else "")}
    e2e = None
    if not args.no_e2e:
        h_d = torch.empty(d.shape, dtype=torch.float32, pin_memory=True).copy_(d)
        h_o = torch.empty(d.shape, dtype=torch.float32, pin_memory=True)
        steps = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(steps):
            d.copy_(h_d, non_blocking=True)
            step()
            h_o.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        sec_e = (time.perf_counter() - t0) / steps
        e2e = {"value": n_vox / sec_e / 1e9, "unit": "Gvoxel/s", "ms_per_step": sec_e * 1e3, "steps": steps,
               "h2d_bytes_per_step": 4 * n_vox, "d2h_bytes_per_step": 4 * n_vox,
               "api": "binding.Plan.pgsf_filter3d_direct on a pinned host cube (torch copies)"}
    cpu = None
    if not args.no_cpu_baseline:
        lo = [max(0, (n - sz) // 2) for n, sz in zip(w.dims, D_SAMPLE)]
        hi = [min(n, l + sz) for n, l, sz in zip(w.dims, lo, D_SAMPLE)]
        sd = d[0, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]].cpu().numpy()
        plan.close()
        threads = pgsf_oracle.set_threads(0)
        t0 = time.perf_counter()
        pgsf_oracle.filter_general(sd, f.astype(np.float64))
        dt = time.perf_counter() - t0
        cpu = {"value": sd.size / dt / 1e9, "unit": "Gvoxel/s", "cores": threads, "kind": "oracle", "seconds": dt,
               "sample": f"centred brick {sd.shape[2]}x{sd.shape[1]}x{sd.shape[0]} of {w.name} taken as a standalone "
                         f"cube, the same {ntaps} taps, oracle Eq. 2 by direct loops (fp64)"}
    line = {"metric": D_METRIC, "value": n_vox / (ms_step * 1e-3) / 1e9, "unit": "Gvoxel/s", "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.fp64 else "f32", "data": "synthetic",
            "config": {"workload": w.name, "path": "direct (Eq. 2, arbitrary filter array)",
                       "filter_extent_xyz": [f.shape[2], f.shape[1], f.shape[0]], "taps": int(ntaps),
                       "l2": "inputs larger than L2" if n_vox * 4 > 2**28 else "inputs fit L2 (small config)"},
            "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline,
            "path_roofline": {"flops_per_voxel": 2.0 * ntaps, "bytes_per_voxel": 8.0,
                              "roofline_ms": flops / (alu_peak * 1e12) * 1e3,
                              "frac": flops / (alu_peak * 1e12) * 1e3 / ms_step},
            "e2e": e2e, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config (1-based); default 3 = the 8 GiB cube the north star is quoted on")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--path", default="find", choices=["find", "weighted", "direct"],
                    help="find = the hot path (default); weighted = Eq. 1 of the paper (NEXT-1); direct = Eq. 2 for "
                         "an arbitrary filter array (NEXT-2); the last two single GPU")
    ap.add_argument("--fp64", action="store_true", help="--path direct: accumulate in fp64 as the paper does")
    ap.add_argument("--flags", type=int, default=0, help="plan flags (8 = PGSF_FLAG_TENSOR_ZPASS, the optional variant)")
    ap.add_argument("--tune", type=int, default=0, help="PGSF_OPT_TUNE bits (kernel variants; same results)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the ms-per-step sweep over the other BASELINE.json configs after the headline")
    args = ap.parse_args()
    global TUNE, FLAGS
    TUNE = args.tune
    FLAGS = args.flags
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    from paper_1507_04941_b200 import synth
    w = synth.WORKLOADS[args.config]
    if args.impl == "reference":
        run_reference(args, w)
        return
    if args.path in ("weighted", "direct"):
        if int(os.environ.get("RANK", "0")) == 0:
            (run_weighted if args.path == "weighted" else run_direct)(args, w)
        return
    line, ctx = run_b200(args, w)
    rank, world = ctx["rank"], ctx["world"]
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import pgsf_oracle
        lo, hi = _oracle_sample_region(w)
        a, e = pgsf_oracle.required_input_box(w.dims, w.sigmas, w.box_half, lo, hi, w.truncate)
        sub = ctx["d"][0, a[2]:e[2], a[1]:e[1], a[0]:e[0]].cpu().numpy()
    if not args.no_e2e:
        line["e2e"] = run_e2e(args, w, ctx)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ctx["plan"].close()
        cpu = run_cpu_baseline(w, sub, a, lo, hi, d_full=sub)
    line["cpu_baseline"] = cpu
    if rank == 0 and world == 1 and not args.no_other_configs:
        ctx["plan"].close()
        for k in ("d", "filt", "mask", "cnt"):
            ctx[k] = None
        line["other_configs"] = run_other_configs(args, w, ctx)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
