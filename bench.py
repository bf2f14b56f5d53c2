#!/usr/bin/env python
"""bench.py -- PSF voxels/s of the hot path (pupil producer -> row DFT -> column DFT -> |E|^2) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl ours|reference]

One "step" is one psf_compute over the whole workload (all planes / emitters).  Prints ONE JSON line (rank 0).
See DESIGN.md §7 for what every key means and how the roofline figures are derived.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import psf_workloads as W  # noqa: E402

METRIC = "psf_voxels_per_s"
UNIT = "voxels/s"
WORKLOADS = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}
SM_COUNT, FMA_LANES_PER_SM = 148, 128
TF32_OVER_BF16 = 1.1 / 2.25            # nominal dense ratio (B200_PROFILING.md table)
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}
# dram__bytes_read.sum + dram__bytes_write.sum per launch come from the committed ncu captures: profiles/traffic.csv has one
# row per (workload, kernel) with the capture it was read from (profiles/traffic.md names the commands).  A row is used only
# when its kernel is one the running plan launches (psf_kernel_names); otherwise `traffic` is null.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "traffic.csv")


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            d["_source"] = "measured"
            return d
        except Exception:
            pass
    d = dict(FALLBACK_PEAKS)
    d["_source"] = "fallback"
    return d


def load_traffic():
    rows = {}
    try:
        import csv
        with open(TRAFFIC_CSV) as f:
            for r in csv.DictReader(f):
                rows[(r["workload"], r["kernel"])] = r
    except Exception:
        pass
    return rows


def traffic_for(rows, case, kernel, planes_per_launch):
    """(bytes per launch, source) for `kernel` on this workload, scaled from the captured launch's plane count; (None, why)
    if no committed capture covers it."""
    r = rows.get((case.name, kernel))
    if r is None:
        return None, f"no ncu capture of {kernel} on {case.name} in profiles/traffic.csv"
    per_plane = (float(r["dram_read_bytes"]) + float(r["dram_write_bytes"])) / float(r["planes_in_launch"])
    return per_plane * planes_per_launch, f"profiles/{r['capture']} (ncu --set full, commit {r['commit']})"


def ffma_peak_tflops(peaks):
    return SM_COUNT * FMA_LANES_PER_SM * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12


def roofline_record(case, res, ms_per_step, peaks, traffic_rows):
    """Roofline of the dominant kernel of one timed workload: achieved = executed flop per launch / mean
    launch duration (CUDA events around every launch on the compute stream, psf_profile_*)."""
    f1, f2 = folded_flops(case)
    stage_ms = res["stage_ms"]
    path = res["path"]
    kernels = res["kernels"]
    fused = path in ("ffma_fused", "fused_tc3xf16") or kernels == ["k12_fused"]      # one kernel does the whole path
    dom = 0 if fused else int(np.argmax(stage_ms[:2]))
    flop_dom = (f1 + f2) if fused else (f1, f2)[dom]
    launches_dom = max(int(res["stage_launches"][dom]), 1)
    dur_ms = stage_ms[dom] / launches_dom
    if path in ("ffma", "ffma_fused", "fused_tc3xf16"):
        bound = "alu"
        peak = ffma_peak_tflops(peaks)
        executed = flop_dom
        peak_note = f"148 SM x 128 FFMA lanes x 2 flop x {peaks.get('sm_max_mhz', 1965.0):.0f} MHz (fp32 FFMA pipe)"
        if path == "fused_tc3xf16":
            # the emitter-batch tensor kernel: its contractions run on tcgen05 (the pipe is ~20 % busy), the kernel is bound by
            # the ALU work that generates, splits and publishes the operands; the fp32-equivalent flop rate is kept against the
            # same FFMA peak as the fp32 kernel it replaces so that the two are comparable
            peak_note += "; fp32-equivalent folded flop of the two DFT stages (executed as 3 fp16 products on tcgen05)"
    else:
        bound = "tensor"
        long_step = ms_per_step > 1000.0
        bf16 = peaks["bf16_tflops_sustained"] if long_step else peaks["bf16_tflops"]
        which = f"{peaks['_source']} bf16 {'sustained' if long_step else 'burst'} {bf16:.1f} TF/s"
        executed = 3.0 * flop_dom
        if path == "tc3xf16":      # kind::f16 runs at the bf16 rate: the measured cuBLAS bf16 figure is the peak itself
            peak = bf16
            peak_note = f"{which} (fp16 = bf16 tensor rate); achieved counts executed FP16 flop (3 products per fp32 product)"
        else:
            peak = bf16 * TF32_OVER_BF16
            peak_note = (f"{which} x nominal tf32/bf16 ratio {TF32_OVER_BF16:.3f}; achieved counts executed TF32 flop "
                         f"(3 products per fp32 product)")
    achieved = executed / launches_dom / (dur_ms * 1e-3) / 1e12
    kname = kernels[min(dom, len(kernels) - 1)] if kernels else "?"
    traffic, tsrc = traffic_for(traffic_rows, case, kname, case.n_planes / launches_dom)
    out_bytes = 4.0 * case.voxels()
    roofline = {"bound": bound, "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": tsrc, "kernel": kname,
                "kernel_role": "whole path (fused)" if fused else ("stage1_rowdft_producer", "stage2_coldft_intensity")[dom],
                "kernel_ms_per_launch": dur_ms, "launches_per_step": launches_dom,
                "algorithmic_tflops": flop_dom / launches_dom / (dur_ms * 1e-3) / 1e12, "peak_source": peak_note,
                "stage_ms_per_step": [float(stage_ms[0]), float(stage_ms[1])],
                "kernel_times_from": res.get("profile_pass"),
                # compulsory HBM traffic = the intensity stack: reported for every workload, the binding
                # bound only where the flop are few (the small-M batched regime)
                "hbm_gbs": out_bytes / (ms_per_step * 1e-3) / 1e9,
                "hbm_frac": out_bytes / (ms_per_step * 1e-3) / 1e9 / peaks["hbm_gbs"]}
    total_flop = f1 + f2
    roofline["step_frac"] = (3.0 if bound == "tensor" else 1.0) * total_flop / (ms_per_step * 1e-3) / 1e12 / peak
    return roofline


def rank_case(cfg: int, rank: int):
    """Weak scaling: every rank owns a full-size shard of a longer stack (rank r: z shifted by r * 10 nm; the
    emitter batch of config 4 is redrawn with another z offset).  No data-path collective."""
    case = W.get_config(cfg)
    if rank:
        from dataclasses import replace
        case = replace(case, z_um=case.z_um + 0.010 * rank)
    return case


def folded_flops(case):
    """Algorithmic real flop of the two DFT stages in the folded formulation:
    stage 1 = C Z 8 chains 2 n^2 m, stage 2 = C Z 8 chains 2 m^2 n; n = ceil(N/2), m = ceil(M/2)."""
    n, m = (case.pupil_n + 1) // 2, (case.out_m + 1) // 2
    C = 1 if getattr(case, "model", "vectorial") == "scalar" else (5 if case.pol == "unpolarized" else 3)
    Z = case.n_planes
    return C * Z * 16.0 * n * n * m, C * Z * 16.0 * m * m * n


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v == "Active":
                    reasons.add(nme)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def time_workload(torch, psf, case, device, steps, warmup, flush, profile=True):
    """Device-timed steps: per step L2 flush (untimed), event, psf_compute, event.  Returns dict."""
    plan = psf.plan_from_case(case, device=device)
    dev = torch.device("cuda", device)
    out = torch.empty((case.n_planes, case.out_m, case.out_m), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev)
    # Per-kernel durations come from psf_profile_enable (an event record behind every launch).  On a one-kernel path that is
    # free, so the timed steps carry it; on a two-kernel path the record sits between the kernels (and switches the
    # programmatic dependent launch of stage 2 off), so the steps are timed without it and a second pass of the same
    # steps, profiled, gives the split.
    multi = plan.launches_per_compute > 1
    inline = profile and not multi
    if inline:
        plan.profile_enable(True)
    for _ in range(warmup):
        plan.compute(out)
    torch.cuda.synchronize(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    stage_ms = np.zeros(4)
    stage_launches = np.zeros(4, dtype=np.int64)
    for i in range(steps):
        flush.fill_(float(i % 251))                    # > L2: evicts tables, scratch and outputs of the previous step
        ev[i][0].record(stream)
        plan.compute(out)
        ev[i][1].record(stream)
        if inline:
            torch.cuda.synchronize(dev)
            ms, ln = plan.profile_read()
            stage_ms += np.array(ms)
            stage_launches += np.array(ln)
    torch.cuda.synchronize(dev)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    psteps = steps
    if profile and multi:
        psteps = min(steps, 10)
        plan.profile_enable(True)
        plan.compute(out)
        for i in range(psteps):
            flush.fill_(float(i % 251))
            plan.compute(out)
            torch.cuda.synchronize(dev)
            ms, ln = plan.profile_read()
            stage_ms += np.array(ms)
            stage_launches += np.array(ln)
        plan.profile_enable(False)
    steps = psteps
    res = {"plan": plan, "out": out, "step_ms": step_ms, "stage_ms": stage_ms / max(steps, 1),
           "stage_launches": stage_launches // max(steps, 1), "path": plan.path,
           "launches": plan.launches_per_compute, "kernels": plan.kernel_names,
           "profile_pass": "none" if not profile else ("separate pass of %d profiled steps behind the timed steps" % psteps if multi
                                                        else "inside the timed steps")}
    return res


def loop_ms_per_call(torch, plan, out, device, calls=100):
    """a tiny stack is timed as a back-to-back loop as well (no flush between calls: launch rate)."""
    dev = torch.device("cuda", device)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(5):
        plan.compute(out)
    torch.cuda.synchronize(dev)
    a.record()
    for _ in range(calls):
        plan.compute(out)
    b.record()
    torch.cuda.synchronize(dev)
    return a.elapsed_time(b) / calls


def e2e_workload(torch, plan, case, device, steps, warmup):
    """End to end through the public API with HOST buffers: per step, host Zernike coefficients / shifts go in through
    psf_set_zernike / psf_set_shifts (host->device table refresh), psf_compute runs, and the intensity stack is copied
    device->host into pinned memory.  Wall clock around the whole step."""
    dev = torch.device("cuda", device)
    out = torch.empty((case.n_planes, case.out_m, case.out_m), dtype=torch.float32, device=dev)
    host = torch.empty(out.shape, dtype=torch.float32, pin_memory=True)
    h2d = 0
    times, refresh = [], []
    for i in range(warmup + steps):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        plan.set_zernike(case.zernike, case.noll_first)
        if i >= warmup:
            refresh.append(time.perf_counter() - t0)
        h2d = plan.last_upload_bytes
        if case.shifts_um is not None:
            plan.set_shifts(case.shifts_um)
            h2d = plan.last_upload_bytes + (case.zernike.nbytes if case.zernike is not None else 0)
        plan.compute(out)
        host.copy_(out, non_blocking=True)
        torch.cuda.synchronize(dev)
        t1 = time.perf_counter()
        if i >= warmup:
            times.append(t1 - t0)
    # the same steps streamed: the device->host copy of step i runs on a copy stream into the other of two pinned buffers
    # while the host refreshes the tables of step i+1 and its kernels run (what a caller that wants throughput does)
    outs = [out, torch.empty_like(out)]
    hosts = [host, torch.empty(out.shape, dtype=torch.float32, pin_memory=True)]
    copy_stream = torch.cuda.Stream(dev)
    done = [torch.cuda.Event(), torch.cuda.Event()]
    copied = [torch.cuda.Event(), torch.cuda.Event()]
    main = torch.cuda.current_stream(dev)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for i in range(steps):
        k = i & 1
        plan.set_zernike(case.zernike, case.noll_first)
        if case.shifts_um is not None:
            plan.set_shifts(case.shifts_um)
        if i >= 2:
            main.wait_event(copied[k])            # the copy of step i-2 has left this output buffer
        plan.compute(outs[k])
        done[k].record(main)
        with torch.cuda.stream(copy_stream):
            copy_stream.wait_event(done[k])
            hosts[k].copy_(outs[k], non_blocking=True)
            copied[k].record(copy_stream)
    torch.cuda.synchronize(dev)
    piped = (time.perf_counter() - t0) / steps
    return {"s_per_step": statistics.mean(times), "s_per_step_streamed": piped, "h2d": int(h2d), "d2h": int(out.numel() * 4),
            "set_zernike_ms": 1e3 * statistics.median(refresh), "checksum": float(host.double().sum())}


def oracle_sample(case, budget_planes):
    """A bounded, evenly spaced sample of planes for the CPU baseline."""
    Z = case.n_planes
    k = max(1, min(Z, budget_planes))
    return np.unique(np.linspace(0, Z - 1, k).round().astype(int))


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [i.get("num_threads", 0) for i in threadpool_info() if i.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


ORACLE_PLANES = {1: 16, 2: 64, 3: 128, 4: 4096, 5: 256}    # about 10-30 s of CPU work each on the 16-core B200 host
ORACLE_PLANES_SWEEP = {1: 16, 2: 64, 3: 32, 4: 4096, 5: 32}    # per-workload lines of the sweep: configs 1, 2, 4 in full


def run_oracle_once(case, planes):
    from oracle import psf_oracle as O
    t0 = time.perf_counter()
    I = O.stack_T2(case, planes)
    dt = time.perf_counter() - t0
    return dt, I


def cpu_baseline(case, cfg, table=ORACLE_PLANES):
    planes = oracle_sample(case, table[cfg])
    dt, I = run_oracle_once(case, planes)
    vox = len(planes) * case.out_m * case.out_m
    return {"value": vox / dt, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
            "sample": f"oracle stack_T2 (fp64 separable direct sum, numpy) on {len(planes)} of {case.n_planes} "
                      f"planes of {case.name}, {dt:.2f} s wall"}


def run_reference(args):
    """--impl reference: the oracle as it stands, timed on the host cores, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = WORKLOADS[args.workload]
    case = W.get_config(cfg)
    planes = oracle_sample(case, max(1, ORACLE_PLANES[cfg] // 2))
    vox = len(planes) * case.out_m * case.out_m
    for _ in range(args.warmup):
        run_oracle_once(case, planes[:1])
    times = []
    for _ in range(args.steps):
        dt, _ = run_oracle_once(case, planes)
        times.append(dt)
    mean = statistics.mean(times)
    val = vox / mean
    sample = (f"each step = oracle stack_T2 on {len(planes)} of {case.n_planes} planes of {case.name} "
              f"({vox} voxels); value scales that to voxels/s")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": mean * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": case.name, "N": case.pupil_n, "M": case.out_m, "Z": case.n_planes,
                       "sample_planes": int(len(planes))},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    import paper_2502_03170_b200 as psf   # raises if the CUDA library is missing: no CPU fallback

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    peaks = load_peaks()
    cfg = WORKLOADS[args.workload]
    case = rank_case(cfg, rank)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # 256 MiB > 126 MB L2

    sampler = ClockSampler(local) if rank == 0 else None
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(dev)
    res = time_workload(torch, psf, case, local, args.steps, args.warmup, flush)
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop() if sampler else None

    total_ms = torch.tensor([sum(res["step_ms"])], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(total_ms.item()) / args.steps
    voxels = case.voxels() * world
    value = voxels / (ms_per_step * 1e-3)

    # end to end through the API with host buffers
    e2e = e2e_workload(torch, res["plan"], case, local, max(3, min(args.steps, 10)), 2)
    e2e_s = torch.tensor([e2e["s_per_step"]], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_val = voxels / float(e2e_s.item())

    # roofline of the dominant kernel
    traffic_rows = load_traffic()
    roofline = roofline_record(case, res, ms_per_step, peaks, traffic_rows)
    path = res["path"]
    step_sorted = sorted(res["step_ms"])

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"tc3xf16": "f16x3", "tc3xtf32": "tf32x3", "fused_tc3xf16": "f16x3"}.get(path, "f32"), "data": "synthetic",
            "config": {"workload": case.name, "N": case.pupil_n, "M": case.out_m, "Z": case.n_planes,
                       "pol": case.pol, "path": path, "kernels": res["kernels"],
                       "planes_per_s": case.n_planes * world / (ms_per_step * 1e-3),
                       "median_ms": float(statistics.median(step_sorted)), "min_ms": float(step_sorted[0]),
                       "l2": "256 MiB buffer written between timed iterations (flush)", "sharding": "z-shards, no collective"},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                    "streamed_value": voxels / world / e2e["s_per_step_streamed"] * world,
                    "set_zernike_ms": e2e["set_zernike_ms"],
                    "note": "value: each step serial (psf_set_zernike = coefficient upload + table refresh, on the device for "
                            "3xFP16 pair plans; kernels; device->host copy); "
                            "streamed_value: same steps with the copy of step i overlapping step i+1 (two pinned buffers)"},
            "gpu_launches": int(res["launches"]) * args.steps,
            "roofline": roofline}
    if path == "tc3xf16" and case.zernike is not None and case.shifts_um is None:
        # A/B of the table refresh: the same call with the device-side refresh switched off (host fp64 tables + upload)
        res["plan"].tune(psf.TUNE_DEVICE_REFRESH, 0)
        ts = []
        for _ in range(6):
            t0 = time.perf_counter()
            res["plan"].set_zernike(case.zernike, case.noll_first)
            ts.append(time.perf_counter() - t0)
        line["e2e"]["set_zernike_host_path_ms"] = 1e3 * statistics.median(ts[1:])
    res["plan"].destroy()

    if rank == 0 and world == 1:
        line["cpu_baseline"] = cpu_baseline(case, cfg)
        if not args.no_sweep:
            sweep = {}
            for name, c in WORKLOADS.items():
                if c == cfg:
                    sweep[name] = {"voxels_per_s": value, "ms_per_step": ms_per_step, "median_ms": float(statistics.median(step_sorted)),
                                   "min_ms": float(step_sorted[0]), "path": path, "kernels": res["kernels"], "roofline": roofline,
                                   "cpu_baseline": line["cpu_baseline"]}
                    continue
                cs = W.get_config(c)
                r = time_workload(torch, psf, cs, local, max(args.steps, 20), 3, flush)
                ms = statistics.mean(r["step_ms"])
                srt = sorted(r["step_ms"])
                sweep[name] = {"voxels_per_s": cs.voxels() / (ms * 1e-3), "planes_per_s": cs.n_planes / (ms * 1e-3),
                               "ms_per_step": ms, "median_ms": float(statistics.median(srt)), "min_ms": float(srt[0]),
                               "path": r["path"], "kernels": r["kernels"], "launches": r["launches"],
                               "roofline": roofline_record(cs, r, ms, peaks, traffic_rows),
                               "cpu_baseline": cpu_baseline(cs, c, ORACLE_PLANES_SWEEP)}
                if cs.shifts_um is not None and cs.zernike is not None and cs.zernike.ndim == 2:
                    # emitter batch: what new per-emitter coefficients and positions cost before the next psf_compute
                    tz, tsft = [], []
                    for _ in range(6):
                        t0 = time.perf_counter()
                        r["plan"].set_zernike(cs.zernike, cs.noll_first)
                        t1 = time.perf_counter()
                        r["plan"].set_shifts(cs.shifts_um)
                        tz.append(t1 - t0)
                        tsft.append(time.perf_counter() - t1)
                    sweep[name]["set_zernike_rows_ms"] = 1e3 * statistics.median(tz[1:])
                    sweep[name]["set_shifts_ms"] = 1e3 * statistics.median(tsft[1:])
                if c == 1:      # launch-rate view of the tiny stack: 100 calls back to back between two events
                    sweep[name]["loop100_ms_per_call"] = loop_ms_per_call(torch, r["plan"], r["out"], local)
                r["plan"].destroy()
            # the spherical (Bessel) path on the two axisymmetric configs: ALU / SFU bound, context only
            for name, c, nodes in (("cfg1_spherical", 1, 2001), ("cfg3_spherical", 3, 2001)):
                cs = W.get_config(c)
                plan = psf.plan_from_case(cs, device=local)
                out = torch.empty((cs.n_planes, cs.out_m, cs.out_m), dtype=torch.float32, device=dev)
                for _ in range(3):
                    plan.compute_spherical(nodes, out)
                torch.cuda.synchronize(dev)
                ts = []
                for i in range(min(args.steps, 10)):
                    flush.fill_(float(i % 251))
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    plan.compute_spherical(nodes, out)
                    b.record()
                    torch.cuda.synchronize(dev)
                    ts.append(a.elapsed_time(b))
                ms = statistics.mean(ts)
                m_half = (cs.out_m + 1) // 2
                radii = m_half * (m_half + 1) // 2
                sweep[name] = {"voxels_per_s": cs.voxels() / (ms * 1e-3), "ms_per_step": ms, "path": "spherical_bessel",
                               "simpson_nodes": nodes, "launches": 2,
                               "bessel_terms_per_s": radii * nodes * cs.n_planes / (ms * 1e-3)}
                plan.destroy()
            # the adjoint: gradients w.r.t. z_b and the Zernike coefficients for a random dL/dI; complex
            # fp32 FFMA products, so the roofline is the FFMA pipe
            for name, c in (("cfg2_gradients", 2), ("cfg5_gradients", 5)):
                cs = W.get_config(c)
                plan = psf.plan_from_case(cs, device=local)
                G = torch.randn((cs.n_planes, cs.out_m, cs.out_m), dtype=torch.float32, device=dev)
                K = cs.zernike.shape[-1]
                for _ in range(2):
                    plan.gradients(G, K)
                torch.cuda.synchronize(dev)
                ts = []
                for i in range(3):
                    flush.fill_(float(i % 251))
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    plan.gradients(G, K)
                    b.record()
                    torch.cuda.synchronize(dev)
                    ts.append(a.elapsed_time(b))
                ms = statistics.mean(ts)
                cg = 6 if cs.pol == "unpolarized" else 3
                flop = 2 * 8.0 * cs.pupil_n * cs.out_m * (cs.pupil_n + cs.out_m) * cg * cs.n_planes     # forward + back-projection
                ffma_peak = SM_COUNT * FMA_LANES_PER_SM * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
                sweep[name] = {"ms_per_step": ms, "planes_per_s": cs.n_planes / (ms * 1e-3), "path": plan.grad_path,
                               "fp32_equivalent_tflops": flop / (ms * 1e-3) / 1e12,
                               "frac_of_ffma_peak": (flop / (ms * 1e-3) / 1e12 / ffma_peak) if plan.grad_path == "adjoint_ffma" else None,
                               "note": "forward field + back-projection (the same tensor kernels on a plan with the grids swapped) + "
                                       "weight/fold and reduction kernels; fp32_equivalent_tflops counts the unfolded complex products",
                               "zernike_terms": int(K)}
                # one iteration of a fit: new shared coefficients in, stack and gradients out (wall clock, one sync at the end),
                # with the table refresh on the device (default) and on the host (PSF_TUNE_DEVICE_REFRESH = 0)
                out = torch.empty((cs.n_planes, cs.out_m, cs.out_m), dtype=torch.float32, device=dev)
                rng = np.random.default_rng(7)
                for mode, key in ((1, "fit_iteration_ms"), (0, "fit_iteration_host_refresh_ms")):
                    plan.tune(psf.TUNE_DEVICE_REFRESH, mode)
                    its = []
                    for i in range(2 + 5):
                        coef = (cs.zernike + 0.01 * rng.standard_normal(K)).astype(np.float32)
                        torch.cuda.synchronize(dev)
                        t0 = time.perf_counter()
                        plan.set_zernike(coef, cs.noll_first)
                        plan.compute(out)
                        plan.gradients(G, K)
                        torch.cuda.synchronize(dev)
                        its.append(time.perf_counter() - t0)
                    sweep[name][key] = 1e3 * statistics.median(its[2:])
                plan.destroy()
            line["workloads"] = sweep
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def time_calls(torch, fn, flush, calls=20, warmup=3):
    """Mean / min milliseconds of `calls` device-timed calls of fn(), L2 flushed before each."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ts = []
    for i in range(calls):
        flush.fill_(float(i % 251))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return statistics.mean(ts), min(ts)


def run_fig5(args):
    """--workload fig5: the paper's own benchmark shape (Fig. 5: one 201 x 201 plane at focus against the
    pupil size, all four propagators) on this build, and the matrix-vs-FFT crossover study of SURVEY 8(f) NEXT-4: the
    tensor-core product form against the chirp-Z / FFT form (PSF_PREC_CZT_FFT) at M = 201 and at M = N.  The paper prints no
    numbers for Fig. 5 (plot only) and its library defaults are not stated: config-1 optics, x-polarised input for the
    vectorial model, are used.  Context, not the headline metric."""
    import torch
    from dataclasses import replace
    import paper_2502_03170_b200 as psf
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    base = replace(W.config1(), out_m=201, z_um=np.array([0.0]), name="fig5_single_plane")
    sizes = [64, 128, 256, 512, 1024, 2048, 4096]
    sampler = ClockSampler(0)
    fig5, cross = [], []

    def timed(case, precision, spherical_nodes=0):
        plan = psf.plan_from_case(case, precision=precision)
        out = torch.empty((case.n_planes, case.out_m, case.out_m), dtype=torch.float32, device=dev)
        if spherical_nodes:
            mean, mn = time_calls(torch, lambda: plan.compute_spherical(spherical_nodes, out), flush)
            path = "spherical_bessel"
        else:
            mean, mn = time_calls(torch, lambda: plan.compute(out), flush)
            path = plan.path
        plan.destroy()
        return {"us_mean": mean * 1e3, "us_min": mn * 1e3, "path": path}

    for N in sizes:
        row = {"N": N, "M": 201}
        for model in ("vectorial", "scalar"):
            c = replace(base, pupil_n=N, model=model)
            row[model + "_cartesian"] = timed(c, "auto")
            row[model + "_cartesian_czt_fft"] = timed(c, "czt_fft")
            row[model + "_spherical"] = timed(c, "auto", spherical_nodes=N + 1)
        fig5.append(row)
    # crossover: stacks of 8 planes so that launch overhead does not hide the kernels; M = 201 and M = N
    z8 = np.linspace(-1.0, 1.0, 8)
    for N in [256, 512, 1024, 2048, 4096]:
        for M in (201, N):
            c = replace(base, pupil_n=N, out_m=M, z_um=z8, pixel_um=0.04 * 201 / M if M != 201 else 0.04)
            a, f = timed(c, "auto"), timed(c, "czt_fft")
            n, m = (N + 1) // 2, (M + 1) // 2
            L = 1 << int(np.ceil(np.log2(N + M - 1)))
            cross.append({"N": N, "M": M, "Z": 8, "matrix": a, "czt_fft": f, "fft_length": L,
                          "matrix_executed_flop": 3 * 3 * 8 * 16.0 * n * m * (n + m),
                          "fft_flop": 3 * 8 * (N + M) * 2 * 5.0 * L * np.log2(L),
                          "ratio_czt_over_matrix": f["us_mean"] / a["us_mean"]})
    clocks = sampler.stop()
    ref = next(r for r in fig5 if r["N"] == 512)
    ms = ref["vectorial_cartesian"]["us_mean"] * 1e-3
    line = {"metric": METRIC, "value": 201 * 201 / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": 20, "warmup": 3,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16x3",
            "data": "synthetic",
            "config": {"workload": "fig5_single_plane (PAPER.md:239: one 201 x 201 plane at focus vs pupil size); value = the "
                                   "N = 512 vectorial Cartesian point", "l2": "256 MiB buffer written between timed calls"},
            "clocks": clocks, "fig5_us_per_psf": fig5, "crossover_matrix_vs_fft": cross, "gpu_launches": 2 * 20}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS) + ["fig5"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the per-workload table of the other four configs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.workload == "fig5":
        if args.impl == "reference":
            print(json.dumps({"impl": "reference", "unavailable": "the fig5 workload has no reference arm: the paper prints no numbers for Fig. 5"}))
            return 0
        return run_fig5(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
