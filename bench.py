#!/usr/bin/env python
"""bench.py -- throughput of the fused SOS + STA/LTA stream path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg3] [--mode chunked|whole] [--layout cm|tm]

One "step" = one pass of the whole hot path (S0..S7, include/filark_stream.h) over one record
of the workload: `reset`, then the record pushed chunk by chunk (cfg3: 60 pushes of 1,500
samples on 6,000 channels = 60 s of the paper's 6,000-channel x 1,500 Hz acquisition shape,
PAPER.md:27) -- or in one push with --mode whole.  Inputs are seeded synthetic DAS-shaped data
(paper_2605_20132_b200/workloads.py) resident in HBM before the timed region; every push reads
a different 36 MB chunk and writes 72 MB, the record (6.5 GB of traffic per step) is far larger
than the 126 MB L2, so no flush is needed between iterations.

Prints ONE JSON line (rank 0).  Keys beyond the driver's contract:
  roofline      dominant (only) kernel vs the measured HBM copy peak of MEASURED_PEAKS.json
  cpu_baseline  the float64 oracle, as it stands, on this box's host cores, bounded sample
  e2e           same metric through filark_stream_push_host with pinned HOST buffers
  detail        the same record in one push / through separate push calls / sustained for seconds with
                its clock record / one output only, and every other BASELINE.json config (all_configs)

N > 1 (torchrun): the path shards by channel with no exchange step; every rank
streams its own 6,000-channel fibre (weak scaling), time = max over ranks, no data-path
collective.  --impl reference times the oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALG_BYTES_PER_SAMPLE = 12.0          # 4 read + 4 filt + 4 cf; 8 when one output is NULL
HBM_NOMINAL_GBS = 8000.0             # the denominator BASELINE.json north_star names
FALLBACK_HBM_GBS = 6650.0            # B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--mode", default="chunked", choices=["chunked", "whole"])
    ap.add_argument("--layout", default="cm", choices=["cm", "tm"])
    ap.add_argument("--force-l", type=int, default=0, help="tuning: force the sub-block length variant")
    ap.add_argument("--outputs", default="both", choices=["both", "filt", "cf"],
                    help="which outputs the pushes ask for (the other pointer is NULL: 8 B/sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-detail", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true", help="skip detail.all_configs (the other BASELINE.json configs)")
    ap.add_argument("--sustain-seconds", type=float, default=5.0, help="length of the detail.sustained loop")
    ap.add_argument("--api", default="push_many", choices=["push_many", "push", "push_overlap"],
                    help="how a step enqueues its pushes: one filark_stream_push_many call (default), separate "
                         "filark_stream_push calls (strict stream order), or separate calls on a handle created with "
                         "FILARK_FLAG_OVERLAP_PUSHES")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample-channels", type=int, default=0, help="0 = sized for ~15 core-s")
    return ap.parse_args()


# ------------------------------------------------------------------------------------ helpers
def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock + throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        self.index, self.period = index, period_s
        self.samples, self.reasons = [], set()
        self.max_mhz = None
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

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap,
                 "hw_power_brake": nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------ oracle arm
def oracle_throughput(w, sos, x_cm_host, schedule, threads):
    """Stream a channel-major host sample through the oracle chunk by chunk; samples/s."""
    from oracle import Oracle
    import numpy as np
    n_ch = x_cm_host.shape[0]
    o = Oracle(n_ch, sos, w.sta_len, w.lta_len)
    chunks, p = [], 0
    for c in schedule:
        chunks.append(np.ascontiguousarray(x_cm_host[:, p:p + c])); p += c
    t0 = time.perf_counter()
    for ch in chunks:
        o.push(ch, threads=threads)
    dt = time.perf_counter() - t0
    o.close()
    return n_ch * p / dt, dt


def run_reference(args, rank):
    """--impl reference: the float64 oracle on the host cores, bounded sample per step."""
    if rank != 0:
        return
    import numpy as np
    import torch
    from paper_2605_20132_b200.workloads import CONFIGS, design_sos, generate, push_schedule
    w = CONFIGS[args.workload]
    sos = design_sos(w)
    cores = os.cpu_count() or 1
    # (the same bounded sample as the cpu_baseline leg of the CUDA arm: a few thousand channels, so that the
    # per-push start of the worker threads does not dominate the 1,500-sample pushes)
    n_ch_s = args.cpu_sample_channels or max(cores, min(w.n_ch, int(15.0 * 30e6 / w.n_t)))
    ws = w.scaled(n_ch=n_ch_s, n_t=w.n_t)
    x = generate(ws, device="cpu").numpy()
    sched = push_schedule(ws) if args.mode == "chunked" else [ws.n_t]
    for _ in range(max(1, min(args.warmup, 1))):
        oracle_throughput(ws, sos, x[:, :sched[0] * 2], sched[:2], cores)
    vals, tot = [], 0.0
    for _ in range(args.steps):
        v, dt = oracle_throughput(ws, sos, x, sched, cores)
        vals.append(v); tot += dt
    value = n_ch_s * ws.n_t * args.steps / tot
    sample = (f"{n_ch_s} of {w.n_ch} channels x {ws.n_t} samples of {w.name} per step, "
              f"{len(sched)} pushes, channels split over {cores} threads")
    out = {"impl": "reference", "metric": "samples/s (fused SOS+STA/LTA stream)", "value": value,
           "unit": "samples/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(w, args, sched),
           "cpu_baseline": {"value": value, "unit": "samples/s", "cores": cores, "kind": "oracle",
                            "sample": sample},
           "e2e": {"value": value, "unit": "samples/s", "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def make_step(stream, api, batch, ins, filts, cfs):
    """One pass of the whole hot path over the record: reset + every push of the schedule."""
    if api == "push_many":
        def step():
            stream.reset()
            stream.push_many(batch)                  # one host call enqueues every push of the record
    else:
        fl = filts if filts is not None else [None] * len(ins)
        cl = cfs if cfs is not None else [None] * len(ins)

        def step():
            stream.reset()
            for xi, fi, ci in zip(ins, fl, cl):
                stream.push(xi, fi, ci)
    return step


def workload_config(w, args, sched):
    return {"workload": f"{w.name}: {w.n_ch} ch x {w.n_t} samples fp32 at fs={w.fs:g} Hz "
                        f"(BASELINE.json configs[{int(w.name[3:]) - 1}])",
            "filter": f"Butterworth bandpass order {w.order} ({w.order} SOS sections) "
                      f"{w.band[0]:g}-{w.band[1]:g} Hz",
            "sta_len": w.sta_len, "lta_len": w.lta_len,
            "layout": "channel-major [n_ch][n_t]" if args.layout == "cm" else "time-major [n_t][n_ch]",
            "pushes_per_step": len(sched), "chunk_samples": sched[0] if len(set(sched)) == 1 else "mixed",
            "l2": "inputs larger than L2: each push reads a distinct chunk; 6.5 GB traffic per step",
            "api": {"push_many": "filark_stream_reset + ONE filark_stream_push_many call per step: chunks that share "
                                 "no buffer run in common launches of up to 64 chunks, the carried state stays on "
                                 "the SM between them (include/filark_stream.h)",
                    "push": "filark_stream_reset + one filark_stream_push call per chunk, strict stream order",
                    "push_overlap": "filark_stream_reset + one filark_stream_push call per chunk on a handle with "
                                    "FILARK_FLAG_OVERLAP_PUSHES: consecutive launches overlap on the device"}[args.api],
            "parallelism": "independent channel shards, one stream handle per GPU, no collective"}


# ------------------------------------------------------------------------------------ CUDA arm
def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2605_20132_b200.stream import FLAG_OVERLAP_PUSHES, FilarkStream, PushBatch, load_library
    from paper_2605_20132_b200.workloads import (CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos,
                                                  generate, push_schedule)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for this path)")
    load_library()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = CONFIGS[args.workload]
    sos = design_sos(w)
    global ALG_BYTES_PER_SAMPLE
    if args.outputs != "both":
        ALG_BYTES_PER_SAMPLE = 8.0
    layout = CHANNEL_MAJOR if args.layout == "cm" else TIME_MAJOR
    sched = push_schedule(w) if args.mode == "chunked" else [w.n_t]

    # ---- inputs resident in HBM: one dense array per push -----------------------------------
    # every rank streams its own fibre: same recipe, rank-dependent seed
    import dataclasses
    wr = dataclasses.replace(w, seed=w.seed + 1000 * rank)
    x = generate(wr, device=dev, layout=CHANNEL_MAJOR)                  # [n_ch][n_t]

    def pack(x_cm, sched, layout):
        ins, p = [], 0
        for c in sched:
            blk = x_cm[:, p:p + c]
            ins.append(blk.contiguous() if layout == CHANNEL_MAJOR else blk.t().contiguous()); p += c
        return ins
    ins = pack(x, sched, layout)
    if len(sched) > 1:
        del x
    filts = [torch.empty_like(t) for t in ins] if args.outputs != "cf" else None
    cfs = [torch.empty_like(t) for t in ins] if args.outputs != "filt" else None
    flags = (args.force_l << 8) | (FLAG_OVERLAP_PUSHES if args.api == "push_overlap" else 0)
    stream = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, layout, flags=flags)
    samples_per_step = w.n_ch * w.n_t
    batch = PushBatch(stream, ins, filts, cfs)       # the step's schedule, marshalled once
    step = make_step(stream, args.api, batch, ins, filts, cfs)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(physical_gpu_index(local_rank))
    l0 = stream.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    barrier()
    torch.cuda.profiler.start()          # ncu --profile-from-start off sees the timed region only
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    torch.cuda.profiler.stop()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = stream.launch_count - l0
    if world > 1:
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    ms_per_step = ms / args.steps
    value = world * samples_per_step / (ms_per_step * 1e-3)

    out = {"metric": "samples/s (fused SOS+STA/LTA stream)", "value": value, "unit": "samples/s",
           "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": workload_config(w, args, sched), "clocks": clocks, "gpu_launches": launches}

    # ---- roofline of the (only) kernel: algorithmic bytes per launch / mean launch duration --
    peak, peak_src = measured_peak()
    per_launch_ms = ms / max(1, launches) if world == 1 else None
    bytes_per_launch = ALG_BYTES_PER_SAMPLE * samples_per_step * args.steps / max(1, launches)
    ach = ALG_BYTES_PER_SAMPLE * samples_per_step / (ms_per_step * 1e-3) / 1e9 / 1.0
    # DRAM bytes of one launch of this command, from the committed ncu --set full capture of the same
    # launch configuration (profiles/r02_traffic.md says which capture each row comes from)
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    try:
        with open(tpath) as f:
            for line in f.read().splitlines()[1:]:
                k, v = line.split(",")
                if k == f"{w.name}_{args.mode}_{args.layout}_{args.api if args.mode == 'chunked' else 'push'}":
                    traffic = float(v)
                    traffic_src = "profiles/r02_traffic.csv (dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full)"
    except Exception:
        pass
    lean = "lean" if True else "all"
    out["roofline"] = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s",
                       "frac": ach / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                       "kernel": ("filark_push_tr_kernel (time-major: one channel per lane, the warps of a CTA are time slices; "
                                  "short launches and handles with a trigger: filark_push_cm_kernel<.., kTM>)" if args.layout == "tm" else
                                  "filark_push_cm_kernel (one instantiation per sub-block length, launch shape, "
                                  "section forms and layout; profiles/ names the one this command launches)"),
                       "algorithmic_bytes_per_launch": bytes_per_launch,
                       "mean_launch_ms": per_launch_ms, "frac_of_nominal_8TBs": ach / HBM_NOMINAL_GBS,
                       "limiter": "instruction issue, not HBM: at 8 sections the kernel executes about 60 (time-major: 75-85) SASS "
                                  "instructions per sample (DESIGN.md 7, profiles/r02_ncu_*.md); HBM is the roof the "
                                  "north star names and the one `frac` is measured against",
                       "note": "achieved = 12 B/sample x samples per step / CUDA-event time of the step (the step is "
                               "the launches of this one kernel + the memsets of reset)"}
    out["detail"] = {"gsamples_per_s": value / 1e9, "alg_gbytes_per_s": ach,
                     "realtime_factor": (w.n_t / w.fs) / (ms_per_step * 1e-3)}

    if rank == 0 and world == 1 and not args.no_detail:
        out["detail"].update(extra_runs(args, w, sos, stream, ins, filts, cfs, sched, torch, dev, peak, step, local_rank))

    # ---- e2e: the same step through filark_stream_push_host with pinned host buffers ---------
    if not args.no_e2e:
        # a host pipeline hands over one chunk at a time: two sets of pinned buffers used
        # alternately (flat, viewed per push so that mixed chunk lengths work too)
        cmax = max(sched)
        pin = [[torch.empty(w.n_ch * cmax, dtype=torch.float32).pin_memory() for _ in range(3)]
               for _ in range(2)]
        for j in range(2):
            pin[j][0][:ins[j % len(ins)].numel()].copy_(ins[j % len(ins)].reshape(-1))
        torch.cuda.synchronize()

        def view(buf, c):
            return buf[:w.n_ch * c].view(w.n_ch, c) if layout == CHANNEL_MAJOR else buf[:w.n_ch * c].view(c, w.n_ch)

        def e2e_step():
            stream.reset()
            for i, c in enumerate(sched):
                hi, hf, hc = pin[i & 1]
                stream.push_host(view(hi, c), view(hf, c), view(hc, c))
            torch.cuda.synchronize()

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        barrier()
        dt = (time.perf_counter() - t0) / args.e2e_steps
        if world > 1:
            t = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        out["e2e"] = {"value": world * samples_per_step / dt, "unit": "samples/s",
                      "h2d_bytes_per_step": 4 * samples_per_step,
                      "d2h_bytes_per_step": 8 * samples_per_step,
                      "ms_per_step": dt * 1e3, "steps": args.e2e_steps,
                      "api": "filark_stream_push_host (pinned host in, filt + cf back to pinned host)"}
        del pin

    # ---- cpu_baseline: the oracle as it stands, on this box's host cores ---------------------
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_ch_s = args.cpu_sample_channels or max(cores, min(w.n_ch, int(15.0 * 30e6 / w.n_t)))
        xs = torch.cat([t[:n_ch_s] if layout == CHANNEL_MAJOR else t[:, :n_ch_s].t() for t in ins],
                       dim=1).contiguous().cpu().numpy()
        v, dt = oracle_throughput(w, sos, xs, sched, cores)
        out["cpu_baseline"] = {"value": v, "unit": "samples/s", "cores": cores, "kind": "oracle",
                               "seconds": dt,
                               "sample": f"first {n_ch_s} of {w.n_ch} channels x all {w.n_t} samples of the "
                                         f"same record, {len(sched)} pushes, channels split over {cores} threads"}

    if rank == 0 and world == 1 and not args.no_detail:
        if not args.no_all_configs:
            # (the headline's buffers stay: 13 GB; the largest config adds 65 GB)
            out["detail"]["all_configs"] = all_configs(args, torch, dev, peak)
        if args.sustain_seconds > 0:
            try:
                out["detail"]["sustained"] = sustained_run(args, torch, step, samples_per_step, peak, local_rank)
            except Exception as exc:
                out["detail"]["sustained"] = {"error": repr(exc)}

    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out), flush=True)


def _time(torch, fn, reps, warm=1):
    """ms per call of fn, CUDA events on the current stream around `reps` back-to-back calls."""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def _row(n_samples, ms, peak, bytes_per_sample=12.0):
    gbs = bytes_per_sample * n_samples / (ms * 1e-3) / 1e9
    return {"ms": ms, "samples_per_s": n_samples / (ms * 1e-3), "alg_gbytes_per_s": gbs, "frac_of_measured_peak": gbs / peak}


def extra_runs(args, w, sos, stream, ins, filts, cfs, sched, torch, dev, peak, step, local_rank):
    """Context beside the headline: the same record in one push, through separate push calls, a
    sustained run with its clock record, one output only, and the other configs of BASELINE.json."""
    from paper_2605_20132_b200.stream import FLAG_OVERLAP_PUSHES, FilarkStream, PushBatch
    from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos, generate, push_schedule
    extra = {}
    n_samples = w.n_ch * w.n_t
    bps = ALG_BYTES_PER_SAMPLE
    layout = CHANNEL_MAJOR if args.layout == "cm" else TIME_MAJOR
    cat_dim = 1 if layout == CHANNEL_MAJOR else 0

    def guarded(name, fn):
        try:
            extra[name] = fn()
        except Exception as exc:                                  # context only
            extra[name] = {"error": repr(exc)}
            torch.cuda.synchronize()

    # ---- the same schedule through separate push calls
    if len(sched) > 1 and args.api == "push_many":
        def per_call(flags):
            s2 = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, layout, flags=(args.force_l << 8) | flags)
            st = make_step(s2, "push", None, ins, filts, cfs)
            ms = _time(torch, st, max(3, args.steps // 2), warm=2)
            s2.destroy()
            return _row(n_samples, ms, peak, bps)
        guarded("separate_push_calls_strict_order", lambda: per_call(0))
        guarded("separate_push_calls_overlapped", lambda: per_call(FLAG_OVERLAP_PUSHES))

    # ---- the record in one push
    if len(sched) > 1:
        def whole():
            x = torch.cat(ins, dim=cat_dim).contiguous()
            f = torch.empty_like(x) if args.outputs != "cf" else None
            c = torch.empty_like(x) if args.outputs != "filt" else None

            def st():
                stream.reset(); stream.push(x, f, c)
            ms = _time(torch, st, max(3, args.steps // 2), warm=2)
            return _row(n_samples, ms, peak, bps)
        guarded("whole_record_push", whole)

    # ---- one output only (the other pointer NULL: 8 B/sample)
    if args.outputs == "both":
        def one_output(which):
            b2 = PushBatch(stream, ins, filts if which == "filt" else None, cfs if which == "cf" else None)

            def st():
                stream.reset(); stream.push_many(b2)
            ms = _time(torch, st, max(3, args.steps // 2), warm=2)
            return _row(n_samples, ms, peak, 8.0)
        guarded("filt_only", lambda: one_output("filt"))
        guarded("cf_only", lambda: one_output("cf"))

        # ---- trigger on the CF fused behind S6 (NEXT-1): both outputs + events, and filt + events with d_cf = NULL
        def with_trigger(want_cf):
            stream.set_trigger(4.0, 2.0, 1 << 20)
            b2 = PushBatch(stream, ins, filts, cfs if want_cf else None)

            def st():
                stream.reset(); stream.push_many(b2)
            ms = _time(torch, st, max(3, args.steps // 2), warm=2)
            ev, dropped = stream.pop_events()
            stream.set_trigger(0.0, 0.0, 0)
            r = _row(n_samples, ms, peak, 12.0 if want_cf else 8.0)
            r.update({"thr_on": 4.0, "thr_off": 2.0, "events_per_step": len(ev) // (max(3, args.steps // 2) + 2), "dropped": dropped})
            return r
        guarded("trigger_both_outputs_and_events", lambda: with_trigger(True))
        guarded("trigger_filt_and_events_no_cf", lambda: with_trigger(False))

    # ---- the two small operators beside the path (NEXT-3, NEXT-4; include/filark_ops.h): pure streaming work
    if layout == CHANNEL_MAJOR and args.outputs == "both":
        def small_ops():
            from paper_2605_20132_b200.ops import FilarkEma, decimate
            x = torch.cat(ins, dim=1).contiguous()
            y = torch.empty_like(x)
            out = {}
            for mode in ("demean", "agc"):
                h = FilarkEma(w.n_ch, w.lta_len, mode, 1e-6)
                ms = _time(torch, lambda: h.push(x, y), 5, warm=1)
                out[f"ema_{mode}"] = _row(n_samples, ms, peak, 8.0)
                h.destroy()
            for mode in ("drop", "peak", "linear"):
                disp = torch.empty((w.n_ch, 2048), device=x.device)
                ms = _time(torch, lambda: decimate(x, mode, 2048, CHANNEL_MAJOR, disp), 5, warm=1)
                out[f"decimate_{mode}_to_2048"] = _row(n_samples, ms, peak, 4.0 if mode == "peak" else 4.0 * 2048 / w.n_t)
            return out
        guarded("small_operators", small_ops)
    return extra


def sustained_run(args, torch, step, n_samples, peak, local_rank):
    """The headline step looped for several seconds, with the clock and power-cap record of that loop
    (run last: it leaves the GPU warm and, at this kernel's power, under the software power cap)."""
    sampler = ClockSampler(physical_gpu_index(local_rank), period_s=0.02)
    ms1 = _time(torch, step, 3)
    reps = max(10, int(args.sustain_seconds * 1e3 / ms1))
    sampler.start()
    ms = _time(torch, step, reps, warm=0)
    clocks = sampler.stop()
    r = _row(n_samples, ms, peak, ALG_BYTES_PER_SAMPLE)
    r.update({"steps": reps, "seconds": reps * ms * 1e-3, "clocks": clocks})
    return r


def all_configs(args, torch, dev, peak):
    """Every BASELINE.json config x {its chunk schedule through push_many, one whole-record push}, both
    layouts for the headline config; a few steps each (bounded: the default run must end within minutes)."""
    from paper_2605_20132_b200.stream import FilarkStream, PushBatch
    from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos, generate, push_schedule
    out = {}
    for name, lay in (("cfg1", "cm"), ("cfg2", "cm"), ("cfg3", "tm"), ("cfg4", "cm"), ("cfg5", "cm")):
        key = f"{name}_{lay}"
        try:
            w = CONFIGS[name]
            layout = CHANNEL_MAJOR if lay == "cm" else TIME_MAJOR
            sos = design_sos(w)
            sched = push_schedule(w)
            x = generate(w, device=dev, layout=CHANNEL_MAJOR)
            ins, p = [], 0
            for c in sched:
                blk = x[:, p:p + c]
                ins.append(blk.contiguous() if layout == CHANNEL_MAJOR else blk.t().contiguous()); p += c
            big = name == "cfg5"
            if layout == TIME_MAJOR:
                xw = x.t().contiguous()
                del x
            else:
                xw = x
            fs = [torch.empty_like(t) for t in ins]; cs = [torch.empty_like(t) for t in ins]
            st = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, layout)
            b = PushBatch(st, ins, fs, cs)

            def chunked():
                st.reset(); st.push_many(b)
            n = w.n_ch * w.n_t
            reps = 2 if big else 5
            row = {"shape": f"{w.n_ch} x {w.n_t}", "sections": w.order, "pushes": len(sched),
                   "chunked_push_many": _row(n, _time(torch, chunked, reps, warm=1), peak)}
            del fs, cs, b
            fw = torch.empty_like(xw); cw = torch.empty_like(xw)

            def whole():
                st.reset(); st.push(xw, fw, cw)
            row["whole_record_push"] = _row(n, _time(torch, whole, reps, warm=1), peak)
            st.destroy()
            out[key] = row
            del ins, xw, fw, cw
            torch.cuda.empty_cache()
        except Exception as exc:
            out[key] = {"error": repr(exc)}
            torch.cuda.synchronize()
            torch.cuda.empty_cache()
    return out


if __name__ == "__main__":
    main()
